"""The seeded input generator: determinism, bit-equality of the numpy and torch fillers, pattern
structure, the C-12 positive-definiteness rescale, and restriction to neighbourhoods."""
import numpy as np
import torch

from workloads import MAT_H, MAT_S, gamma_table, hash_uniform_np, hash_uniform_torch, make_system, to_scipy


def test_hash_numpy_and_torch_agree_bitwise():
    rng = np.random.default_rng(0)
    lo = rng.integers(0, 1 << 20, 5000)
    hi = lo + rng.integers(0, 1 << 20, 5000)
    el = rng.integers(0, 4096, 5000)
    a = hash_uniform_np(7, MAT_S, lo, hi, el)
    b = hash_uniform_torch(7, MAT_S, torch.from_numpy(lo), torch.from_numpy(hi), torch.from_numpy(el)).numpy()
    assert np.array_equal(a, b)
    assert 0.0 <= a.min() and a.max() < 1.0 and abs(a.mean() - 0.5) < 0.02


def test_cfg0_recipe():
    s = make_system("cfg0")
    assert s.n_atoms == 64 and s.box is None and (s.atom_nb == 4).all()
    edge = (64 / 0.1) ** (1 / 3)
    assert (s.pos >= 0).all() and (s.pos < edge).all()
    d = np.sqrt(((s.pos[:, None] - s.pos[None]) ** 2).sum(-1)) + 10 * np.eye(64)
    assert d.min() >= 1.0
    rows = s.slot_rows()
    pat = np.zeros((64, 64), bool)
    pat[rows, s.col_idx] = True
    assert np.array_equal(pat, pat.T) and pat.diagonal().all()
    for i in range(64):
        c = s.col_idx[s.row_ptr[i]:s.row_ptr[i + 1]]
        assert (np.diff(c) > 0).all()
    Hv, Sv = s.fill_np(MAT_H), s.fill_np(MAT_S)
    assert np.array_equal(Hv, s.fill_torch(MAT_H).numpy()) and np.array_equal(Sv, s.fill_torch(MAT_S).numpy())
    S = to_scipy(s, Sv).toarray()
    H = to_scipy(s, Hv).toarray()
    assert np.array_equal(S, S.T) and np.array_equal(H, H.T)
    assert np.array_equal(S.diagonal(), np.ones(256))
    lam = np.linalg.eigvalsh(S)
    assert abs(lam[0] - 0.2) < 1e-6                      # C-12: gamma puts lambda_min(S) on the floor
    on = H.diagonal().reshape(64, 4)
    assert (on[:, :2] < -0.5).all() and (on[:, 2:] > 0.5).all()
    assert abs(on[:, :2].mean() + 1) < 0.05 and 0.05 < on[:, :2].std() < 0.15
    # off-site block amplitudes follow the radial laws
    p = s.row_ptr[3] + 1 if s.col_idx[s.row_ptr[3]] == 3 else s.row_ptr[3]
    r = s.dist[p]
    blk = s.blk_off()
    assert np.abs(Sv[blk[p]:blk[p + 1]]).max() <= s.gamma * 0.3 * np.exp(-r * r / 8) + 1e-15
    assert np.abs(Hv[blk[p]:blk[p + 1]]).max() <= 0.5 * np.exp(-r / 1.5) + 1e-15


def test_periodic_small_proxy_and_restrict():
    s = make_system("cfg1", n_atoms=400)
    assert s.box is not None and s.box >= 12.0
    nn = np.diff(s.row_ptr)
    assert 60 < nn.mean() < 120                           # (4/3) pi 6^3 * 0.1 = 90.5 neighbours
    Hv = s.fill_np(MAT_H)
    atoms = np.unique(np.concatenate([s.col_idx[s.row_ptr[i]:s.row_ptr[i + 1]] for i in (5, 77)]))
    sub = s.restrict(atoms)
    blk = s.blk_off()
    want = np.concatenate([Hv[blk[p]:blk[p + 1]] for p in sub.meta["parent_slots"]])
    assert np.array_equal(sub.fill_np(MAT_H), want)
    assert set(gamma_table()) >= {"cfg0", "cfg1", "cfg2", "cfg3", "cfg4"}


def test_mixed_basis_blocks_are_transposes():
    s = make_system("cfg3", n_atoms=600)
    assert set(np.unique(s.atom_nb)) == {5, 13}
    Sv = s.fill_np(MAT_S)
    S = to_scipy(s, Sv).toarray()
    assert np.array_equal(S, S.T)
    assert np.linalg.eigvalsh(S)[0] > 0.2
