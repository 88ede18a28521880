"""GPU parity tests: the CUDA path, called through the C ABI (include/nolsm.h), against the FP64 oracle
on the same seeded inputs. Tolerances are BASELINE.json's: index sets bit-exact; FP16/FP32 mixed
max|dD| <= 2e-2 and |dE|/|E| <= 1e-3; all-FP32 <= 1e-5 on both."""
import numpy as np
import pytest
import torch

from oracle import nolsm_oracle as orc
from tests.helpers import compare_atoms, oracle_on_atoms
from workloads import MAT_H, MAT_S, make_system

pytestmark = pytest.mark.gpu

TOL_MIXED_D, TOL_MIXED_E = 2e-2, 1e-3
TOL_FP32 = 1e-5


def _nolsm(**kw):
    from paper_2205_12182_b200 import Nolsm
    kw.setdefault("timeout_s", 90.0)              # a stalled kernel fails the test instead of holding the GPU for minutes
    return Nolsm(0, **kw)


def _arrays(s, device="cuda"):
    Hv = torch.from_numpy(s.fill_np(MAT_H)).to(device)
    Sv = torch.from_numpy(s.fill_np(MAT_S)).to(device)
    return (torch.from_numpy(s.atom_nb).to(device), torch.from_numpy(s.row_ptr).to(device),
            torch.from_numpy(s.col_idx).to(device), Hv, Sv)


def _run(s, atoms=None, device="cuda", d_dtype=torch.float64, **kw):
    from paper_2205_12182_b200 import PREC_FP32
    nb, rp, ci, Hv, Sv = _arrays(s, device)
    with _nolsm(**kw) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        D = torch.zeros(Hv.shape[0], dtype=d_dtype, device=device)
        ctx.density_matrix(s.mu, D)
        E = ctx.energy()
        st = ctx.atom_stats()
        stats = ctx.stats()
    return D.cpu().numpy(), E, st, stats


@pytest.fixture(scope="module")
def cfg0():
    return make_system("cfg0")


def test_index_sets_bit_exact_cfg0(cfg0):
    s = cfg0
    with _nolsm() as ctx:
        ctx.assemble(*_arrays(s))
        for i in range(s.n_atoms):
            N, dim = ctx.index_set(i)
            ref = orc.index_set(i, s.row_ptr, s.col_idx)
            assert N.dtype == np.int32 and np.array_equal(N, ref)
            assert dim == int(s.atom_nb[ref].sum())


def test_index_sets_with_eps_filter_bit_exact(cfg0):
    s = cfg0
    Hv, Sv = s.fill_np(MAT_H), s.fill_np(MAT_S)
    blk = s.blk_off()
    eps = 0.02
    with _nolsm(eps_filter=eps) as ctx:
        ctx.assemble(*_arrays(s))
        smaller = 0
        for i in range(s.n_atoms):
            N, dim = ctx.index_set(i)
            ref = orc.index_set(i, s.row_ptr, s.col_idx, s.atom_nb, blk, Hv, Sv, eps)
            assert np.array_equal(N, ref)
            smaller += len(ref) < (s.row_ptr[i + 1] - s.row_ptr[i])
        assert smaller > 0


def test_gather_bit_exact(cfg0):
    """P13: no arithmetic happens in a gather -- FP32 output equals float32(oracle), FP16 output equals
    the RN-even rounding of the oracle's FP64 submatrix, bit for bit."""
    s = cfg0
    Hv, Sv = s.fill_np(MAT_H), s.fill_np(MAT_S)
    blk = s.blk_off()
    with _nolsm() as ctx:
        ctx.assemble(*_arrays(s))
        for i in (0, 7, 63):
            N = orc.index_set(i, s.row_ptr, s.col_idx)
            for which, vals in ((0, Sv), (1, Hv)):
                T, _ = orc.submatrix(N, s.atom_nb, s.row_ptr, s.col_idx, blk, vals)
                g16 = ctx.gather_submatrix(i, which, fp16=True)
                g32 = ctx.gather_submatrix(i, which, fp16=False)
                assert np.array_equal(g16.view(np.uint16), T.astype(np.float16).view(np.uint16))
                assert np.array_equal(g32, T.astype(np.float32))


@pytest.mark.parametrize("name,n_atoms,combine", [("cfg2", 300, 0), ("cfg3", 20000, 0), ("cfg2", 300, 1), ("cfg3", 900, 1)])
def test_gather_bit_exact_large(name, n_atoms, combine):
    """P13 at the sizes where the gather task has more than one path: submatrices of 1200-2100 dimensions (the dense
    strip of a row-atom takes several passes once 2 n16 exceeds 48 KB / 13 rows), mixed 5- and 13-function blocks
    (cfg3 at full size: the largest submatrix of the blob), and a combined unit's union set (the dense matrix the group is
    evaluated on). FP16 output == RN-even(FP64 -> FP16) of the oracle's dense submatrix, bit for bit."""
    s = make_system(name, n_atoms=None if (name, n_atoms) == ("cfg3", 20000) else n_atoms)
    dims = np.array([int(s.atom_nb[s.col_idx[s.row_ptr[i]:s.row_ptr[i + 1]]].sum()) for i in range(s.n_atoms)])
    picks = [int(np.argmax(dims)), int(np.argsort(dims)[len(dims) // 2])]
    if name == "cfg3":
        mixed = [i for i in np.argsort(-dims)[:2000] if len(set(s.atom_nb[s.col_idx[s.row_ptr[i]:s.row_ptr[i + 1]]].tolist())) == 2]
        picks.append(int(mixed[0]))                                  # a large submatrix with both block sizes
    need = np.unique(np.concatenate([s.col_idx[s.row_ptr[a]:s.row_ptr[a + 1]] for a in picks]))
    if combine:
        sets = [orc.index_set(i, s.row_ptr, s.col_idx) for i in range(s.n_atoms)]
        groups = orc.combine_groups(s.atom_nb, sets, mode=1)
        big = max(groups, key=len)
        assert len(big) > 1
        picks = [big[0], big[-1]]
    blk = s.blk_off()
    if s.n_atoms > 5000:                                             # values on the device only; the oracle sees the neighbourhoods
        Hd, Sd = s.fill_torch(MAT_H, "cuda"), s.fill_torch(MAT_S, "cuda")
        sub = s.restrict(need)
        Hn, Sn = sub.fill_np(MAT_H), sub.fill_np(MAT_S)
        sblk = orc.block_offsets(sub.atom_nb, sub.row_ptr, sub.col_idx)
        parent = sub.meta["parent_atoms"]
        dense = lambda i, vals: orc.submatrix(np.searchsorted(parent, s.col_idx[s.row_ptr[i]:s.row_ptr[i + 1]]),
                                              sub.atom_nb, sub.row_ptr, sub.col_idx, sblk, vals)[0]
        arrays = (torch.from_numpy(s.atom_nb).cuda(), torch.from_numpy(s.row_ptr).cuda(), torch.from_numpy(s.col_idx).cuda(), Hd, Sd)
    else:
        Hn, Sn = s.fill_np(MAT_H), s.fill_np(MAT_S)
        arrays = _arrays(s)
        if combine:
            dense = lambda i, vals: orc.submatrix(np.unique(np.concatenate([sets[m] for m in next(g for g in groups if i in g)])),
                                                  s.atom_nb, s.row_ptr, s.col_idx, blk, vals)[0]
        else:
            dense = lambda i, vals: orc.submatrix(orc.index_set(i, s.row_ptr, s.col_idx), s.atom_nb, s.row_ptr, s.col_idx, blk, vals)[0]
    biggest = 0
    with _nolsm(combine=combine) as ctx:
        ctx.assemble(*arrays)
        for i in picks:
            for which, vals in ((0, Sn), (1, Hn)):
                T = dense(i, vals)
                g16 = ctx.gather_submatrix(i, which, fp16=True)
                assert g16.shape == T.shape
                assert np.array_equal(g16.view(np.uint16), T.astype(np.float16).view(np.uint16))
                biggest = max(biggest, T.shape[0])
    assert biggest >= (1400 if name == "cfg2" or not combine else 1000)   # 13-row atoms: more than one strip pass from n16 = 1904 on
    print("gather bit-exact", name, combine, [int(dims[i]) for i in picks], biggest)


def test_cfg0_fp32_mode(cfg0):
    from paper_2205_12182_b200 import PREC_FP32
    s = cfg0
    D, E, st, stats = _run(s, precision=PREC_FP32)
    cmp = compare_atoms(s, D, st["e_atom"], range(s.n_atoms))
    print("fp32 cfg0", {k: v for k, v in cmp.items() if k != "ref"}, stats)
    assert (st["status"] == 0).all()
    assert cmp["max_abs_dD"] <= TOL_FP32
    assert cmp["rel_dE"] <= TOL_FP32
    assert abs(E - cmp["e_ref"]) / abs(cmp["e_ref"]) <= TOL_FP32


@pytest.mark.parametrize("backend", ["umma", "umma-fulltiles", "lowdin", "lowdin-fulltiles", "simt"])
def test_cfg0_mixed_mode(cfg0, backend):
    """umma: tcgen05 GEMMs in the persistent engine (the default path: Eq. 6 form, the symmetric Schulz products multiply the
    upper triangle of tiles only); -fulltiles: every tile multiplied; lowdin: the symmetric form (C-21);
    simt: FP16 operands with FFMA GEMMs (round engine)."""
    from paper_2205_12182_b200 import ENGINE_PERSISTENT, GEMM_SIMT, GEMM_UMMA, ITER_LOWDIN
    s = cfg0
    kw = {"umma": dict(gemm_backend=GEMM_UMMA, engine=ENGINE_PERSISTENT),
          "umma-fulltiles": dict(symmetric_tiles=-1),
          "lowdin": dict(iteration=ITER_LOWDIN),
          "lowdin-fulltiles": dict(iteration=ITER_LOWDIN, symmetric_tiles=-1),
          "simt": dict(gemm_backend=GEMM_SIMT)}[backend]
    D, E, st, stats = _run(s, **kw)
    cmp = compare_atoms(s, D, st["e_atom"], range(s.n_atoms))
    print("mixed cfg0", backend, {k: v for k, v in cmp.items() if k != "ref"}, stats)
    assert (st["status"] == 0).all()
    assert cmp["max_abs_dD"] <= TOL_MIXED_D
    assert cmp["rel_dE"] <= TOL_MIXED_E
    assert abs(E - cmp["e_ref"]) / abs(cmp["e_ref"]) <= TOL_MIXED_E


def test_cfg0_host_buffers_and_fp32_output(cfg0):
    """Host (numpy) inputs and a host float32 output go through the same C-ABI calls."""
    s = cfg0
    Hv, Sv = s.fill_np(MAT_H), s.fill_np(MAT_S)
    with _nolsm() as ctx:
        ctx.assemble(s.atom_nb, s.row_ptr, s.col_idx, Hv, Sv)
        D = np.zeros(len(Hv), dtype=np.float32)
        ctx.density_matrix(s.mu, D)
        E = ctx.energy()
        st = ctx.atom_stats()
    cmp = compare_atoms(s, D, st["e_atom"], range(0, s.n_atoms, 5))
    assert cmp["max_abs_dD"] <= TOL_MIXED_D and cmp["rel_dE"] <= TOL_MIXED_E
    assert np.isfinite(E)


def test_density_matrix_range_touches_only_its_rows(cfg0):
    s = cfg0
    nb, rp, ci, Hv, Sv = _arrays(s)
    blk = s.blk_off()
    with _nolsm() as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        D = torch.full((Hv.shape[0],), 7.0, dtype=torch.float64, device="cuda")
        e = ctx.density_matrix_range(s.mu, 10, 20, D, want_energy=True)
        st = ctx.atom_stats()
    Dh = D.cpu().numpy()
    v0, v1 = blk[s.row_ptr[10]], blk[s.row_ptr[20]]
    assert (Dh[:v0] == 7.0).all() and (Dh[v1:] == 7.0).all()
    cmp = compare_atoms(s, Dh, st["e_atom"], range(10, 20))
    assert cmp["max_abs_dD"] <= TOL_MIXED_D
    assert abs(e - cmp["e_ref"]) / abs(cmp["e_ref"]) <= TOL_MIXED_E


@pytest.mark.parametrize("engine", ["persistent", "persistent-fulltiles", "persistent-untransposed", "lowdin", "rounds"])
@pytest.mark.parametrize("name,n_atoms,sample", [("cfg1", 600, 6), ("cfg2", 300, 3), ("cfg3", 1500, 6)])
def test_small_proxies_mixed(name, n_atoms, sample, engine):
    """Reduced-size versions of configs 1-3 (same density, basis and generator): several tiles per
    matrix (mirrored off-diagonal tiles, ragged tails, transposed tiles of the last row block, half-height corner tiles),
    mixed 5/13 basis for cfg3. Oracle on a seeded sample of atoms. -untransposed: the last row block as M = 256 / 128 tiles;
    rounds: the FFMA round engine on FP16 operands."""
    from paper_2205_12182_b200 import ENGINE_PERSISTENT, ENGINE_ROUNDS, ITER_LOWDIN
    s = make_system(name, n_atoms=n_atoms)
    atoms = np.random.default_rng(1).choice(s.n_atoms, sample, replace=False)
    kw = {"persistent": dict(engine=ENGINE_PERSISTENT), "persistent-fulltiles": dict(symmetric_tiles=-1),
          "persistent-untransposed": dict(transposed_tiles=-1), "lowdin": dict(iteration=ITER_LOWDIN), "rounds": dict(engine=ENGINE_ROUNDS)}[engine]
    D, E, st, stats = _run(s, **kw)
    cmp = compare_atoms(s, D, st["e_atom"], atoms)
    print(name, {k: v for k, v in cmp.items() if k != "ref"}, stats)
    assert (st["status"] == 0).all()
    assert cmp["max_abs_dD"] <= TOL_MIXED_D
    assert cmp["rel_dE"] <= TOL_MIXED_E


def test_transposed_last_row_block_over_every_remainder():
    """The tiles of a ragged last row block are computed as C^T = B^T A^T (TI_TRANS): submatrix dimensions whose remainder
    modulo 256 runs over 16 .. 240 (both sides of the 128-row limit of the half-height corner tile, one and two boxes per
    CTA), every tile multiplied so that the symmetric products take the transposed tiles too; against the oracle on a
    sample and against the untransposed engine on every atom."""
    s = make_system("cfg2", n_atoms=300)
    runs = {}
    for key, kw in (("trans", dict(symmetric_tiles=-1)), ("plain", dict(symmetric_tiles=-1, transposed_tiles=-1))):
        runs[key] = _run(s, **kw)
        assert (runs[key][2]["status"] == 0).all()
    Dt, Dp = runs["trans"][0], runs["plain"][0]
    dims = runs["trans"][2]["dims"]
    rem = np.unique(((dims[dims > 256] + 15) // 16 * 16) % 256)
    print("remainders", rem)
    assert (rem > 128).any() and ((rem > 0) & (rem <= 128)).any() and len(rem) >= 8
    # same arithmetic per element (k order of the MMA, FP32 accumulation); run-to-run differences come from the order of the
    # residual atomics only, which can move a convergence decision by one iteration
    assert np.abs(Dt - Dp).max() <= TOL_MIXED_D
    atoms = np.random.default_rng(9).choice(s.n_atoms, 3, replace=False)
    cmp = compare_atoms(s, Dt, runs["trans"][2]["e_atom"], atoms)
    assert cmp["max_abs_dD"] <= TOL_MIXED_D and cmp["rel_dE"] <= TOL_MIXED_E
    # the executed (padded) work shrinks, the useful work does not change
    assert runs["trans"][3]["flops_padded"] < runs["plain"][3]["flops_padded"]
    assert runs["trans"][3]["flops_padded"] >= runs["trans"][3]["flops_useful"]


def test_plain_newton_schulz_matches_scaled():
    """sign_scaled_iters = -1 runs Eq. 6 unscaled after X0 = A / rho; the scaled schedule (default) must reach
    the same D within the mixed tolerances and with fewer GEMMs."""
    s = make_system("cfg2", n_atoms=300)
    atoms = np.random.default_rng(4).choice(s.n_atoms, 3, replace=False)
    D0, E0, st0, stats0 = _run(s, sign_scaled_iters=-1)
    D1, E1, st1, stats1 = _run(s)
    c0 = compare_atoms(s, D0, st0["e_atom"], atoms)
    c1 = compare_atoms(s, D1, st1["e_atom"], atoms)
    print("plain", c0["max_abs_dD"], c0["rel_dE"], stats0["gemms_executed"], "scaled", c1["max_abs_dD"], c1["rel_dE"], stats1["gemms_executed"])
    for c in (c0, c1):
        assert c["max_abs_dD"] <= TOL_MIXED_D and c["rel_dE"] <= TOL_MIXED_E
    assert stats1["gemms_executed"] < stats0["gemms_executed"]
    assert abs(E0 - E1) / abs(E0) <= TOL_MIXED_E


def test_small_proxy_fp32():
    from paper_2205_12182_b200 import PREC_FP32
    s = make_system("cfg1", n_atoms=400)
    atoms = np.random.default_rng(2).choice(s.n_atoms, 4, replace=False)
    D, E, st, stats = _run(s, precision=PREC_FP32)
    cmp = compare_atoms(s, D, st["e_atom"], atoms)
    print("fp32 cfg1@400", {k: v for k, v in cmp.items() if k != "ref"})
    assert cmp["max_abs_dD"] <= TOL_FP32 and cmp["rel_dE"] <= TOL_FP32


def test_single_atom_and_errors():
    from paper_2205_12182_b200 import NolsmError
    nb = np.array([3], np.int32)
    rp = np.array([0, 1], np.int64)
    ci = np.array([0], np.int32)
    H = np.diag([-1.0, 0.5, 2.0]).reshape(-1)
    S = np.eye(3).reshape(-1)
    with _nolsm() as ctx:
        with pytest.raises(NolsmError) as ei:
            ctx.density_matrix(0.0, np.zeros(9))
        assert ei.value.code == 4                                   # ESTATE
        ctx.assemble(nb, rp, ci, H, S)
        D = np.zeros(9)
        ctx.density_matrix(0.0, D)
        E = ctx.energy()
        assert np.allclose(D.reshape(3, 3), np.diag([1.0, 0.0, 0.0]), atol=2e-3)   # P2/P7: projector on eps < mu
        assert abs(E + 1.0) < 2e-3
        with pytest.raises(NolsmError) as ei:                       # unsorted columns
            ctx.assemble(np.array([1, 1], np.int32), np.array([0, 2, 4], np.int64), np.array([1, 0, 0, 1], np.int32),
                         np.ones(4), np.ones(4))
        assert ei.value.code == 1
        with pytest.raises(NolsmError) as ei:                       # non-symmetric pattern
            ctx.assemble(np.array([1, 1], np.int32), np.array([0, 2, 3], np.int64), np.array([0, 1, 1], np.int32),
                         np.ones(3), np.ones(3))
        assert ei.value.code == 1
        with pytest.raises(NolsmError) as ei:                       # missing diagonal
            ctx.assemble(np.array([1, 1], np.int32), np.array([0, 1, 2], np.int64), np.array([1, 0], np.int32),
                         np.ones(2), np.ones(2))
        assert ei.value.code == 1


@pytest.mark.parametrize("iteration", [0, 1])
def test_eigenvalue_at_mu_is_flagged_noconv_and_half_occupied(iteration):
    """C-9: a generalised eigenvalue exactly at mu. Three atoms with two functions each, full pattern, S = I, and the two
    functions of atom 0 duplicates of each other (equal rows and columns of H0): v = (1, -1, 0, ...) / sqrt 2 is an
    eigenvector with eigenvalue exactly 0 = mu, and it stays an exact null vector of every iterate (columns 0 and 1 of
    every polynomial of H0 are computed by identical operations). The sign iteration can never converge on it: the call
    reports NOLSM_ENOCONV, sets the status bit, and still writes D - with the mode half occupied (sign(0) = 0), which is the
    mean of the oracle's D just below and just above mu."""
    from paper_2205_12182_b200 import NolsmError
    nb = np.array([2, 2, 2], np.int32)
    rp = np.array([0, 3, 6, 9], np.int64)
    ci = np.array([0, 1, 2] * 3, np.int32)
    a, b, c, d, e, f, g, h, i_, j, k, l, m, n_, o = 0.5, 0.25, -0.375, 0.125, 0.3125, -1.25, 0.1875, -0.25, 0.0625, 0.75, 0.125, -0.1875, 1.5, 0.25, -0.875
    Hd = np.array([[a, a, b, c, d, e], [a, a, b, c, d, e], [b, b, f, g, h, i_], [c, c, g, j, k, l], [d, d, h, k, m, n_], [e, e, i_, l, n_, o]])
    assert np.array_equal(Hd, Hd.T)
    eps = np.linalg.eigvalsh(Hd)
    assert np.sum(np.abs(eps) < 1e-12) == 1 and np.sort(np.abs(eps))[1] > 0.05
    Sd = np.eye(6)
    to_blocks = lambda M: np.concatenate([M[2 * i:2 * i + 2, 2 * jj:2 * jj + 2].reshape(-1) for i in range(3) for jj in range(3)])
    Hv, Sv = to_blocks(Hd), to_blocks(Sd)
    with _nolsm(iteration=iteration, max_sign_iters=40) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        D = np.zeros(36)
        ctx.density_matrix(0.0, D)
        with pytest.raises(NolsmError) as ei:
            ctx.energy()
        assert ei.value.code == 6                                   # NOLSM_ENOCONV, after writing the result
        st = ctx.atom_stats()
        assert (st["status"] == 2).all() and (st["sign_iters"] >= 39).all()
    blk = orc.block_offsets(nb, rp, ci)
    for atom in range(3):
        lo = orc.atom_result(atom, nb, rp, ci, blk, Hv, Sv, -0.01)
        hi = orc.atom_result(atom, nb, rp, ci, blk, Hv, Sv, +0.01)
        ref = 0.5 * (lo["Dcols"] + hi["Dcols"])                    # [6 rows, 2 columns of the atom]
        got = np.stack([D[blk[3 * atom + jj]:blk[3 * atom + jj + 1]].reshape(2, 2).T for jj in range(3)]).reshape(6, 2)   # slot (i, j) = (D_ji)^T
        assert np.abs(got - ref).max() <= TOL_MIXED_D
        assert abs(float(st["e_atom"][atom]) - 0.5 * (lo["e_i"] + hi["e_i"])) <= 2e-3


@pytest.mark.parametrize("iteration", [0, 1])
def test_electron_counts_for_several_mu_in_one_pass(cfg0, iteration):
    """nolsm_electron_counts: Tr(D(mu_j) S) and Tr(D(mu_j) H0) for several trial mu on the resident S_sub^-1 and A0 (C-20)
    against the oracle's count at each mu, and against one nolsm_density_matrix call per mu."""
    s = cfg0
    nb, rp, ci, Hv, Sv = _arrays(s)
    Hn, Sn = s.fill_np(MAT_H), s.fill_np(MAT_S)
    mus = [-0.6, -0.05, 0.3, 1.1]
    n_tot = float(s.atom_nb.sum())
    with _nolsm(iteration=iteration) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        counts, energies = ctx.electron_counts(mus, with_energy=True)
        D = torch.zeros(Hv.shape[0], dtype=torch.float64, device="cuda")
        for j, mu in enumerate(mus):
            ref = orc.electron_count(s.atom_nb, s.row_ptr, s.col_idx, Hn, Sn, mu)
            assert abs(counts[j] - ref) <= TOL_MIXED_E * n_tot
            ctx.density_matrix(mu, D)
            E1 = ctx.energy()
            assert abs(ctx.electron_count() - counts[j]) <= TOL_MIXED_E * n_tot
            assert abs(E1 - energies[j]) <= TOL_MIXED_E * abs(E1) + 1e-3
        assert all(counts[j + 1] >= counts[j] - 1e-3 for j in range(len(mus) - 1))       # never decreases with mu
    print("electron_counts", iteration, counts, energies)


def test_fp32_mode_on_13_function_submatrices():
    """The all-FP32 validation mode (plain FFMA round engine) where it is hard: submatrices of ~1200 dimensions with 13
    functions per atom, whose spectra reach within 1e-3 of mu (cfg2) - and the mixed 5 / 13 blob of cfg3. BASELINE.json
    asks for 1e-5 on D and E."""
    from paper_2205_12182_b200 import PREC_FP32
    for name, n_atoms, count in (("cfg2", 300, 12), ("cfg3", 900, 12)):
        s = make_system(name, n_atoms=n_atoms)
        nb, rp, ci, Hv, Sv = _arrays(s)
        with _nolsm(precision=PREC_FP32) as ctx:
            ctx.assemble(nb, rp, ci, Hv, Sv)
            D = torch.zeros(Hv.shape[0], dtype=torch.float64, device="cuda")
            ctx.density_matrix_range(s.mu, 0, count, D, want_energy=True)
            st = ctx.atom_stats()
        cmp = compare_atoms(s, D.cpu().numpy(), st["e_atom"], range(count))
        print("fp32", name, {k: v for k, v in cmp.items() if k != "ref"})
        assert (st["status"][:count] == 0).all()
        assert cmp["max_abs_dD"] <= TOL_FP32 and cmp["rel_dE"] <= TOL_FP32


def test_one_heavy_token_and_many_small_units():
    """Stress of the token hand-off of the persistent engine (persist.cuh p_token_release): ONE token, many small units
    whose transitions are fast, every slot parks and is woken hundreds of times; a lost wake-up would leave the kernel
    waiting for its time limit. Repeated calls, results equal to the default run."""
    s = make_system("cfg1", n_atoms=600)
    nb, rp, ci, Hv, Sv = _arrays(s)
    D0, E0, st0, _ = _run(s)
    with _nolsm(heavy_slots=1, batch_atoms=24, timeout_s=60.0) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        D = torch.zeros(Hv.shape[0], dtype=torch.float64, device="cuda")
        for _ in range(3):
            ctx.density_matrix(s.mu, D)
            E = ctx.energy()
            assert abs(E - E0) <= TOL_MIXED_E * abs(E0)           # two valid runs (residual sums are atomics: iteration counts may differ)
    assert np.abs(D.cpu().numpy() - D0).max() <= TOL_MIXED_D


def test_boundary_errors_and_diagnostics_of_the_round_2_calls(cfg0):
    """Argument checks of nolsm_set_perf_table / nolsm_electron_counts, the engine counters, and the stand-alone side-task
    timing (bytes and times are positive; the results of the density call before it are declared stale)."""
    from paper_2205_12182_b200 import PREC_FP32, NolsmError
    s = cfg0
    nb, rp, ci, Hv, Sv = _arrays(s)
    with _nolsm() as ctx:
        for bad_n, bad_t in (([300, 200], [1.0, 2.0]), ([100, 200], [1.0, -2.0]), ([0, 200], [1.0, 2.0]), ([100, 9000], [1.0, 2.0])):
            with pytest.raises(NolsmError) as ei:
                ctx.set_perf_table(bad_n, bad_t)
            assert ei.value.code == 1
        ctx.set_perf_table([128, 1024], [100.0, 900.0])
        ctx.set_perf_table([], [])                                   # removes the table
        with pytest.raises(NolsmError) as ei:
            ctx.electron_counts([0.0])                               # not assembled
        assert ei.value.code == 4
        ctx.assemble(nb, rp, ci, Hv, Sv)
        with pytest.raises(NolsmError) as ei:
            ctx.electron_counts([0.1 * k for k in range(9)])         # more than 8 trial mu
        assert ei.value.code == 1
        D = torch.zeros(Hv.shape[0], dtype=torch.float64, device="cuda")
        ctx.density_matrix(s.mu, D)
        ctx.energy()
        ct = ctx.engine_counters()
        assert ct["persistent"] and ct["tiles"] > 0 and ct["pairs"] == 74 and ct["mma_kloop_ms"] > 0
        n_counts = ctx.electron_counts([s.mu])                       # a count-only pass leaves no energy to read
        with pytest.raises(NolsmError) as ei:
            ctx.energy()
        assert ei.value.code == 4
        ctx.density_matrix(s.mu, D)
        assert abs(ctx.electron_count() - n_counts[0]) <= TOL_MIXED_E * float(s.atom_nb.sum())
        for which in (0, 1):
            ms, nbytes = ctx.side_task_bandwidth(which, reps=2)
            assert ms > 0 and nbytes > 0
        with pytest.raises(NolsmError) as ei:                        # the timing overwrote the energies
            ctx.energy()
        assert ei.value.code == 4
    with _nolsm(precision=PREC_FP32) as ctx:                         # round engine: one trial mu per call only
        ctx.assemble(nb, rp, ci, Hv, Sv)
        with pytest.raises(NolsmError) as ei:
            ctx.electron_counts([0.0, 0.1])
        assert ei.value.code == 4


def test_indefinite_S_is_reported(cfg0):
    """gamma = 1 (BASELINE.json's literal amplitude 0.3) is indefinite on cfg0 (SURVEY finding 1): the
    Schulz inverse cannot converge for the affected submatrices and the library must say so."""
    from paper_2205_12182_b200 import NolsmError
    s = make_system("cfg0", gamma=1.0)
    with _nolsm() as ctx:
        ctx.assemble(*_arrays(s))
        D = torch.zeros(int(s.blk_off()[-1]), dtype=torch.float64, device="cuda")
        ctx.density_matrix(s.mu, D)
        with pytest.raises(NolsmError) as ei:
            ctx.energy()
        assert ei.value.code == 5
        st = ctx.atom_stats()
    bad_gpu = set(np.flatnonzero(st["status"] & 1))
    bad_ref = set()
    Hv, Sv = s.fill_np(MAT_H), s.fill_np(MAT_S)
    blk = s.blk_off()
    for i in range(s.n_atoms):
        N = orc.index_set(i, s.row_ptr, s.col_idx)
        T, _ = orc.submatrix(N, s.atom_nb, s.row_ptr, s.col_idx, blk, Sv)
        if np.linalg.eigvalsh(T)[0] <= 0:
            bad_ref.add(i)
    assert bad_ref and bad_ref <= bad_gpu


# ---- submatrix combination (Eq. 9 / Eq. 10; C-19) ---------------------------------------
def _oracle_groups(s, mode, **kw):
    sets = [orc.index_set(i, s.row_ptr, s.col_idx) for i in range(s.n_atoms)]
    return orc.combine_groups(s.atom_nb, sets, mode=mode, **kw), sets


def _measured_perf_table():
    """p(n) measured on B200 (workloads/pn_b200.json): (dimensions, TFLOP/s) for the library, (dimensions, integer
    GFLOP/s) for the oracle."""
    import json
    import os
    with open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "workloads", "pn_b200.json")) as f:
        tab = json.load(f)["table"]
    n, tf = [int(r["n"]) for r in tab], [float(r["tflops"]) for r in tab]
    return (n, tf), (n, [int(round(t * 1000)) for t in tf])


@pytest.mark.parametrize("mode", [1, 2, "2+table"])
@pytest.mark.parametrize("name,n_atoms", [("cfg0", None), ("cfg2", 300), ("cfg3", 900)])
def test_combined_groups_bit_exact_and_parity(name, n_atoms, mode):
    """The library's greedy groups and union index sets equal the oracle's bit for bit; D and e_i of every member
    of the sampled groups match the oracle's group evaluation (one Eq. 8 on the union, columns of each member,
    rows restricted to N(member)) within the mixed-precision tolerances. "2+table": Eq. 10 with the measured,
    interpolated p(n) handed to both sides; 2: the tile-step fallback."""
    s = make_system(name, n_atoms=n_atoms)
    lib_table, orc_table = _measured_perf_table()
    with_table = mode == "2+table"
    mode = 2 if with_table else mode
    groups, sets = _oracle_groups(s, mode, perf_table=orc_table if with_table else None)
    if with_table and name == "cfg2":
        assert groups != _oracle_groups(s, 2)[0]                    # the measured table decides differently from the model
    nb, rp, ci, Hv, Sv = _arrays(s)
    blk = s.blk_off()
    Hn, Sn = s.fill_np(MAT_H), s.fill_np(MAT_S)
    with _nolsm(combine=mode) as ctx:
        if with_table:
            ctx.set_perf_table(*lib_table)
        ctx.assemble(nb, rp, ci, Hv, Sv)
        for g in groups:
            mem, st_, dim = ctx.group(g[0])
            union = np.unique(np.concatenate([sets[i] for i in g]))
            assert mem.tolist() == g and np.array_equal(st_, union.astype(np.int32))
            assert dim == int(s.atom_nb[union].sum())
        for i in (0, s.n_atoms - 1):
            N, d = ctx.index_set(i)
            assert np.array_equal(N, sets[i])                       # per-atom index sets are unchanged
        D = torch.zeros(Hv.shape[0], dtype=torch.float64, device="cuda")
        ctx.density_matrix(s.mu, D)
        E = ctx.energy()
        st = ctx.atom_stats()
        stats = ctx.stats()
    assert stats["n_units"] == len(groups) and (st["status"] == 0).all()
    assert int((st["dims"] > 0).sum()) == len(groups)
    Dh = D.cpu().numpy()
    rng = np.random.default_rng(11)
    pick = [groups[k] for k in rng.choice(len(groups), min(3, len(groups)), replace=False)]
    pick.append(max(groups, key=len))
    max_d, e_ref, e_gpu = 0.0, 0.0, 0.0
    from tests.helpers import d_row_from_oracle
    for g in pick:
        res = orc.group_result(g, s.atom_nb, s.row_ptr, s.col_idx, blk, Hn, Sn, s.mu)
        for i in g:
            row = d_row_from_oracle(s, i, res[i], blk)
            p0, p1 = int(s.row_ptr[i]), int(s.row_ptr[i + 1])
            max_d = max(max_d, float(np.abs(Dh[blk[p0]:blk[p1]] - row).max()))
            e_ref += res[i]["e_i"]
            e_gpu += float(st["e_atom"][i])
    print(name, "combine", mode, "groups", len(groups), "of", s.n_atoms, "max|dD|", max_d, "rel dE", abs(e_gpu - e_ref) / abs(e_ref),
          "dim mean", stats["dim_mean"], "gemms", stats["gemms_executed"])
    assert max_d <= TOL_MIXED_D
    assert abs(e_gpu - e_ref) / abs(e_ref) <= TOL_MIXED_E
    assert abs(E - st["e_atom"].sum()) <= 1e-9 * abs(E)


def test_combine_with_atom_ranges_and_round_engine(cfg0):
    """nolsm_density_matrix_range with combination: every group with a member in the range is evaluated and serves its
    members inside the range only - those rows equal the whole-system evaluation, all other rows stay untouched, and the
    range energy is the sum of the members' e_i. The round engine rejects combine."""
    from paper_2205_12182_b200 import ENGINE_ROUNDS, NolsmError
    s = cfg0
    nb, rp, ci, Hv, Sv = _arrays(s)
    blk = s.blk_off()
    with _nolsm(combine=1) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        D_all = torch.zeros(Hv.shape[0], dtype=torch.float64, device="cuda")
        ctx.density_matrix(s.mu, D_all)
        ctx.energy()
        e_all = ctx.atom_stats()["e_atom"]
        D = torch.full((Hv.shape[0],), 7.0, dtype=torch.float64, device="cuda")
        a0, a1 = 10, 30
        e_rng = ctx.density_matrix_range(s.mu, a0, a1, D, want_energy=True)
        e_at = ctx.atom_stats()["e_atom"]
    v0, v1 = int(blk[s.row_ptr[a0]]), int(blk[s.row_ptr[a1]])
    Dh, Dall = D.cpu().numpy(), D_all.cpu().numpy()
    assert (Dh[:v0] == 7.0).all() and (Dh[v1:] == 7.0).all()
    assert np.abs(Dh[v0:v1] - Dall[v0:v1]).max() <= 2e-3
    assert abs(e_rng - e_at[a0:a1].sum()) <= 1e-9 * abs(e_rng)
    assert abs(e_rng - e_all[a0:a1].sum()) <= TOL_MIXED_E * abs(e_rng)
    with _nolsm(combine=1, engine=ENGINE_ROUNDS) as ctx:
        with pytest.raises(NolsmError) as ei:
            ctx.assemble(nb, rp, ci, Hv, Sv)
        assert ei.value.code == 1


# ---- electron count and chemical-potential search ---------------------------------------
@pytest.mark.parametrize("combine", [0, 1])
def test_electron_count_matches_oracle(cfg0, combine):
    s = cfg0
    nb, rp, ci, Hv, Sv = _arrays(s)
    Hn, Sn = s.fill_np(MAT_H), s.fill_np(MAT_S)
    blk = s.blk_off()
    with _nolsm(combine=combine) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        D = torch.zeros(Hv.shape[0], dtype=torch.float64, device="cuda")
        for mu in (0.0, -1.2):
            ctx.density_matrix(mu, D)
            n_gpu, q = ctx.electron_count(per_atom=True)
            if combine:
                sets = [orc.index_set(i, s.row_ptr, s.col_idx) for i in range(s.n_atoms)]
                q_ref = np.zeros(s.n_atoms)
                for g in orc.combine_groups(s.atom_nb, sets, mode=1):
                    res = orc.group_result(g, s.atom_nb, s.row_ptr, s.col_idx, blk, Hn, Sn, mu)
                    for i in g:
                        q_ref[i] = res[i]["q_i"]
            else:
                q_ref = np.array([orc.atom_result(i, s.atom_nb, s.row_ptr, s.col_idx, blk, Hn, Sn, mu)["q_i"] for i in range(s.n_atoms)])
            print("electron count mu", mu, "combine", combine, n_gpu, q_ref.sum(), np.abs(q - q_ref).max())
            assert abs(n_gpu - q.sum()) <= 1e-9 * abs(n_gpu)
            assert abs(n_gpu - q_ref.sum()) <= TOL_MIXED_E * abs(q_ref.sum())
            assert np.abs(q - q_ref).max() <= 2e-2


def test_find_mu_reaches_the_target_count(cfg0):
    """Bisection through the C ABI: the returned mu gives the requested Tr(D S) within tol_n on the GPU, and the oracle's
    count at that mu agrees within the mixed-precision tolerance; D_vals holds D(mu)."""
    s = cfg0
    nb, rp, ci, Hv, Sv = _arrays(s)
    Hn, Sn = s.fill_np(MAT_H), s.fill_np(MAT_S)
    target = 0.5 * float(s.atom_nb.sum())
    with _nolsm() as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        D = torch.zeros(Hv.shape[0], dtype=torch.float64, device="cuda")
        mu, n_mu, evals = ctx.find_mu(target, -7.0, 8.0, D, tol_n=0.05, tol_mu=1e-4)
        E = ctx.energy()
        st = ctx.atom_stats()
        # evaluations: the two end points, then bisection of a bracket of 15 down to tol_mu = 1e-4 (log2(15 / 1e-4) = 17.2 ->
        # at most 18 trial mu) unless tol_n is met first, then the final density-matrix call: at most 21; the search also
        # stops at max_evals = 40 (the default), which this case must not reach
        assert abs(n_mu - target) <= 0.05 and 3 < evals <= 21 and -0.9 < mu < 0.9
        n_ref = orc.electron_count(s.atom_nb, s.row_ptr, s.col_idx, Hn, Sn, mu)
        assert abs(n_ref - n_mu) <= TOL_MIXED_E * target
        s_mu = make_system("cfg0")
        s_mu.mu = mu
        cmp = compare_atoms(s_mu, D.cpu().numpy(), st["e_atom"], range(0, s.n_atoms, 4))
        print("find_mu", mu, n_mu, evals, n_ref, cmp["max_abs_dD"], cmp["rel_dE"])
        assert cmp["max_abs_dD"] <= TOL_MIXED_D and cmp["rel_dE"] <= TOL_MIXED_E
        from paper_2205_12182_b200 import NolsmError
        with pytest.raises(NolsmError) as ei:                       # target above the number of basis functions
            ctx.find_mu(2.0 * float(s.atom_nb.sum()), -8.0, 8.0, D)
        assert ei.value.code == 1


def test_find_mu_with_three_trials_per_pass(cfg0):
    """nolsm_find_mu with options.mu_trials = 3 (bench.py runs it): three equidistant trial mu per pass on the resident
    S_sub^-1 and A0, the bracket shrinks by four per pass. The returned mu gives the requested Tr(D S) within tol_n, the
    oracle's count at that mu agrees within the mixed-precision tolerance, and D_vals holds D(mu)."""
    s = cfg0
    nb, rp, ci, Hv, Sv = _arrays(s)
    Hn, Sn = s.fill_np(MAT_H), s.fill_np(MAT_S)
    target = 0.5 * float(s.atom_nb.sum())
    with _nolsm(mu_trials=3) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        D = torch.zeros(Hv.shape[0], dtype=torch.float64, device="cuda")
        mu, n_mu, evals = ctx.find_mu(target, -7.0, 8.0, D, tol_n=0.05, tol_mu=1e-4)
        E = ctx.energy()
        st = ctx.atom_stats()
    # two end points, then passes of three trial mu (bracket / 4 each: log4(15 / 1e-4) = 8.6 -> at most 9 passes), the final call
    assert abs(n_mu - target) <= 0.05 and 3 < evals <= 2 + 3 * 9 + 1 and -0.9 < mu < 0.9
    n_ref = orc.electron_count(s.atom_nb, s.row_ptr, s.col_idx, Hn, Sn, mu)
    assert abs(n_ref - n_mu) <= TOL_MIXED_E * target
    s_mu = make_system("cfg0")
    s_mu.mu = mu
    cmp = compare_atoms(s_mu, D.cpu().numpy(), st["e_atom"], range(0, s.n_atoms, 4))
    print("find_mu K=3", mu, n_mu, evals, n_ref, cmp["max_abs_dD"], cmp["rel_dE"])
    assert cmp["max_abs_dD"] <= TOL_MIXED_D and cmp["rel_dE"] <= TOL_MIXED_E and abs(E - st["e_atom"].sum()) <= 1e-9 * abs(E)


@pytest.mark.parametrize("kw", [dict(combine=1, iteration=1), dict(combine=2, eps_filter=0.02), dict(combine=1, sign_scaled_iters=-1)])
def test_combination_with_other_options(kw):
    """Combination together with the symmetric (Loewdin) form, with the max-abs block filter (filtered index sets feed the
    grouping) and with plain Eq. 6: groups bit-exact, host float32 output, parity on sampled groups."""
    s = make_system("cfg1", n_atoms=500)
    Hn, Sn = s.fill_np(MAT_H), s.fill_np(MAT_S)
    blk = s.blk_off()
    eps = kw.get("eps_filter", 0.0)
    sets = [orc.index_set(i, s.row_ptr, s.col_idx, s.atom_nb, blk, Hn, Sn, eps) for i in range(s.n_atoms)]
    groups = orc.combine_groups(s.atom_nb, sets, mode=kw["combine"])
    from tests.helpers import d_row_from_oracle
    with _nolsm(**kw) as ctx:
        ctx.assemble(s.atom_nb, s.row_ptr, s.col_idx, Hn, Sn)                   # host inputs
        for g in groups[::7]:
            mem, st_, dim = ctx.group(g[0])
            assert mem.tolist() == g and np.array_equal(st_, np.unique(np.concatenate([sets[i] for i in g])).astype(np.int32))
        D = np.zeros(len(Hn), dtype=np.float32)                                  # host float32 output
        ctx.density_matrix(s.mu, D)
        E = ctx.energy()
        st = ctx.atom_stats()
        assert ctx.stats()["n_units"] == len(groups)
    max_d, e_ref, e_gpu = 0.0, 0.0, 0.0
    for g in groups[3::29]:
        res = orc.group_result(g, s.atom_nb, s.row_ptr, s.col_idx, blk, Hn, Sn, s.mu, eps_filter=eps)
        for i in g:
            row = d_row_from_oracle(s, i, res[i], blk)
            p0, p1 = int(s.row_ptr[i]), int(s.row_ptr[i + 1])
            max_d = max(max_d, float(np.abs(D[blk[p0]:blk[p1]] - row).max()))
            e_ref += res[i]["e_i"]
            e_gpu += float(st["e_atom"][i])
    print("options", kw, "groups", len(groups), "max|dD|", max_d, "rel dE", abs(e_gpu - e_ref) / abs(e_ref))
    assert max_d <= TOL_MIXED_D and abs(e_gpu - e_ref) / abs(e_ref) <= TOL_MIXED_E
    assert abs(E - st["e_atom"].sum()) <= 1e-9 * abs(E)


# ---- randomized shapes: basis sizes 1..16, submatrix dimensions around the tile boundaries -----------------------
def _random_system(rng, n_at, nb_choices, p_link):
    """Random symmetric pattern (diagonal set), random basis sizes, S = I + small symmetric, H0 symmetric with a gap."""
    atom_nb = rng.choice(nb_choices, n_at).astype(np.int32)
    pat = rng.random((n_at, n_at)) < p_link
    pat = np.triu(pat, 1)
    pat = pat | pat.T | np.eye(n_at, dtype=bool)
    first = np.concatenate([[0], np.cumsum(atom_nb)])
    N = int(first[-1])
    A = rng.normal(size=(N, N))
    H = 0.05 * (A + A.T)
    half = rng.random(N) < 0.5
    H[np.diag_indices(N)] = np.where(half, -1.0, 1.0) + 0.1 * rng.normal(size=N)
    B = rng.normal(size=(N, N))
    S = np.eye(N) + 0.004 * (B + B.T)
    row_ptr, col_idx, Hv, Sv = [0], [], [], []
    for i in range(n_at):
        for j in np.flatnonzero(pat[i]):
            col_idx.append(j)
            Hv.append(H[first[i]:first[i + 1], first[j]:first[j + 1]].reshape(-1))
            Sv.append(S[first[i]:first[i + 1], first[j]:first[j + 1]].reshape(-1))
        row_ptr.append(len(col_idx))
    return atom_nb, np.array(row_ptr, np.int64), np.array(col_idx, np.int32), np.concatenate(Hv), np.concatenate(Sv)


@pytest.mark.parametrize("seed,n_at,nbs,p_link,combine", [
    (0, 60, [1, 3, 5], 0.5, 0), (1, 90, [13, 16], 0.25, 0), (2, 70, [8, 16, 1], 0.6, 1),
    (3, 120, [5, 13], 0.35, 2), (4, 40, [16], 1.0, 0), (5, 150, [2, 7], 0.8, 1)])
def test_random_shapes_against_oracle(seed, n_at, nbs, p_link, combine):
    """Random patterns and basis sizes (1..16 functions per atom): submatrix dimensions from a few functions to ~1000,
    not multiples of 16, last row blocks on both sides of the half-height threshold, with and without combination."""
    rng = np.random.default_rng(100 + seed)
    atom_nb, rp, ci, Hv, Sv = _random_system(rng, n_at, nbs, p_link)
    blk = orc.block_offsets(atom_nb, rp, ci)
    with _nolsm(combine=combine) as ctx:
        ctx.assemble(atom_nb, rp, ci, Hv, Sv)
        D = np.zeros(len(Hv))
        ctx.density_matrix(0.0, D)
        E = ctx.energy()
        st = ctx.atom_stats()
        stats = ctx.stats()
    assert (st["status"] == 0).all()
    sets = [orc.index_set(i, rp, ci) for i in range(n_at)]
    groups = orc.combine_groups(atom_nb, sets, mode=combine) if combine else [[i] for i in range(n_at)]
    assert stats["n_units"] == len(groups)
    max_d, e_ref, e_gpu = 0.0, 0.0, 0.0
    for g in groups[::max(1, len(groups) // 12)]:
        res = orc.group_result(g, atom_nb, rp, ci, blk, Hv, Sv, 0.0)
        for i in g:
            p0, p1 = int(rp[i]), int(rp[i + 1])
            ref = np.zeros(int(blk[p1] - blk[p0]))
            cols = ci[p0:p1]
            for a, j in enumerate(res[i]["N"]):
                p = p0 + int(np.searchsorted(cols, j))
                ref[blk[p] - blk[p0]:blk[p + 1] - blk[p0]] = res[i]["Dcols"][res[i]["off"][a]:res[i]["off"][a + 1], :].T.reshape(-1)
            max_d = max(max_d, float(np.abs(D[blk[p0]:blk[p1]] - ref).max()))
            e_ref += res[i]["e_i"]
            e_gpu += float(st["e_atom"][i])
    print("random shapes", seed, "dims", stats["dim_min"], stats["dim_max"], "units", stats["n_units"], "max|dD|", max_d,
          "rel dE", abs(e_gpu - e_ref) / abs(e_ref))
    assert max_d <= TOL_MIXED_D
    assert abs(e_gpu - e_ref) <= TOL_MIXED_E * abs(e_ref)


def test_time_limit_abort_is_reported_by_the_next_wait_and_the_context_recovers():
    """options.timeout_s counts from the launch. A kernel that overruns it is stopped by the call that waits, and the abort is
    not forgotten when a later call on the context went through in the meantime (a series of density_matrix_range calls
    followed by one wait): the wait reports which call of the series was stopped. The context stays usable."""
    from paper_2205_12182_b200 import NolsmError
    s = make_system("cfg2", n_atoms=1200)
    nb, rp, ci, Hv, Sv = _arrays(s)
    D = torch.zeros_like(Hv)
    with _nolsm(timeout_s=0.05) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        ctx.density_matrix_range(s.mu, 0, 1000, D)             # > 100 ms of work: overruns the 50 ms
        ctx.density_matrix_range(s.mu, 1000, 1004, D)          # a few ms: runs to its end after the first was stopped
        with pytest.raises(NolsmError) as ei:
            ctx.energy()
        assert ei.value.code == 2 and "time limit" in str(ei.value) and "call 1 of the 2" in str(ei.value), str(ei.value)
        e = ctx.density_matrix_range(s.mu, 1000, 1004, D, want_energy=True)
        st = ctx.atom_stats()
        assert (st["status"][1000:1004] == 0).all() and abs(e - st["e_atom"][1000:1004].sum()) <= 1e-9 * abs(e)
    cmp = compare_atoms(s, D.cpu().numpy(), st["e_atom"], [1000, 1003])
    assert cmp["max_abs_dD"] <= TOL_MIXED_D and cmp["rel_dE"] <= TOL_MIXED_E


def test_pageable_host_output_arrives_with_the_wait(cfg0):
    """D_vals in pageable host memory is filled by the call that waits for the results (the watched wait comes first), in
    pinned host memory by a copy behind the kernel; both equal the device output of the same call within the tolerance."""
    s = cfg0
    nb, rp, ci, Hv, Sv = _arrays(s)
    with _nolsm() as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        Dd = torch.zeros_like(Hv)
        ctx.density_matrix(s.mu, Dd)
        e0 = ctx.energy()
        Dp = np.full(Hv.shape[0], np.nan)
        ctx.density_matrix(s.mu, Dp)
        e1 = ctx.energy()
        Dq = torch.full((Hv.shape[0],), float("nan"), dtype=torch.float64).pin_memory()
        ctx.density_matrix(s.mu, Dq)
        e2 = ctx.energy()
        Dr = np.full(Hv.shape[0], np.nan)
        ctx.density_matrix(s.mu, Dr)                           # never waited for explicitly: the next call delivers it
        ctx.density_matrix(s.mu, Dd)
        ctx.energy()
    ref = Dd.cpu().numpy()
    for got, e in ((Dp, e1), (Dq.numpy(), e2), (Dr, e0)):
        assert np.isfinite(got).all() and np.abs(got - ref).max() <= 2e-3 and abs(e - e0) <= 1e-4 * abs(e0)


def test_eigenvalue_outside_the_bulk_is_not_flipped_by_the_scaled_steps():
    """rho(A) comes from a few block power steps on a +-1 start block. One eigenvalue well outside a dense bulk (here 1.0
    against 1,507 eigenvalues of modulus 0.60-0.68) has weight 1 / n in that start: after the default six steps the estimate
    is 0.67 rho, the 1.25 safety leaves alpha x = 1.79 > sqrt(3), and the first scaled Newton-Schulz step would carry that
    eigenvalue to the other sign -- a wrong D with no status bit (one electron too many in the state built here, whose
    eigenvector is a single basis function: D_00 = 1 instead of 0). The power iteration goes on while its estimate is
    visibly not settled (growth rising from step to step), so D matches the oracle; the extra steps are counted."""
    rng = np.random.default_rng(11)
    n_at, nb = 116, 13
    n = n_at * nb
    lam = np.concatenate([[1.0], rng.uniform(0.60, 0.68, n - 1) * rng.choice([-1.0, 1.0], n - 1)])
    Q, _ = np.linalg.qr(rng.standard_normal((n - 1, n - 1)))
    H = np.zeros((n, n))
    H[0, 0] = lam[0]
    H[1:, 1:] = (Q * lam[1:]) @ Q.T
    H = 0.5 * (H + H.T)
    atom_nb = np.full(n_at, nb, dtype=np.int32)
    row_ptr = np.arange(n_at + 1, dtype=np.int64) * n_at
    col_idx = np.tile(np.arange(n_at, dtype=np.int32), n_at)
    blocks = lambda M: np.ascontiguousarray(M.reshape(n_at, nb, n_at, nb).transpose(0, 2, 1, 3)).reshape(-1)
    Hv, Sv = blocks(H), blocks(np.eye(n))
    D = torch.zeros(Hv.shape[0], dtype=torch.float64, device="cuda")
    with _nolsm() as ctx:
        ctx.assemble(torch.from_numpy(atom_nb).cuda(), torch.from_numpy(row_ptr).cuda(), torch.from_numpy(col_idx).cuda(),
                     torch.from_numpy(Hv).cuda(), torch.from_numpy(Sv).cuda())
        ctx.density_matrix(0.0, D)
        E = ctx.energy()
        n_elec = ctx.electron_count()
        st = ctx.atom_stats()
        extra = ctx.engine_counters()["power_steps_extra"]
    assert (st["status"] == 0).all()
    # full pattern: every submatrix is the whole matrix (P3), so the oracle is Eq. 5 on the dense matrices
    w, V = np.linalg.eigh(H)
    D_ref = (V[:, w < 0] @ V[:, w < 0].T)
    got = D.cpu().numpy().reshape(n_at, n_at, nb, nb).transpose(0, 2, 1, 3).reshape(n, n)     # slot (i, j) = (D_ji)^T: D^T = D
    print("outlier: extra power steps", extra, "max|dD|", np.abs(got - D_ref).max(), "D_00", got[0, 0], "Tr(DS)", n_elec, int((w < 0).sum()))
    assert abs(got[0, 0]) <= TOL_MIXED_D and np.abs(got - D_ref).max() <= TOL_MIXED_D
    assert abs(n_elec - (w < 0).sum()) <= 0.05
    assert abs(E - w[w < 0].sum()) <= TOL_MIXED_E * abs(w[w < 0].sum())
    assert extra >= n_at                                               # every submatrix needed more than the default steps
