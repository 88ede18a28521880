"""Pins for the FP64 oracle: the oracle is checked against what the paper and
the mathematics fix -- closed forms, invariants, textbook special cases, brute force -- never against
itself or against the CUDA path."""
import numpy as np
import pytest
import scipy.linalg as sla

from oracle import nolsm_oracle as orc
from workloads import MAT_H, MAT_S, make_system


def _rand_sym(n, rng, scale=1.0):
    A = rng.normal(size=(n, n)) * scale
    return 0.5 * (A + A.T)


def _rand_spd(n, rng, lo=0.3, hi=1.8):
    Q, _ = np.linalg.qr(rng.normal(size=(n, n)))
    return (Q * rng.uniform(lo, hi, n)) @ Q.T


@pytest.fixture(scope="module")
def cfg0():
    s = make_system("cfg0")
    return s, s.fill_np(MAT_H), s.fill_np(MAT_S)


# ---- P1, P2, P9: the sign function (Eq. 6-7 limit) ---------------------------------
def test_P1_sign_squared_is_identity():
    rng = np.random.default_rng(1)
    A = _rand_sym(40, rng)
    X = orc.sign_matrix(A)
    assert np.abs(X @ X - np.eye(40)).max() < 1e-10
    S, H = _rand_spd(40, rng), _rand_sym(40, rng)
    B = np.linalg.solve(S, H) - 0.1 * np.eye(40)          # non-symmetric, real spectrum
    Y = orc.sign_matrix(B)
    assert np.abs(Y @ Y - np.eye(40)).max() < 1e-9
    assert np.abs(Y @ B - B @ Y).max() < 1e-9              # sign(A) commutes with A


def test_P2_sign_of_diagonal():
    d = np.array([3.0, -0.2, 1e-3, -7.0, 0.0])
    assert np.array_equal(orc.sign_matrix(np.diag(d)), np.diag([1.0, -1.0, 1.0, -1.0, 0.0]))


def test_P9_sign_2x2_closed_form():
    a, b = 0.7, -1.9
    A = np.array([[a, b], [b, -a]])
    assert np.allclose(orc.sign_matrix(A), A / np.hypot(a, b), atol=1e-14)


def test_newton_schulz_iteration_reaches_the_oracle_sign():
    """Eq. 6 run literally in FP64 (X0 = A scaled into the convergence region) reaches sign_matrix."""
    rng = np.random.default_rng(2)
    S, H = _rand_spd(30, rng), _rand_sym(30, rng)
    A = np.linalg.solve(S, H) - 0.05 * np.eye(30)
    X = A / (1.01 * np.abs(np.linalg.eigvals(A)).max())
    for _ in range(60):
        X = 0.5 * X @ (3 * np.eye(30) - X @ X)
    assert np.abs(X - orc.sign_matrix(A)).max() < 1e-9


# ---- P5-P8: Eq. 5 ---------------------------------------------------------------------
def test_P5_P6_projector_invariants_and_band_energy():
    rng = np.random.default_rng(3)
    n, mu = 50, 0.13
    S, H = _rand_spd(n, rng), _rand_sym(n, rng)
    D, e, s = orc.density_eigh(H, S, mu)
    w = sla.eigh(H, S, eigvals_only=True)                    # textbook generalised eigenproblem
    assert np.allclose(np.sort(e), w, atol=1e-11)
    assert np.abs(D - D.T).max() < 1e-12
    assert np.abs(D @ S @ D - D).max() < 1e-11
    assert abs(np.trace(D @ S) - (w < mu).sum()) < 1e-10
    assert abs(np.trace(D @ H) - w[w < mu].sum()) < 1e-10    # P6: Tr(D H0) = sum of occupied eps


def test_density_eigh_equals_literal_eq5_and_textbook_sum():
    rng = np.random.default_rng(4)
    n, mu = 35, -0.2
    S, H = _rand_spd(n, rng), _rand_sym(n, rng)
    D, _, _ = orc.density_eigh(H, S, mu)
    assert np.abs(D - orc.density_literal(H, S, mu)).max() < 1e-9
    w, C = sla.eigh(H, S)                                     # H c = eps S c, c^T S c = 1
    Dtb = (C[:, w < mu]) @ (C[:, w < mu]).T
    assert np.abs(D - Dtb).max() < 1e-11


def test_P7_orthogonal_basis_is_plain_projector():
    rng = np.random.default_rng(5)
    H = _rand_sym(30, rng)
    D, _, _ = orc.density_eigh(H, np.eye(30), 0.0)
    w, V = np.linalg.eigh(H)
    P = V[:, w < 0] @ V[:, w < 0].T
    assert np.abs(D - P).max() < 1e-12
    assert np.abs(D @ D - D).max() < 1e-12


def test_P8_mu_outside_spectrum():
    rng = np.random.default_rng(6)
    S, H = _rand_spd(20, rng), _rand_sym(20, rng)
    w = sla.eigh(H, S, eigvals_only=True)
    D_lo, _, _ = orc.density_eigh(H, S, w[0] - 1.0)
    assert np.abs(D_lo).max() < 1e-13
    D_hi, _, _ = orc.density_eigh(H, S, w[-1] + 1.0)
    assert np.abs(D_hi - np.linalg.inv(S)).max() < 1e-10
    assert abs(np.trace(D_hi @ H) - np.trace(np.linalg.solve(S, H))) < 1e-10


def test_sign_zero_gives_half_occupation():
    D, _, _ = orc.density_eigh(np.diag([-1.0, 0.0, 2.0]), np.eye(3), 0.0)
    assert np.allclose(np.diag(D), [1.0, 0.5, 0.0])


def test_not_spd_is_reported():
    with pytest.raises(orc.NotSPDError):
        orc.density_eigh(np.eye(3), np.diag([1.0, -0.1, 1.0]), 0.0)


def test_P14_scaling_invariance():
    rng = np.random.default_rng(7)
    S, H = _rand_spd(25, rng), _rand_sym(25, rng)
    D1, _, _ = orc.density_eigh(H, S, 0.3)
    D2, _, _ = orc.density_eigh(2.5 * H, S, 2.5 * 0.3)
    assert np.abs(D1 - D2).max() < 1e-11
    assert abs(np.trace(D2 @ (2.5 * H)) - 2.5 * np.trace(D1 @ H)) < 1e-10


# ---- P3, P4, P12: the submatrix method ----------------------------------------------
def _dense_pattern_system(n_at, nb, rng, pattern):
    """Tiny block-CSR system with a given boolean atom-pattern (symmetric, diagonal set)."""
    atom_nb = np.full(n_at, nb, np.int32) if np.isscalar(nb) else np.asarray(nb, np.int32)
    first = np.concatenate([[0], np.cumsum(atom_nb)])
    N = int(first[-1])
    H = _rand_sym(N, rng)
    S = np.eye(N) + 0.08 * _rand_sym(N, rng)
    row_ptr, col_idx, Hv, Sv = [0], [], [], []
    for i in range(n_at):
        for j in range(n_at):
            if pattern[i, j]:
                col_idx.append(j)
                Hv.append(H[first[i]:first[i + 1], first[j]:first[j + 1]].reshape(-1))
                Sv.append(S[first[i]:first[i + 1], first[j]:first[j + 1]].reshape(-1))
        row_ptr.append(len(col_idx))
    mask = np.kron(pattern, np.ones((1, 1)))
    Hd = np.zeros_like(H)
    Sd = np.zeros_like(S)
    for i in range(n_at):
        for j in range(n_at):
            if pattern[i, j]:
                Hd[first[i]:first[i + 1], first[j]:first[j + 1]] = H[first[i]:first[i + 1], first[j]:first[j + 1]]
                Sd[first[i]:first[i + 1], first[j]:first[j + 1]] = S[first[i]:first[i + 1], first[j]:first[j + 1]]
    return (atom_nb, np.array(row_ptr, np.int64), np.array(col_idx, np.int32),
            np.concatenate(Hv), np.concatenate(Sv), Hd, Sd)


def test_P3_full_cutoff_equals_full_matrix_eq5():
    rng = np.random.default_rng(8)
    n_at = 7
    atom_nb, rp, ci, Hv, Sv, Hd, Sd = _dense_pattern_system(n_at, [2, 3, 1, 4, 2, 3, 2], rng,
                                                            np.ones((n_at, n_at), bool))
    mu = 0.1
    Dv, e_atom, info = orc.nolsm(atom_nb, rp, ci, Hv, Sv, mu)
    D_full = orc.density_literal(Hd, Sd, mu)
    D_sm = orc.dense_from_blocks(atom_nb, rp, ci, Dv, transpose_blocks=True)
    assert np.abs(D_sm - D_full).max() < 1e-9
    assert abs(e_atom.sum() - np.trace(D_full @ Hd)) < 1e-9
    assert all(len(info[i]["N"]) == n_at for i in range(n_at))


def test_P4_block_diagonal_cliques_are_exact():
    rng = np.random.default_rng(9)
    groups = [[0, 1, 2], [3, 4], [5, 6, 7, 8]]
    pat = np.zeros((9, 9), bool)
    for g in groups:
        pat[np.ix_(g, g)] = True
    atom_nb, rp, ci, Hv, Sv, Hd, Sd = _dense_pattern_system(9, 3, rng, pat)
    mu = -0.05
    Dv, e_atom, _ = orc.nolsm(atom_nb, rp, ci, Hv, Sv, mu)
    D_full = orc.density_literal(Hd, Sd, mu)
    assert np.abs(orc.dense_from_blocks(atom_nb, rp, ci, Dv, transpose_blocks=True) - D_full).max() < 1e-9
    assert abs(e_atom.sum() - np.trace(D_full @ Hd)) < 1e-9


def test_non_clique_pattern_is_only_approximate_and_keeps_input_sparsity():
    """A chain pattern (not a clique): the result differs from Eq. 5 on the full matrix (the method is
    an approximation) and D has exactly the input pattern (L60)."""
    rng = np.random.default_rng(10)
    n_at = 8
    pat = np.abs(np.subtract.outer(np.arange(n_at), np.arange(n_at))) <= 1
    atom_nb, rp, ci, Hv, Sv, Hd, Sd = _dense_pattern_system(n_at, 2, rng, pat)
    Dv, _, info = orc.nolsm(atom_nb, rp, ci, Hv, Sv, 0.0)
    assert len(Dv) == len(Hv)
    assert [list(info[i]["N"]) for i in (0, 3, 7)] == [[0, 1], [2, 3, 4], [6, 7]]
    D_full = orc.density_literal(Hd, Sd, 0.0)
    D_sm = orc.dense_from_blocks(atom_nb, rp, ci, Dv, transpose_blocks=True)
    err = np.abs(D_sm - D_full * np.kron(pat, np.ones((2, 2)))).max()
    assert 1e-6 < err < 0.5


def test_P12_identity_padding_is_exact():
    rng = np.random.default_rng(11)
    n, pad, mu = 21, 11, 0.2
    S, H = _rand_spd(n, rng), _rand_sym(n, rng)
    Sp = np.eye(n + pad)
    Sp[:n, :n] = S
    Hp = (mu + 1.0) * np.eye(n + pad)
    Hp[:n, :n] = H
    D, _, _ = orc.density_eigh(H, S, mu)
    Dp, _, _ = orc.density_eigh(Hp, Sp, mu)
    assert np.abs(Dp[:n, :n] - D).max() < 1e-12
    assert np.abs(Dp[n:, :]).max() < 1e-13


# ---- P10: an independent restatement of the iteration agrees with the eigen route --------------------
def test_P10_hotelling_plus_newton_schulz_agree_with_eigen_route(cfg0):
    s, Hv, Sv = cfg0
    blk = s.blk_off()
    res = orc.atom_result(17, s.atom_nb, s.row_ptr, s.col_idx, blk, Hv, Sv, s.mu)
    H, S, n = res["H_sub"], res["S_sub"], res["n"]
    I = np.eye(n)
    Y = I / np.linalg.norm(S, 2)
    for _ in range(40):                                       # Schulz 1933 (ref [14])
        Y = Y @ (2 * I - S @ Y)
    A = Y @ H - s.mu * I
    X = A / (1.01 * np.abs(np.linalg.eigvals(A)).max())
    for _ in range(80):                                       # Eq. 6
        X = 0.5 * X @ (3 * I - X @ X)
    D = 0.5 * (I - X) @ Y
    c0 = res["pos"]
    assert np.abs(D[:, c0:c0 + 4] - res["Dcols"]).max() < 1e-11
    assert abs((D[:, c0:c0 + 4] * H[:, c0:c0 + 4]).sum() - res["e_i"]) < 1e-11


# ---- P11: index sets ------------------------------------------------------------------------------------
def test_P11_index_sets_equal_brute_force_distance_scan(cfg0):
    s, _, _ = cfg0
    for i in range(s.n_atoms):
        d = np.sqrt(((s.pos - s.pos[i]) ** 2).sum(1))
        brute = np.flatnonzero((d < 6.0) | (np.arange(s.n_atoms) == i)).astype(np.int32)
        assert np.array_equal(orc.index_set(i, s.row_ptr, s.col_idx), brute)


def test_P11_relabelling_invariance(cfg0):
    s, Hv, Sv = cfg0
    sub_atoms = np.arange(0, 64, 2)                            # any sub-system, relabelled 0..31
    sub = s.restrict(sub_atoms)
    Hs, Ss = sub.fill_np(MAT_H), sub.fill_np(MAT_S)
    D1, e1, info1 = orc.nolsm(sub.atom_nb, sub.row_ptr, sub.col_idx, Hs, Ss, 0.0)
    perm = np.random.default_rng(12).permutation(sub.n_atoms)  # new id of old atom a is perm[a]
    inv = np.argsort(perm)
    # permuted block-CSR built by brute force
    first = np.concatenate([[0], np.cumsum(sub.atom_nb)])
    Hd = orc.dense_from_blocks(sub.atom_nb, sub.row_ptr, sub.col_idx, Hs)
    Sd = orc.dense_from_blocks(sub.atom_nb, sub.row_ptr, sub.col_idx, Ss)
    pat = np.zeros((sub.n_atoms, sub.n_atoms), bool)
    rows = sub.slot_rows()
    pat[perm[rows], perm[sub.col_idx]] = True
    rp, ci, Hp, Sp = [0], [], [], []
    for i in range(sub.n_atoms):
        for j in np.flatnonzero(pat[i]):
            a, b = inv[i], inv[j]
            ci.append(j)
            Hp.append(Hd[first[a]:first[a + 1], first[b]:first[b + 1]].reshape(-1))
            Sp.append(Sd[first[a]:first[a + 1], first[b]:first[b + 1]].reshape(-1))
        rp.append(len(ci))
    nbp = sub.atom_nb[inv]
    D2, e2, info2 = orc.nolsm(nbp, np.array(rp, np.int64), np.array(ci, np.int32),
                              np.concatenate(Hp), np.concatenate(Sp), 0.0)
    assert np.allclose(e2[perm], e1, atol=1e-12)
    for a in range(sub.n_atoms):
        assert np.array_equal(np.sort(perm[info1[a]["N"]]), info2[perm[a]]["N"])


def test_eps_filter_uses_max_abs_and_keeps_diagonal(cfg0):
    s, Hv, Sv = cfg0
    blk = s.blk_off()
    i = 5
    full = orc.index_set(i, s.row_ptr, s.col_idx)
    eps = 0.02
    expect = []
    for p in range(s.row_ptr[i], s.row_ptr[i + 1]):
        j = s.col_idx[p]
        m = max(np.abs(Hv[blk[p]:blk[p + 1]]).max(), np.abs(Sv[blk[p]:blk[p + 1]]).max())
        if j == i or m > eps:
            expect.append(j)
    got = orc.index_set(i, s.row_ptr, s.col_idx, s.atom_nb, blk, Hv, Sv, eps)
    assert list(got) == expect and i in got and len(got) < len(full)


# ---- P13: submatrix extraction ---------------------------------------------------------------------------
def test_P13_submatrix_is_the_principal_submatrix_of_the_dense_matrix(cfg0):
    s, Hv, Sv = cfg0
    blk = s.blk_off()
    Hd = orc.dense_from_blocks(s.atom_nb, s.row_ptr, s.col_idx, Hv)
    assert np.array_equal(Hd, Hd.T)
    for i in (0, 31, 63):
        N = orc.index_set(i, s.row_ptr, s.col_idx)
        T, off = orc.submatrix(N, s.atom_nb, s.row_ptr, s.col_idx, blk, Hv)
        idx = (N[:, None] * 4 + np.arange(4)).ravel()
        assert np.array_equal(T, Hd[np.ix_(idx, idx)])


def test_cfg0_whole_method_properties(cfg0):
    """Config 0 end to end: every S_sub is SPD (C-12 rescale), Tr(D_sub S_sub) is an integer
    (P5 per submatrix), and the result is close to (but not equal to) full-matrix Eq. 5."""
    s, Hv, Sv = cfg0
    Dv, e_atom, info = orc.nolsm(s.atom_nb, s.row_ptr, s.col_idx, Hv, Sv, s.mu)
    assert min(v["s_min"] for v in info.values()) >= 0.2 - 1e-9
    blk = s.blk_off()
    res = orc.atom_result(9, s.atom_nb, s.row_ptr, s.col_idx, blk, Hv, Sv, s.mu)
    t = np.trace(res["D_sub"] @ res["S_sub"])
    assert abs(t - round(t)) < 1e-9
    Hd = orc.dense_from_blocks(s.atom_nb, s.row_ptr, s.col_idx, Hv)
    Sd = orc.dense_from_blocks(s.atom_nb, s.row_ptr, s.col_idx, Sv)
    E_full = np.trace(orc.density_literal(Hd, Sd, s.mu) @ Hd)
    assert abs(e_atom.sum() - E_full) / abs(E_full) < 0.05
