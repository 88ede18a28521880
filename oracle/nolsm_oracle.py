"""FP64 CPU oracle for the NOLSM hot path (arXiv 2205.12182).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this file. It shares no code with the CUDA path (paper_2205_12182_b200/), does not
import it, and takes plain numpy arrays.

What it computes (citations are PAPER.md line numbers):
  * submatrix method, steps 1-3 (L54-58) in its non-orthogonal form (L60): for every atom i,
    the retained rows/columns are the atoms j whose block (j, i) is present in the combined
    pattern of H0 and S; T_i(H0), T_i(S) are the dense principal submatrices on that set;
  * the per-submatrix matrix function Eq. 8 (L62)
        T_i(D) = 1/2 (I - sign(T_i(S)^-1 T_i(H0) - mu I)) T_i(S)^-1
    evaluated EXACTLY by symmetric eigendecomposition (the iterations of Eq. 6-7, converge
    to this; BASELINE.json north_star asks for the eigendecomposition route);
  * write-back of the columns of atom i (L58) and E_elec = Tr(D H0), Eq. 4 (L37).

Readings of silent points: structural pattern with
optional max-abs block filter (C-1), union pattern supplied by the caller (C-2), ascending atom
order inside a submatrix (C-3), one submatrix per atom (C-4), structurally symmetric pattern (C-5),
sign(0) = 0 (C-9), block (j,i) of D comes from submatrix i and is stored transposed in slot
(i,j) (C-10), no spin factor (C-11).

Parity pins: tests/test_oracle_pins.py (P1-P14 of SURVEY.md 8(c)). Parity with the paper's OWN
numbers is UNPINNED: PAPER.md prints no worked numerical example and Table II depends on the
spike-protein dataset, which is not available.
"""
from __future__ import annotations

import numpy as np


class NotSPDError(ValueError):
    """Raised when a submatrix of S is not positive definite (Eq. 8 undefined)."""


# ------------------------------------------------------------------------------------------
# step 1: index sets and dense submatrices
# ------------------------------------------------------------------------------------------
def block_offsets(atom_nb, row_ptr, col_idx):
    """Element offset of every block slot: slot s = (i, j) holds nb(i) x nb(j) values row-major."""
    rows = np.repeat(np.arange(len(atom_nb)), np.diff(np.asarray(row_ptr, dtype=np.int64)))
    size = np.asarray(atom_nb, dtype=np.int64)[rows] * np.asarray(atom_nb, dtype=np.int64)[col_idx]
    off = np.zeros(len(col_idx) + 1, dtype=np.int64)
    off[1:] = np.cumsum(size)
    return off


def index_set(i, row_ptr, col_idx, atom_nb=None, blk_off=None, H_vals=None, S_vals=None,
              eps_filter=0.0):
    """N(i): ascending atom ids j whose block (j, i) is non-negligible in column i (L56).

    The pattern is structurally symmetric (C-5), so column i is read from row i. With
    eps_filter > 0 a block is negligible iff max(|H0 block|_max, |S block|_max) <= eps_filter
    (C-1); the diagonal block is always kept."""
    out = []
    for p in range(int(row_ptr[i]), int(row_ptr[i + 1])):
        j = int(col_idx[p])
        keep = True
        if eps_filter > 0.0 and j != i:
            lo, hi = int(blk_off[p]), int(blk_off[p + 1])
            m = max(np.abs(H_vals[lo:hi]).max(), np.abs(S_vals[lo:hi]).max())
            keep = m > eps_filter
        if keep:
            out.append(j)
    if i not in out:
        raise ValueError(f"atom {i}: diagonal block missing from the pattern")
    out = np.array(sorted(out), dtype=np.int32)
    return out


def find_slot(j, k, row_ptr, col_idx):
    """Slot of block (j, k) or -1 (columns are ascending inside a row)."""
    lo, hi = int(row_ptr[j]), int(row_ptr[j + 1])
    p = lo + int(np.searchsorted(col_idx[lo:hi], k))
    return p if p < hi and col_idx[p] == k else -1


def submatrix(N_i, atom_nb, row_ptr, col_idx, blk_off, vals):
    """T_i(A): dense principal submatrix on the atoms N_i; absent blocks are zero (L56, L60)."""
    nb = [int(atom_nb[j]) for j in N_i]
    off = np.concatenate([[0], np.cumsum(nb)]).astype(np.int64)
    n = int(off[-1])
    T = np.zeros((n, n), dtype=np.float64)
    for a, j in enumerate(N_i):
        for b, k in enumerate(N_i):
            s = find_slot(int(j), int(k), row_ptr, col_idx)
            if s >= 0:
                T[off[a]:off[a + 1], off[b]:off[b + 1]] = \
                    np.asarray(vals[blk_off[s]:blk_off[s + 1]], dtype=np.float64).reshape(nb[a], nb[b])
    return T, off


# ------------------------------------------------------------------------------------------
# step 2 (Eq. 5, L62 Eq. 8): the matrix function
# ------------------------------------------------------------------------------------------
def sign_scalar(x):
    """sign with sign(0) = 0 (C-9)."""
    return np.sign(x)


def density_eigh(H, S, mu):
    """D = 1/2 (I - sign(S^-1 H - mu I)) S^-1 for symmetric H and SPD S, by two symmetric
    eigendecompositions.

    S = U s U^T, Z = U s^-1/2 U^T (= S^-1/2), Ht = Z H Z = V e V^T. S^-1 H = Z Ht Z^-1 is similar
    to Ht, so sign(S^-1 H - mu I) = Z sign(Ht - mu I) Z^-1 and
    D = Z 1/2(I - sign(Ht - mu I)) Z = (Z V) theta(e) (Z V)^T, theta(e) = 1/2 (1 - sign(e - mu)).
    Returns (D, e, s)."""
    s, U = np.linalg.eigh(S)
    if not s[0] > 0.0:
        raise NotSPDError(f"S not positive definite: lambda_min = {s[0]:.3e}")
    Z = (U / np.sqrt(s)) @ U.T
    Ht = Z @ H @ Z
    Ht = 0.5 * (Ht + Ht.T)
    e, V = np.linalg.eigh(Ht)
    theta = 0.5 * (1.0 - sign_scalar(e - mu))
    C = Z @ V
    D = (C * theta) @ C.T
    return D, e, s


def sign_matrix(A):
    """sign(A) for a diagonalisable A with real spectrum: A = P diag(l) P^-1 -> P diag(sign l) P^-1.
    This is the definition the Newton-Schulz iteration Eq. 6-7 (L47-50) converges to."""
    l, P = np.linalg.eig(A)
    if np.abs(l.imag).max() > 1e-8 * max(1.0, np.abs(l.real).max()):
        raise ValueError("spectrum is not real")
    X = (P * sign_scalar(l.real)) @ np.linalg.inv(P)
    return X.real


def density_literal(H, S, mu):
    """Eq. 5 written out literally with a general (non-symmetric) eigendecomposition for the sign."""
    n = len(H)
    Sinv = np.linalg.inv(S)
    A = Sinv @ H - mu * np.eye(n)
    return 0.5 * (np.eye(n) - sign_matrix(A)) @ Sinv


# ------------------------------------------------------------------------------------------
# step 3 + Eq. 4 (L37)
# ------------------------------------------------------------------------------------------
def atom_result(i, atom_nb, row_ptr, col_idx, blk_off, H_vals, S_vals, mu, eps_filter=0.0):
    """Everything submatrix i produces: index set, dims, D columns of atom i, energy partial.

    Returns dict(N=index set, n=dimension, pos=column offset of atom i inside the submatrix,
    Dcols = D_sub[:, cols(i)] (n x nb(i)), e_i = sum(Dcols * H_sub[:, cols(i)]),
    eps = generalised eigenvalues, s = eigenvalues of S_sub)."""
    N_i = index_set(i, row_ptr, col_idx, atom_nb, blk_off, H_vals, S_vals, eps_filter)
    H_sub, off = submatrix(N_i, atom_nb, row_ptr, col_idx, blk_off, H_vals)
    S_sub, _ = submatrix(N_i, atom_nb, row_ptr, col_idx, blk_off, S_vals)
    D_sub, eps, s = density_eigh(H_sub, S_sub, mu)
    a = int(np.searchsorted(N_i, i))
    c0, c1 = int(off[a]), int(off[a + 1])
    Dcols = D_sub[:, c0:c1].copy()
    e_i = float((Dcols * H_sub[:, c0:c1]).sum())
    q_i = float((Dcols * S_sub[:, c0:c1]).sum())           # atom i's share of Tr(D S), the electron count (L149)
    return dict(N=N_i, n=int(off[-1]), pos=c0, off=off, Dcols=Dcols, e_i=e_i, q_i=q_i, eps=eps, s=s,
                H_sub=H_sub, S_sub=S_sub, D_sub=D_sub)


def scatter_atom(i, res, atom_nb, row_ptr, col_idx, blk_off, D_vals):
    """Write block (j, i) of D for all j in N(i) (L58). Storage (C-10): the output uses the input
    pattern and slot (i, j) holds (D_ji)^T, i.e. the array is D^T in block-CSR; blocks of the
    pattern that the filter dropped stay zero."""
    nbi = int(atom_nb[i])
    for a, j in enumerate(res["N"]):
        s = find_slot(i, int(j), row_ptr, col_idx)
        Dji = res["Dcols"][res["off"][a]:res["off"][a + 1], :]          # nb(j) x nb(i)
        D_vals[blk_off[s]:blk_off[s + 1]] = Dji.T.reshape(-1)
    return D_vals


def nolsm(atom_nb, row_ptr, col_idx, H_vals, S_vals, mu, atoms=None, eps_filter=0.0):
    """The whole path for all (or the listed) atoms.

    Returns (D_vals, e_atom, info): D_vals float64 in the C-10 layout (zero for atoms not
    listed), e_atom float64[n_atoms] energy partials (E_elec = e_atom.sum() when all atoms are
    evaluated), info = per-atom dict(N, n, min_gap)."""
    n_at = len(atom_nb)
    blk_off = block_offsets(atom_nb, row_ptr, col_idx)
    D_vals = np.zeros(int(blk_off[-1]), dtype=np.float64)
    e_atom = np.zeros(n_at, dtype=np.float64)
    info = {}
    for i in (range(n_at) if atoms is None else atoms):
        i = int(i)
        res = atom_result(i, atom_nb, row_ptr, col_idx, blk_off, H_vals, S_vals, mu, eps_filter)
        scatter_atom(i, res, atom_nb, row_ptr, col_idx, blk_off, D_vals)
        e_atom[i] = res["e_i"]
        info[i] = dict(N=res["N"], n=res["n"], min_gap=float(np.abs(res["eps"] - mu).min()),
                       s_min=float(res["s"][0]), s_max=float(res["s"][-1]),
                       eps_min=float(res["eps"][0]), eps_max=float(res["eps"][-1]))
    return D_vals, e_atom, info


# ------------------------------------------------------------------------------------------
# full-matrix helpers used by the pins (dense, small systems only)
# ------------------------------------------------------------------------------------------
def dense_from_blocks(atom_nb, row_ptr, col_idx, vals, transpose_blocks=False):
    """Dense N x N matrix from block-CSR values. With transpose_blocks=True the array is read in
    the C-10 output layout (slot (i,j) holds (M_ji)^T) and the dense M is returned."""
    blk_off = block_offsets(atom_nb, row_ptr, col_idx)
    first = np.concatenate([[0], np.cumsum(atom_nb)]).astype(np.int64)
    M = np.zeros((int(first[-1]), int(first[-1])), dtype=np.float64)
    s = 0
    for i in range(len(atom_nb)):
        for p in range(int(row_ptr[i]), int(row_ptr[i + 1])):
            j = int(col_idx[p])
            blk = np.asarray(vals[blk_off[s]:blk_off[s + 1]], dtype=np.float64).reshape(
                int(atom_nb[i]), int(atom_nb[j]))
            if transpose_blocks:
                M[first[j]:first[j + 1], first[i]:first[i + 1]] = blk.T
            else:
                M[first[i]:first[i + 1], first[j]:first[j + 1]] = blk
            s += 1
    return M


# ------------------------------------------------------------------------------------------
# submatrix combination ("one submatrix for multiple columns", Eq. 9 / Eq. 10)
# ------------------------------------------------------------------------------------------
def perf_rate(perf_table, n):
    """r(n) of Eq. 10 (L89: "the matrix multiplication performance p(n) of the GPUs is measured for different matrix
    sizes n and interpolated"): perf_table = (dimensions ascending, rates in integer GFLOP/s); linear interpolation
    between neighbouring points, constant outside the table, in integers (floor division of non-negative numbers)."""
    tn, tr = perf_table
    n = int(n)
    if n <= tn[0]:
        return int(tr[0])
    if n >= tn[-1]:
        return int(tr[-1])
    k = 0
    while tn[k + 1] <= n:
        k += 1
    return (int(tr[k]) * (int(tn[k + 1]) - n) + int(tr[k + 1]) * (n - int(tn[k]))) // (int(tn[k + 1]) - int(tn[k]))


def combine_cost(n, mode, perf_table=None):
    """What the evaluation of a submatrix of dimension n costs in the combination criterion.
    mode 1, Eq. 9 (L87): n^3, the FLOP count of a dense multiplication. mode 2, Eq. 10 (L91): the predicted runtime
    "p(n) x n^3" with the measured performance characteristic of the GPU, i.e. n^3 / r(n) for a measured rate r(n)
    (perf_rate), scaled by 10^6 and floored so that everything stays an integer. Without a table mode 2 falls back to
    a model of the B200 engine, the number of 256 x 256 x 64 tile steps of a multiplication,
    ceil(n16/256)^2 ceil(n16/64) with n16 = n rounded up to 16 (C-19)."""
    n = int(n)
    if mode == 1:
        return n * n * n
    if perf_table is not None:
        return 10 ** 6 * n * n * n // perf_rate(perf_table, n)
    n16 = (n + 15) // 16 * 16
    t = (n16 + 255) // 256
    return t * t * ((n16 + 63) // 64)


def predicted_seconds(flop, rate_flops):
    """Predicted runtime of `flop` floating-point operations at a measured rate (FLOP/s): flop / rate. This is the reading
    of Eq. 10's "predicted runtime p(n) x n^3" (L89-91) that Table II (L119-126) fixes: its "estimated speedup" column is
    (FLOP count / estimated performance) of the uncombined set over that of the combined set (C-19)."""
    return float(flop) / float(rate_flops)


def estimated_performance(dims, perf_table):
    """Table II's "estimated performance" of a set of submatrices for one multiplication each: total FLOP (2 n^3, L156)
    over total predicted runtime, sum 2 n^3 / sum (2 n^3 / r(n)), in the unit of the table's rates."""
    flop = sum(2.0 * float(n) ** 3 for n in dims)
    sec = sum(predicted_seconds(2.0 * float(n) ** 3, perf_rate(perf_table, n)) for n in dims)
    return flop / sec


def combine_groups(atom_nb, index_sets, mode=1, max_dim=2048, max_members=16, max_candidates=24, perf_table=None):
    """Greedy combination of columns (atoms) into groups that share ONE submatrix (C-19).

    Atoms are visited in ascending id. An atom i that is still free seeds a group G = N(i). Its
    candidates are the free atoms j of N(i), ordered by the overlap dim(N(i) & N(j)) (descending,
    ties by id), the first max_candidates of them. A candidate joins iff the criterion of Eq. 9
    (mode 1) or Eq. 10 (mode 2) holds for the group as it stands,
        cost(n_G + n_j - n_{G & j}) < cost(n_G) + cost(n_j),
    and the union stays within max_dim; then G <- G | N(j). All quantities are integers. perf_table: the measured
    (dimensions, GFLOP/s) of Eq. 10 (perf_rate).
    Returns the list of groups (member lists in joining order, seed first)."""
    nb = np.asarray(atom_nb, dtype=np.int64)
    n_at = len(nb)
    dim = [int(nb[N].sum()) for N in index_sets]
    free = np.ones(n_at, dtype=bool)
    groups = []
    for i in range(n_at):
        if not free[i]:
            continue
        free[i] = False
        members = [i]
        if max_members > 1 and mode in (1, 2):
            Ni = np.asarray(index_sets[i])
            G = Ni
            n_g = dim[i]
            cand = []
            for j in Ni:
                j = int(j)
                if j != i and free[j]:
                    ov = int(nb[np.intersect1d(Ni, index_sets[j], assume_unique=True)].sum())
                    cand.append((-ov, j))
            cand.sort()
            for _, j in cand[:max_candidates]:
                if len(members) >= max_members:
                    break
                n_gj = int(nb[np.intersect1d(G, index_sets[j], assume_unique=True)].sum())
                n_u = n_g + dim[j] - n_gj
                if n_u > max_dim:
                    continue
                if combine_cost(n_u, mode, perf_table) < combine_cost(n_g, mode, perf_table) + combine_cost(dim[j], mode, perf_table):
                    members.append(j)
                    free[j] = False
                    G = np.union1d(G, index_sets[j])
                    n_g = n_u
        groups.append(members)
    return groups


def group_result(members, atom_nb, row_ptr, col_idx, blk_off, H_vals, S_vals, mu, eps_filter=0.0):
    """One submatrix for several columns (L65): the index set of the group is the union of its members'
    index sets, Eq. 8 is evaluated once on it, and every member i takes its own columns, restricted to the
    rows j in N(i) - the blocks (j, i) that exist in the pattern of the result (L58, L60).
    Returns {i: dict like atom_result(i)} plus key "G" (the union) and "n" (its dimension)."""
    sets = {int(i): index_set(int(i), row_ptr, col_idx, atom_nb, blk_off, H_vals, S_vals, eps_filter) for i in members}
    G = np.unique(np.concatenate(list(sets.values())))
    H_G, off_G = submatrix(G, atom_nb, row_ptr, col_idx, blk_off, H_vals)
    S_G, _ = submatrix(G, atom_nb, row_ptr, col_idx, blk_off, S_vals)
    D_G, eps, s = density_eigh(H_G, S_G, mu)
    out = {"G": G, "n": int(off_G[-1])}
    for i, N_i in sets.items():
        a_i = int(np.searchsorted(G, i))
        c0, c1 = int(off_G[a_i]), int(off_G[a_i + 1])
        rows = np.concatenate([np.arange(off_G[a], off_G[a + 1]) for a in np.searchsorted(G, N_i)])
        Dcols = D_G[np.ix_(rows, np.arange(c0, c1))].copy()
        off = np.zeros(len(N_i) + 1, dtype=np.int64)
        off[1:] = np.cumsum(np.asarray(atom_nb, dtype=np.int64)[N_i])
        e_i = float((Dcols * H_G[np.ix_(rows, np.arange(c0, c1))]).sum())
        q_i = float((Dcols * S_G[np.ix_(rows, np.arange(c0, c1))]).sum())
        out[i] = dict(N=N_i, n=int(off[-1]), off=off, Dcols=Dcols, e_i=e_i, q_i=q_i, eps=eps, s=s, n_group=int(off_G[-1]))
    return out


# ------------------------------------------------------------------------------------------
# chemical potential: mu is iterated until the electron count Tr(D S) is right
# ------------------------------------------------------------------------------------------
def electron_count(atom_nb, row_ptr, col_idx, H_vals, S_vals, mu, atoms=None):
    """Tr(D(mu) S) of the submatrix method: sum over atoms i of q_i = sum_{j in N(i)} <D_ji, S_ji>."""
    blk_off = block_offsets(atom_nb, row_ptr, col_idx)
    q = 0.0
    for i in (range(len(atom_nb)) if atoms is None else atoms):
        q += atom_result(int(i), atom_nb, row_ptr, col_idx, blk_off, H_vals, S_vals, mu)["q_i"]
    return q


def find_mu(count, n_target, mu_lo, mu_hi, tol_n=1e-3, tol_mu=1e-6, max_evals=40):
    """Bisection on mu for count(mu) = n_target; count never decreases with mu (every generalised eigenvalue of
    every submatrix that drops below mu adds a non-negative share). Returns (mu, count(mu), evaluations)."""
    n_lo, n_hi = count(mu_lo), count(mu_hi)
    evals = 2
    if n_lo - tol_n > n_target or n_hi + tol_n < n_target:
        raise ValueError("electron count not bracketed")
    mu, n_mu = mu_hi, n_hi
    while evals < max_evals and abs(n_mu - n_target) > tol_n and (mu_hi - mu_lo) > tol_mu:
        mu = 0.5 * (mu_lo + mu_hi)
        n_mu = count(mu)
        evals += 1
        if n_mu < n_target:
            mu_lo = mu
        else:
            mu_hi = mu
    return mu, n_mu, evals
