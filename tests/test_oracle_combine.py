"""Pins for the oracle's submatrix combination (Eq. 9 / Eq. 10; C-19): the
grouping is checked against the paper's criterion by brute force with Python sets, and the group evaluation
against the cases where the method is exact (full cutoff, block-diagonal cliques), against the single-column
method, and against Eq. 5 on the full matrix."""
import numpy as np

from oracle import nolsm_oracle as orc
from tests.test_oracle_pins import _dense_pattern_system
from workloads import MAT_H, MAT_S, make_system


def _sets(s):
    return [orc.index_set(i, s.row_ptr, s.col_idx) for i in range(s.n_atoms)]


def test_cost_functions():
    assert orc.combine_cost(10, 1) == 1000 and orc.combine_cost(543, 1) == 543 ** 3
    # tile-time model: 256 x 256 tiles, 64-deep k-blocks, dimension rounded up to 16
    assert orc.combine_cost(256, 2) == 1 * 1 * 4
    assert orc.combine_cost(257, 2) == 2 * 2 * 5          # 272 -> 2 x 2 tiles, 5 k-blocks
    assert orc.combine_cost(1184, 2) == 5 * 5 * 19
    assert all(orc.combine_cost(n + 1, m) >= orc.combine_cost(n, m) for n in range(1, 1500, 7) for m in (1, 2))


def test_groups_partition_the_atoms_and_obey_the_criterion_brute_force():
    """Replays every group with Python sets: members are free neighbours of the seed, each accepted merge
    satisfies Eq. 9 for the group as it stood ((n_G + n_j - n_Gj)^3 < n_G^3 + n_j^3, L87), the union stays
    within max_dim, and every candidate that was passed over violates the criterion (or a cap)."""
    s = make_system("cfg1", n_atoms=300)
    sets = _sets(s)
    nb = s.atom_nb.astype(int)
    pysets = [set(int(x) for x in N) for N in sets]
    dim = lambda A: sum(nb[a] for a in A)
    for mode in (1, 2):
        groups = orc.combine_groups(s.atom_nb, sets, mode=mode, max_dim=900, max_members=5, max_candidates=10)
        flat = sorted(a for g in groups for a in g)
        assert flat == list(range(s.n_atoms))                       # a partition
        assert [g[0] for g in groups] == sorted(g[0] for g in groups)   # seeds in ascending order
        free = set(range(s.n_atoms))
        n_merged = 0
        for g in groups:
            seed = g[0]
            assert seed == min(free)                                 # the smallest free atom seeds the next group
            free.discard(seed)
            cand = sorted((-dim(pysets[seed] & pysets[j]), j) for j in pysets[seed] if j != seed and j in free)[:10]
            G, members = set(pysets[seed]), [seed]
            for _, j in cand:
                if len(members) >= 5:
                    break
                n_u = dim(G | pysets[j])
                ok = n_u <= 900 and orc.combine_cost(n_u, mode) < orc.combine_cost(dim(G), mode) + orc.combine_cost(dim(pysets[j]), mode)
                if ok:
                    members.append(j)
                    free.discard(j)
                    G |= pysets[j]
            assert members == g
            n_merged += len(g) > 1
        assert n_merged > 10


def test_single_member_groups_equal_the_single_column_method():
    s = make_system("cfg0")
    Hv, Sv = s.fill_np(MAT_H), s.fill_np(MAT_S)
    blk = s.blk_off()
    groups = orc.combine_groups(s.atom_nb, _sets(s), mode=1, max_members=1)
    assert groups == [[i] for i in range(s.n_atoms)]
    for i in (0, 17, 63):
        a = orc.atom_result(i, s.atom_nb, s.row_ptr, s.col_idx, blk, Hv, Sv, s.mu)
        g = orc.group_result([i], s.atom_nb, s.row_ptr, s.col_idx, blk, Hv, Sv, s.mu)[i]
        assert np.array_equal(a["N"], g["N"]) and np.abs(a["Dcols"] - g["Dcols"]).max() < 1e-13
        assert abs(a["e_i"] - g["e_i"]) < 1e-12


def test_full_cutoff_groups_are_exact():
    """Every N(i) is the whole system: any grouping evaluates Eq. 5 on the full matrix (L56)."""
    rng = np.random.default_rng(21)
    n_at = 6
    atom_nb, rp, ci, Hv, Sv, Hd, Sd = _dense_pattern_system(n_at, [2, 3, 1, 4, 2, 3], rng, np.ones((n_at, n_at), bool))
    blk = orc.block_offsets(atom_nb, rp, ci)
    D_full = orc.density_literal(Hd, Sd, 0.1)
    sets = [orc.index_set(i, rp, ci) for i in range(n_at)]
    groups = orc.combine_groups(atom_nb, sets, mode=1)
    assert groups == [list(range(n_at))]                              # n_u = n: n^3 < 2 n^3 always merges
    first = np.concatenate([[0], np.cumsum(atom_nb)])
    res = orc.group_result(groups[0], atom_nb, rp, ci, blk, Hv, Sv, 0.1)
    e = 0.0
    for i in range(n_at):
        assert np.abs(res[i]["Dcols"] - D_full[:, first[i]:first[i + 1]]).max() < 1e-9
        e += res[i]["e_i"]
    assert abs(e - np.trace(D_full @ Hd)) < 1e-9


def test_block_diagonal_cliques_are_exact_when_combined():
    rng = np.random.default_rng(22)
    cl = [[0, 1, 2], [3, 4], [5, 6, 7, 8]]
    pat = np.zeros((9, 9), bool)
    for g in cl:
        pat[np.ix_(g, g)] = True
    atom_nb, rp, ci, Hv, Sv, Hd, Sd = _dense_pattern_system(9, 3, rng, pat)
    blk = orc.block_offsets(atom_nb, rp, ci)
    groups = orc.combine_groups(atom_nb, [orc.index_set(i, rp, ci) for i in range(9)], mode=1)
    assert [sorted(g) for g in groups] == cl
    D_full = orc.density_literal(Hd, Sd, -0.05)
    for g in groups:
        res = orc.group_result(g, atom_nb, rp, ci, blk, Hv, Sv, -0.05)
        for i in g:
            rows = np.concatenate([np.arange(3 * j, 3 * j + 3) for j in res[i]["N"]])
            assert np.abs(res[i]["Dcols"] - D_full[np.ix_(rows, np.arange(3 * i, 3 * i + 3))]).max() < 1e-9


def test_combination_is_at_least_as_close_to_full_eq5_on_cfg0():
    """L65: generating one submatrix for multiple columns improves efficiency AND accuracy - a member's columns
    come from a superset of its own index set. Checked on config 0 against Eq. 5 on the full 256 x 256 matrices."""
    s = make_system("cfg0")
    Hv, Sv = s.fill_np(MAT_H), s.fill_np(MAT_S)
    blk = s.blk_off()
    Hd = orc.dense_from_blocks(s.atom_nb, s.row_ptr, s.col_idx, Hv)
    Sd = orc.dense_from_blocks(s.atom_nb, s.row_ptr, s.col_idx, Sv)
    D_full = orc.density_literal(Hd, Sd, s.mu)
    first = np.concatenate([[0], np.cumsum(s.atom_nb)])
    groups = orc.combine_groups(s.atom_nb, _sets(s), mode=1)
    assert len(groups) < s.n_atoms // 2
    err_single = err_comb = 0.0
    for g in groups:
        res = orc.group_result(g, s.atom_nb, s.row_ptr, s.col_idx, blk, Hv, Sv, s.mu)
        for i in g:
            one = orc.atom_result(i, s.atom_nb, s.row_ptr, s.col_idx, blk, Hv, Sv, s.mu)
            rows = np.concatenate([np.arange(first[j], first[j + 1]) for j in one["N"]])
            ref = D_full[np.ix_(rows, np.arange(first[i], first[i + 1]))]
            err_single += float(((one["Dcols"] - ref) ** 2).sum())
            err_comb += float(((res[i]["Dcols"] - ref) ** 2).sum())
    assert err_comb < err_single
