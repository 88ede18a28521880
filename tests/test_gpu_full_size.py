"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default options,
device-resident FP64 block-CSR inputs generated with the torch filler): D and e_i are compared with the
FP64 oracle on seeded samples of atoms - valid because submatrix i depends only on H0/S restricted to N(i)
 - and properties that hold at any size are checked on everything (status words, zero rows
only for failed atoms, E = sum of e_i). Tolerances: BASELINE.json (mixed: max|dD| <= 2e-2, rel dE <= 1e-3)."""
import numpy as np
import pytest
import torch

from tests.helpers import compare_atoms
from workloads import MAT_H, MAT_S, make_system

pytestmark = pytest.mark.gpu

TOL_D, TOL_E = 2e-2, 1e-3


class _DeviceRows:
    """Indexable view of a device array that hands slices to the host (compare_atoms reads one row at a time)."""

    def __init__(self, t):
        self.t = t

    def __getitem__(self, sl):
        return self.t[sl].cpu().numpy()


def _device_inputs(s):
    dev = torch.device("cuda", 0)
    return (torch.from_numpy(s.atom_nb).to(dev), torch.from_numpy(s.row_ptr).to(dev), torch.from_numpy(s.col_idx).to(dev),
            s.fill_torch(MAT_H, dev), s.fill_torch(MAT_S, dev))


def _check_sample(s, D, e_atom, atoms, label):
    cmp = compare_atoms(s, _DeviceRows(D), e_atom, atoms)
    print(label, {k: v for k, v in cmp.items() if k != "ref"})
    assert cmp["max_abs_dD"] <= TOL_D
    assert cmp["rel_dE"] <= TOL_E
    return cmp


@pytest.mark.parametrize("name,sample", [("cfg1", 16), ("cfg2", 64), ("cfg3", 24)])
def test_full_config_sampled(name, sample):
    """configs[1], [2] (the headline config, 64 seeded-random atoms as BASELINE.json asks) and [3] (mixed 5/13
    basis, dims ~100-2000: ragged tiles in both directions, every slot size)."""
    from paper_2205_12182_b200 import Nolsm
    s = make_system(name)
    nb, rp, ci, Hv, Sv = _device_inputs(s)
    D = torch.empty_like(Hv)
    with Nolsm(0) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        ctx.density_matrix(s.mu, D)
        E = ctx.energy()
        st = ctx.atom_stats()
        stats = ctx.stats()
    assert (st["status"] == 0).all()
    assert stats["gemms_executed"] == int(st["gemms"].sum())
    assert abs(E - st["e_atom"].sum()) <= 1e-9 * abs(E)
    atoms = np.sort(np.random.default_rng(2024).choice(s.n_atoms, sample, replace=False))
    _check_sample(s, D, st["e_atom"], atoms, f"{name} full, {sample} atoms")
    # the extremes of the size distribution are always in the sample
    dims = st["dims"]
    _check_sample(s, D, st["e_atom"], [int(np.argmin(dims)), int(np.argmax(dims))], f"{name} full, smallest and largest")


def test_cfg4_streamed_in_atom_batches():
    """configs[4]: 262,144 atoms, block-CSR H0/S resident, D evaluated in atom batches with
    nolsm_density_matrix_range; the energy of every checked batch equals the sum of its e_i, D is compared
    with the oracle on 128 seeded-random atoms of the evaluated batches. (Four batches of 8,192 atoms are
    evaluated: first, last and two seeded ones - the whole system is throughput-only in BASELINE.json.)"""
    from paper_2205_12182_b200 import Nolsm
    s = make_system("cfg4")
    nb, rp, ci, Hv, Sv = _device_inputs(s)
    D = torch.full_like(Hv, 7.0)
    B = 8192
    nbatch = s.n_atoms // B
    rng = np.random.default_rng(4)
    batches = sorted({0, nbatch - 1, *rng.choice(nbatch, 2, replace=False).tolist()})
    blk = s.blk_off()
    with Nolsm(0) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        e_atom = np.zeros(s.n_atoms)
        for b in batches:
            a0, a1 = b * B, (b + 1) * B
            e_b = ctx.density_matrix_range(s.mu, a0, a1, D, want_energy=True)
            st = ctx.atom_stats(a0, B)
            assert (st["status"] == 0).all()
            assert abs(e_b - st["e_atom"].sum()) <= 1e-9 * abs(e_b)
            e_atom[a0:a1] = st["e_atom"]
    # rows outside the evaluated batches are untouched
    lo = int(blk[s.row_ptr[B]])
    hi = int(blk[s.row_ptr[batches[1] * B]])
    if hi > lo:
        assert bool((D[lo:min(hi, lo + (1 << 22))] == 7.0).all())
    pool = np.concatenate([np.arange(b * B, (b + 1) * B) for b in batches])
    atoms = np.sort(rng.choice(pool, 128, replace=False))
    _check_sample(s, D, e_atom, atoms, "cfg4, 128 atoms of 4 batches")


def test_cfg1_full_combined_groups_and_parity():
    """configs[1] at full size with submatrix combination (Eq. 9): the library's groups equal the oracle's greedy
    groups bit for bit over all 3,000 atoms; D and e_i of the members of sampled groups match the oracle."""
    from oracle import nolsm_oracle as orc
    from paper_2205_12182_b200 import Nolsm
    from tests.helpers import d_row_from_oracle
    s = make_system("cfg1")
    sets = [orc.index_set(i, s.row_ptr, s.col_idx) for i in range(s.n_atoms)]
    groups = orc.combine_groups(s.atom_nb, sets, mode=1)
    nb, rp, ci, Hv, Sv = _device_inputs(s)
    D = torch.empty_like(Hv)
    with Nolsm(0, combine=1) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        for g in groups:
            mem, st_, dim = ctx.group(g[0])
            assert mem.tolist() == g
            assert np.array_equal(st_, np.unique(np.concatenate([sets[i] for i in g])).astype(np.int32))
        ctx.density_matrix(s.mu, D)
        E = ctx.energy()
        st = ctx.atom_stats()
        stats = ctx.stats()
    assert stats["n_units"] == len(groups) < s.n_atoms // 2 and (st["status"] == 0).all()
    blk = s.blk_off()
    Hn, Sn = s.fill_np(MAT_H), s.fill_np(MAT_S)
    rows = _DeviceRows(D)
    rng = np.random.default_rng(7)
    max_d, e_ref, e_gpu = 0.0, 0.0, 0.0
    for k in rng.choice(len(groups), 6, replace=False):
        g = groups[int(k)]
        res = orc.group_result(g, s.atom_nb, s.row_ptr, s.col_idx, blk, Hn, Sn, s.mu)
        for i in g:
            ref = d_row_from_oracle(s, i, res[i], blk)
            p0, p1 = int(s.row_ptr[i]), int(s.row_ptr[i + 1])
            max_d = max(max_d, float(np.abs(rows[blk[p0]:blk[p1]] - ref).max()))
            e_ref += res[i]["e_i"]
            e_gpu += float(st["e_atom"][i])
    print("cfg1 full combined", len(groups), "groups, max|dD|", max_d, "rel dE", abs(e_gpu - e_ref) / abs(e_ref))
    assert max_d <= TOL_D and abs(e_gpu - e_ref) / abs(e_ref) <= TOL_E
    assert abs(E - st["e_atom"].sum()) <= 1e-9 * abs(E)


def test_large_dimension_submatrices():
    """Maximum sizes: the largest system of the p(n) sweep (`pn-14-8.5`: 14 functions per atom, cutoff 8.5 A, submatrices of
    ~3,600 dimensions = 15 x 15 tiles, 57 k-blocks per tile), the regime of the paper's largest submatrices after
    combination (Table II: thousands of dimensions). A range of atoms through nolsm_density_matrix_range, one of them
    against the oracle (a 3,600-dimensional generalised eigenproblem in FP64)."""
    from paper_2205_12182_b200 import Nolsm
    s = make_system("pn-14-8.5", n_atoms=1024)
    nb, rp, ci, Hv, Sv = _device_inputs(s)
    D = torch.zeros_like(Hv)
    a0, a1 = 100, 112
    with Nolsm(0) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        e = ctx.density_matrix_range(s.mu, a0, a1, D, want_energy=True)
        st = ctx.atom_stats()
        stats = ctx.stats()
    dims = st["dims"][a0:a1]
    print("large", dims.min(), dims.max(), stats["gemms_executed"] / (a1 - a0))
    assert dims.min() >= 3000
    assert (st["status"][a0:a1] == 0).all()
    assert abs(e - st["e_atom"][a0:a1].sum()) <= 1e-9 * abs(e)
    _check_sample(s, D, st["e_atom"], [a0 + 5], "pn-14-8.5, one atom of ~3600 dimensions")


# ---------------------------------------------------------------------------------------------------------------------
# The variants bench.py quotes on the full headline config (32,768 atoms): symmetric (Loewdin) form, Eq. 9 groups, Eq. 10
# groups with the measured p(n). The oracle sees the neighbourhoods of the sampled atoms / groups only (restrict), the
# library the whole system; groups are compared over ALL atoms (the oracle's grouping is integer work).
# ---------------------------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def cfg2_full():
    s = make_system("cfg2")
    return s, _device_inputs(s)


def test_cfg2_full_lowdin_form(cfg2_full):
    """configs[2] at full size in the symmetric form (C-21): twice the chains in flight, every
    product on the upper triangle of tiles with mirrored stores. 32 seeded atoms and the two extremes against the oracle."""
    from paper_2205_12182_b200 import ITER_LOWDIN, Nolsm
    s, (nb, rp, ci, Hv, Sv) = cfg2_full
    D = torch.empty_like(Hv)
    with Nolsm(0, iteration=ITER_LOWDIN) as ctx:
        ctx.assemble(nb, rp, ci, Hv, Sv)
        ctx.density_matrix(s.mu, D)
        E = ctx.energy()
        st = ctx.atom_stats()
        stats = ctx.stats()
    # every product of the form is symmetric except M = H0 Z (one per submatrix)
    assert (st["status"] == 0).all() and stats["gemms_symmetric"] == stats["gemms_executed"] - s.n_atoms > 0
    assert abs(E - st["e_atom"].sum()) <= 1e-9 * abs(E)
    atoms = np.sort(np.random.default_rng(52).choice(s.n_atoms, 32, replace=False))
    _check_sample(s, D, st["e_atom"], atoms, "cfg2 full, Loewdin form, 32 atoms")
    _check_sample(s, D, st["e_atom"], [int(np.argmin(st["dims"])), int(np.argmax(st["dims"]))], "cfg2 full, Loewdin form, extremes")


def _perf_table():
    import json
    import os
    with open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "workloads", "pn_b200.json")) as f:
        tab = json.load(f)["table"]
    n, tf = [int(r["n"]) for r in tab], [float(r["tflops"]) for r in tab]
    return (n, tf), (n, [int(round(x * 1000)) for x in tf])


@pytest.mark.parametrize("mode", [1, "2+table"])
def test_cfg2_full_combined_groups_and_parity(cfg2_full, mode):
    """configs[2] at full size with submatrix combination (Eq. 9; Eq. 10 with the measured and
    interpolated p(n), L89-91): the library's groups and union index sets equal the oracle's over all 32,768 atoms bit for
    bit; D and e_i of every member of six groups (the largest by dimension and five seeded ones) match the oracle's
    evaluation of Eq. 8 on the union set."""
    from oracle import nolsm_oracle as orc
    from paper_2205_12182_b200 import Nolsm
    from tests.helpers import d_row_from_oracle
    s, (nb, rp, ci, Hv, Sv) = cfg2_full
    lib_table, orc_table = _perf_table()
    sets = [orc.index_set(i, s.row_ptr, s.col_idx) for i in range(s.n_atoms)]
    groups = orc.combine_groups(s.atom_nb, sets, mode=1 if mode == 1 else 2, perf_table=None if mode == 1 else orc_table)
    D = torch.empty_like(Hv)
    with Nolsm(0, combine=1 if mode == 1 else 2) as ctx:
        if mode != 1:
            ctx.set_perf_table(*lib_table)
        ctx.assemble(nb, rp, ci, Hv, Sv)
        gdims = []
        for g in groups:
            mem, st_, dim = ctx.group(g[0])
            assert mem.tolist() == g
            assert np.array_equal(st_, np.unique(np.concatenate([sets[i] for i in g])).astype(np.int32))
            gdims.append(dim)
        ctx.density_matrix(s.mu, D)
        E = ctx.energy()
        st = ctx.atom_stats()
        stats = ctx.stats()
    assert stats["n_units"] == len(groups) < s.n_atoms // 2 and (st["status"] == 0).all()
    assert abs(E - st["e_atom"].sum()) <= 1e-9 * abs(E)
    blk = s.blk_off()
    rows = _DeviceRows(D)
    picks = {int(np.argmax(gdims)), *np.random.default_rng(9).choice(len(groups), 5, replace=False).tolist()}
    max_d, e_ref, e_gpu = 0.0, 0.0, 0.0
    for k in sorted(picks):
        g = groups[k]
        need = np.unique(np.concatenate([sets[i] for i in g]))
        sub = s.restrict(need)
        parent = sub.meta["parent_atoms"]
        sblk = orc.block_offsets(sub.atom_nb, sub.row_ptr, sub.col_idx)
        local = [int(np.searchsorted(parent, i)) for i in g]
        res = orc.group_result(local, sub.atom_nb, sub.row_ptr, sub.col_idx, sblk, sub.fill_np(MAT_H), sub.fill_np(MAT_S), s.mu)
        assert res["n"] == gdims[k]
        for i, li in zip(g, local):
            r = dict(res[li])
            r["N"] = parent[r["N"]].astype(np.int32)
            ref = d_row_from_oracle(s, i, r, blk)
            p0, p1 = int(s.row_ptr[i]), int(s.row_ptr[i + 1])
            max_d = max(max_d, float(np.abs(rows[blk[p0]:blk[p1]] - ref).max()))
            e_ref += r["e_i"]
            e_gpu += float(st["e_atom"][i])
    print("cfg2 full combined", mode, len(groups), "groups, largest", max(gdims), "max|dD|", max_d, "rel dE", abs(e_gpu - e_ref) / abs(e_ref))
    assert max_d <= TOL_D and abs(e_gpu - e_ref) / abs(e_ref) <= TOL_E
