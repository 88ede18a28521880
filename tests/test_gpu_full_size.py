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
