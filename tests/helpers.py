"""Shared helpers of the parity tests: run the CUDA path through the C-ABI binding, run the oracle on
(sampled) atoms, and compare in the output layout of include/nolsm.h."""
import numpy as np

from oracle import nolsm_oracle as orc
from workloads import MAT_H, MAT_S


def oracle_on_atoms(system, atoms):
    """Oracle results for the listed atoms of `system`, evaluated on the restriction of the system to
    the union of their index sets (a submatrix depends only on H0/S restricted to N(i)).
    Returns {atom: dict(N=index set in parent ids, Dcols, e_i, n, slots=parent slot ids of row i)}."""
    atoms = [int(a) for a in atoms]
    need = np.unique(np.concatenate([system.col_idx[system.row_ptr[a]:system.row_ptr[a + 1]] for a in atoms]))
    sub = system.restrict(need)
    Hs, Ss = sub.fill_np(MAT_H), sub.fill_np(MAT_S)
    blk = orc.block_offsets(sub.atom_nb, sub.row_ptr, sub.col_idx)
    parent_atoms = sub.meta["parent_atoms"]
    out = {}
    for a in atoms:
        la = int(np.searchsorted(parent_atoms, a))
        res = orc.atom_result(la, sub.atom_nb, sub.row_ptr, sub.col_idx, blk, Hs, Ss, system.mu)
        res["N"] = parent_atoms[res["N"]].astype(np.int32)
        out[a] = res
    return out


def d_row_from_oracle(system, atom, res, blk_off):
    """The values of row `atom` of the output array (slot (i,j) = (D_ji)^T) from an oracle result."""
    nbi = int(system.atom_nb[atom])
    p0, p1 = int(system.row_ptr[atom]), int(system.row_ptr[atom + 1])
    row = np.zeros(int(blk_off[p1] - blk_off[p0]))
    cols = system.col_idx[p0:p1]
    for a, j in enumerate(res["N"]):
        p = p0 + int(np.searchsorted(cols, j))
        Dji = res["Dcols"][res["off"][a]:res["off"][a + 1], :]
        row[blk_off[p] - blk_off[p0]:blk_off[p + 1] - blk_off[p0]] = Dji.T.reshape(-1)
    return row


def compare_atoms(system, D_gpu, e_gpu_atoms, atoms, blk_off=None):
    """max |dD| over the sampled atoms' rows and relative error of sum e_i over the sample."""
    blk_off = system.blk_off() if blk_off is None else blk_off
    ref = oracle_on_atoms(system, atoms)
    max_d, e_ref, e_gpu, min_gap = 0.0, 0.0, 0.0, np.inf
    for a in atoms:
        a = int(a)
        row = d_row_from_oracle(system, a, ref[a], blk_off)
        p0, p1 = int(system.row_ptr[a]), int(system.row_ptr[a + 1])
        got = np.asarray(D_gpu[blk_off[p0]:blk_off[p1]], dtype=np.float64)
        max_d = max(max_d, float(np.abs(got - row).max()))
        e_ref += ref[a]["e_i"]
        e_gpu += float(e_gpu_atoms[a])
        min_gap = min(min_gap, float(np.abs(ref[a]["eps"] - system.mu).min()))
    return dict(max_abs_dD=max_d, rel_dE=abs(e_gpu - e_ref) / abs(e_ref), e_ref=e_ref, e_gpu=e_gpu, min_gap=min_gap,
                ref=ref)
