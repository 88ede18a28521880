"""Pins for the oracle's electron count Tr(D S) and chemical-potential search."""
import numpy as np
import scipy.linalg as sla

from oracle import nolsm_oracle as orc
from tests.test_oracle_pins import _dense_pattern_system
from workloads import MAT_H, MAT_S, make_system


def test_full_cutoff_count_is_the_number_of_states_below_mu():
    """Every N(i) is the whole system: Tr(D S) = #{generalised eigenvalues below mu}, an integer (P5), and the q_i are
    the Mulliken populations of the atoms, which sum to it."""
    rng = np.random.default_rng(31)
    n_at = 6
    atom_nb, rp, ci, Hv, Sv, Hd, Sd = _dense_pattern_system(n_at, [2, 3, 1, 4, 2, 3], rng, np.ones((n_at, n_at), bool))
    eps = sla.eigh(Hd, Sd, eigvals_only=True)
    for k in (0, 4, 9, len(eps)):
        mu = eps[0] - 1 if k == 0 else (eps[-1] + 1 if k == len(eps) else 0.5 * (eps[k - 1] + eps[k]))
        assert abs(orc.electron_count(atom_nb, rp, ci, Hv, Sv, mu) - k) < 1e-9
    # Mulliken populations against the dense definition (D S)_aa summed over the atom's functions
    mu = 0.5 * (eps[6] + eps[7])
    D = orc.density_literal(Hd, Sd, mu)
    pop = np.diag(D @ Sd)
    first = np.concatenate([[0], np.cumsum(atom_nb)])
    blk = orc.block_offsets(atom_nb, rp, ci)
    for i in range(n_at):
        q_i = orc.atom_result(i, atom_nb, rp, ci, blk, Hv, Sv, mu)["q_i"]
        assert abs(q_i - pop[first[i]:first[i + 1]].sum()) < 1e-9


def test_count_is_monotone_in_mu_and_bisection_brackets_the_target():
    s = make_system("cfg0", n_atoms=32)
    Hv, Sv = s.fill_np(MAT_H), s.fill_np(MAT_S)
    n_basis = int(s.atom_nb.sum())
    count = lambda mu: orc.electron_count(s.atom_nb, s.row_ptr, s.col_idx, Hv, Sv, mu)
    grid = np.linspace(-8.0, 8.0, 9)
    vals = [count(m) for m in grid]
    assert all(b >= a - 1e-9 for a, b in zip(vals, vals[1:]))
    assert abs(vals[0]) < 1e-9 and abs(vals[-1] - n_basis) < 1e-6        # mu below / above every spectrum: D = 0 / D = S^-1 (P8)
    # half filling sits in the gap between the two on-site levels (-1 and +1) of the generator
    mu, n_mu, evals = orc.find_mu(count, n_basis / 2, -8.0, 8.0, tol_n=0.05, tol_mu=1e-3)
    assert abs(n_mu - n_basis / 2) <= 0.05 and -0.8 < mu < 0.8 and evals <= 20
    # a target inside a step of the count: the bisection closes the bracket around the jump
    target = 0.3 * n_basis
    mu2, n2, ev2 = orc.find_mu(count, target, -8.0, 8.0, tol_n=1e-9, tol_mu=1e-2)
    assert count(mu2 - 2e-2) <= target <= count(mu2 + 2e-2)
