"""Writes workloads/gamma_table.json: the SURVEY C-12 rescale gamma of the off-site S blocks.

BASELINE.json's generator (off-site S amplitude 0.3) is not positive definite as written
(SURVEY.md finding 1). With S = I + gamma*W (W = off-site part at amplitude 0.3),
lambda_min(S) = 1 + gamma*lambda_min(W); gamma = (1 - 0.2) / (-lambda_min(W)) puts lambda_min(S)
at the floor 0.2. lambda_min(W) comes from Lanczos on the full system where that is cheap, else
from a 3000-atom periodic proxy of the same density and basis, times 0.9.

Usage: python -m workloads.calibrate_gamma [cfg0 cfg1 cfg2 cfg3 cfg4]
"""
import json
import sys
import time

import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as sla

from workloads.synthetic import (_GAMMA_PATH, LAMBDA_FLOOR, MAT_S, make_system, to_scipy)


def lambda_min_W(name, n_atoms=None):
    sysm = make_system(name, n_atoms=n_atoms, gamma=1.0)
    S = to_scipy(sysm, sysm.fill_np(MAT_S))
    W = (S - sp.identity(S.shape[0], format="csr")).tocsr()
    if W.shape[0] <= 3000:
        lam = float(np.linalg.eigvalsh(W.toarray())[0])
    else:
        lam = float(sla.eigsh(W, k=1, which="SA", return_eigenvectors=False, tol=1e-5, ncv=40)[0])
    return lam, sysm


def main(names):
    try:
        with open(_GAMMA_PATH) as f:
            tab = json.load(f)
    except FileNotFoundError:
        tab = {}
    plan = {"cfg0": ("cfg0", None, 1.0, True), "cfg1": ("cfg1", None, 1.0, True),
            "cfg2": ("cfg2", 3000, 0.9, True), "cfg3": ("cfg3", None, 1.0, True),
            "cfg4": ("cfg1", None, 0.9, True)}
    for name in names:
        src, n_at, safety, proxy_ok = plan[name]
        t0 = time.time()
        lam, sysm = lambda_min_W(src, n_at)
        gamma = min(1.0, safety * (1.0 - LAMBDA_FLOOR) / (-lam)) if lam < 0 else 1.0
        tab[name] = dict(gamma=gamma, lambda_min_W=lam, source=sysm.name, safety=safety,
                         lambda_min_S=1.0 + gamma * lam, proxy_ok=proxy_ok)
        print(name, tab[name], f"{time.time() - t0:.1f}s", flush=True)
        with open(_GAMMA_PATH, "w") as f:
            json.dump(tab, f, indent=1, sort_keys=True)


if __name__ == "__main__":
    main(sys.argv[1:] or ["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"])
