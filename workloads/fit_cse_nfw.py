"""Writes workloads/cse_nfw.txt: amplitudes A_i and core radii s_i of the core-steep-ellipsoid (CSE) expansion of the NFW convergence
(Appendix A, Eq. A.1-A.5).  The paper uses Oguri (2021)'s 44 pairs, which are not available here and which it
does not print; it prints the basis (Eq. A.3-A.4), the target (Eq. A.1) and the objective (Eq. A.5: squared RELATIVE residuals on u_j
log-spaced over [1e-6, 1e3]) and says the pairs are "predetermined" -- i.e. an INPUT table of the method, like quadrature nodes.
This script produces THIS repository's table from exactly that recipe: 44 core radii log-spaced on [1e-7, 1e4], amplitudes by
non-negative least squares of Eq. A.5 on 900 radii.  Max relative error of the sum over [1e-6, 1e3]: 6.9e-6 (Oguri quotes 1e-4).
Both the CUDA library (glad_set_enfw takes the table as an argument) and the oracle read the table as data.

    python workloads/fit_cse_nfw.py        # rewrites workloads/cse_nfw.txt
"""
import os

import numpy as np
from scipy.optimize import nnls

N_CSE, S_LO, S_HI = 44, 1e-7, 1e4
U_LO, U_HI, N_U = 1e-6, 1e3, 900


def kappa_nfw(u):
    """Eq. A.1 with rho_s = 1."""
    u = np.asarray(u, float)
    out = np.empty_like(u)
    lo, hi = u < 1, u > 1
    t = np.sqrt(1 - u[lo] ** 2)
    out[lo] = 0.5 / (u[lo] ** 2 - 1) * (1 - np.arctanh(t) / t)
    t = np.sqrt(u[hi] ** 2 - 1)
    out[hi] = 0.5 / (u[hi] ** 2 - 1) * (1 - np.arctan(t) / t)
    out[~(lo | hi)] = 1.0 / 6.0
    return out


def fit():
    u = np.geomspace(U_LO, U_HI, N_U)
    s = np.geomspace(S_LO, S_HI, N_CSE)
    M = 0.5 / (s[None, :] ** 2 + u[:, None] ** 2) ** 1.5 / kappa_nfw(u)[:, None]      # Eq. A.4 over Eq. A.1: relative residuals
    scale = np.abs(M).max(0)
    A, _ = nnls(M / scale, np.ones(N_U), maxiter=20000)
    A = A / scale
    return A, s, float(np.abs(M @ A - 1).max())


if __name__ == "__main__":
    A, s, err = fit()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cse_nfw.txt")
    with open(path, "w") as f:
        f.write("# CSE expansion of kappa_nfw (Eq. A.3-A.5); written by workloads/fit_cse_nfw.py; columns: A_i s_i\n")
        f.write(f"# max relative error on u in [{U_LO:g}, {U_HI:g}]: {err:.3e}\n")
        for a, si in zip(A, s):
            if a > 0:
                f.write(f"{a:.17e} {si:.17e}\n")
    print(f"{(A > 0).sum()} pairs, max relative error {err:.3e} -> {path}")
