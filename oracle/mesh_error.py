"""Oracle of the paper's wall-layer test (section 2.3, Fig. 2.3; NEXT-4).

TEST INFRASTRUCTURE (see oracle/__init__.py).  "The most numerically sensitive operation ... requires the solution of
multiple homogeneous Helmholtz equations to impose the boundary conditions.  For high Reynolds numbers and small
wavelengths, these solutions include very thin boundary layers near the wall" (L100).  The test: solve
phi'' = lam phi, phi = 1 at one wall, 0 at the other, with the compact second-derivative rows of reading R4 (exact
rationals, oracle/compact_fd.py) and compare with the closed form on the first mesh points.
"""
import numpy as np

from . import compact_fd as cfd


def exact_wall_layer(d, lam):
    """phi(d) = sinh(k (2 - d)) / sinh(2 k), k = sqrt(lam), d = distance from the wall that carries phi = 1 (0 <= d <= 2),
    written with decaying exponentials only."""
    k = np.sqrt(lam)
    return np.exp(-k * d) * (1.0 - np.exp(-2.0 * k * (2.0 - d))) / (1.0 - np.exp(-4.0 * k))


def helmholtz_wall_error(y, lam, nfirst, tables=None):
    """(error at y = -1, error at y = +1): max over the first ``nfirst`` interior points next to the wall of
    |phi_j - phi_exact(y_j)| for the discrete solution of (B2 - lam A2) phi = 0 with Dirichlet rows (step 6 form)."""
    y = np.asarray(y, dtype=np.float64)
    ny = y.size
    A2, B2 = tables if tables is not None else cfd.build_operators(y)[2:]
    M = B2 - lam * A2
    M[0] = M[-1] = 0.0
    M[0, 3] = M[-1, 3] = 1.0
    out = []
    for side in (0, 1):
        r = np.zeros(ny)
        r[0 if side == 0 else -1] = 1.0
        phi = cfd.banded_solve(M, r)
        d = 1.0 + y if side == 0 else 1.0 - y
        err = np.abs(phi - exact_wall_layer(d, lam))
        idx = np.arange(1, nfirst + 1) if side == 0 else ny - 1 - np.arange(1, nfirst + 1)
        out.append(float(err[idx].max()))
    return tuple(out)
