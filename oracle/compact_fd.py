"""Seven-point compact finite differences on a non-uniform mesh (oracle side; test infrastructure).

PAPER.md L80 (section 2.1): "Derivatives in that direction are computed on the mesh using seven-point
compact finite differences with spectral-like resolution [23]"; L100 (section 2.3): "compact finite
differences of up to twelfth order of consistency are used for the discretisation of the second
derivative".  The paper prints no coefficients; reading R4 fixes them:

  row j of the d-th derivative operator:   sum_m a_{j,m} f^(d)_{j+m} = sum_m b_{j,m} f_{j+m},
  a_{j,0} = 1, both sums over the same centred window |m| <= s_j = min(3, j, Ny-1-j), and the
  4 s_j + 1 unknowns are the unique solution that makes the row exact for every polynomial of
  degree <= 4 s_j on the actual mesh (degree 12 in the interior = "twelfth order").
  First-derivative wall rows (j = 0 and, mirrored, j = Ny-1): left window {0, 1}, right window
  {0, 1, 2, 3}, exact to degree 4.  Second-derivative wall rows are never used (reading R6).

The coefficients are computed here in EXACT rational arithmetic (python ``fractions``) from the
mesh values as given (a double is a rational), and rounded once to double at the end, so there is
no conditioning argument to make.  The CUDA library computes its own tables independently.

Band storage used throughout the oracle: ``T[j, 3 + m]`` holds the entry in row j, column j + m.
"""
from fractions import Fraction

import numpy as np

HALF = 3  # seven-point: offsets -3..3


def _solve_exact(M, r):
    """Gaussian elimination with row exchanges over the rationals (exact)."""
    n = len(M)
    M = [row[:] + [r[i]] for i, row in enumerate(M)]
    for c in range(n):
        p = next(i for i in range(c, n) if M[i][c] != 0)
        M[c], M[p] = M[p], M[c]
        inv = 1 / M[c][c]
        for i in range(c + 1, n):
            if M[i][c] != 0:
                f = M[i][c] * inv
                for k in range(c, n + 1):
                    M[i][k] -= f * M[c][k]
    x = [Fraction(0)] * n
    for i in range(n - 1, -1, -1):
        x[i] = (M[i][n] - sum(M[i][k] * x[k] for k in range(i + 1, n))) / M[i][i]
    return x


def compact_row(y, j, lhs_offsets, rhs_offsets, deriv):
    """Coefficients (a, b) of one compact row, exact for all polynomials up to the unknown count - 1.

    ``lhs_offsets`` must contain 0 (a_0 = 1 is the normalisation).  Test polynomials are the
    monomials t^k, t = y - y_j, k = 0 .. n_unknowns - 1.  Returns dicts offset -> Fraction.
    """
    yy = [Fraction(float(v)) for v in y]
    lhs_free = [m for m in lhs_offsets if m != 0]
    n = len(lhs_free) + len(rhs_offsets)

    def dmono(t, k):  # d-th derivative of t^k
        if deriv == 1:
            return Fraction(k) * t ** (k - 1) if k >= 1 else Fraction(0)
        return Fraction(k * (k - 1)) * t ** (k - 2) if k >= 2 else Fraction(0)

    M, r = [], []
    for k in range(n):
        row = [dmono(yy[j + m] - yy[j], k) for m in lhs_free]
        row += [-((yy[j + m] - yy[j]) ** k) for m in rhs_offsets]
        M.append(row)
        r.append(-dmono(Fraction(0), k))  # the a_0 = 1 term moved to the right
    x = _solve_exact(M, r)
    a = {0: Fraction(1)}
    a.update({m: x[i] for i, m in enumerate(lhs_free)})
    b = {m: x[len(lhs_free) + i] for i, m in enumerate(rhs_offsets)}
    return a, b


def build_operators(y, half_lhs=HALF, half_rhs=HALF):
    """Band tables A1, B1 (first derivative) and A2, B2 (second derivative), each (Ny, 7) float64.

    ``half_lhs``/``half_rhs`` < 3 give the narrower schemes of reading R4 ("band tables are data").
    A2/B2 rows 0 and Ny-1 are left as zeros (never used, reading R6).
    """
    y = np.asarray(y, dtype=np.float64)
    ny = y.size
    assert ny >= 8 and np.all(np.diff(y) > 0)
    T = {k: np.zeros((ny, 7)) for k in ("A1", "B1", "A2", "B2")}
    for j in range(ny):
        room = min(j, ny - 1 - j)
        for d, (ka, kb) in ((1, ("A1", "B1")), (2, ("A2", "B2"))):
            if room == 0:
                if d == 2:
                    continue
                sgn = 1 if j == 0 else -1
                lo = [0, sgn]
                ro = [0, sgn, 2 * sgn, 3 * sgn]
            else:
                sl, sr = min(half_lhs, room), min(half_rhs, room)
                lo = list(range(-sl, sl + 1))
                ro = list(range(-sr, sr + 1))
            a, b = compact_row(y, j, lo, ro, d)
            for m, v in a.items():
                T[ka][j, 3 + m] = float(v)
            for m, v in b.items():
                T[kb][j, 3 + m] = float(v)
    return T["A1"], T["B1"], T["A2"], T["B2"]


def band_to_dense(T):
    ny = T.shape[0]
    D = np.zeros((ny, ny))
    for j in range(ny):
        for m in range(-3, 4):
            if 0 <= j + m < ny:
                D[j, j + m] = T[j, 3 + m]
    return D


def band_matvec(T, f):
    """(T f)_j = sum_m T[j,3+m] f_{j+m}; ``f`` has y as its LAST axis; T is (Ny,7) or (...,Ny,7)."""
    ny = f.shape[-1]
    out = np.zeros(np.broadcast_shapes(f.shape, T.shape[:-1]), dtype=np.result_type(f, T))
    for m in range(-3, 4):
        lo, hi = max(0, -m), min(ny, ny - m)
        out[..., lo:hi] += T[..., lo:hi, 3 + m] * f[..., lo + m:hi + m]
    return out


def banded_solve(T, r):
    """Solve T x = r by plain Gaussian elimination WITHOUT pivoting, rows in ascending order.

    ``T``: (Ny,7) or (batch,Ny,7) band table (not modified); ``r``: (..., Ny) with y last; the
    leading axes of ``r`` must broadcast against T's batch axis as r[batch, k, Ny] (T gets a
    singleton axis inserted for k).  Seven diagonals do not fill in without pivoting.
    Pinned against a dense pivoted solve in tests/test_oracle_compact.py.
    """
    T = np.array(T, dtype=np.float64, copy=True)
    ny = T.shape[-2]
    batched = T.ndim == 3
    x = np.array(r, copy=True)
    if batched:
        assert x.ndim == 3 and x.shape[0] == T.shape[0]
    for j in range(ny - 1):
        piv = T[..., j, 3]
        for t in range(1, 4):
            i = j + t
            if i >= ny:
                break
            l = T[..., i, 3 - t] / piv
            for cc in range(1, 4):
                if 3 - t + cc <= 6:
                    T[..., i, 3 - t + cc] -= l * T[..., j, 3 + cc]
            T[..., i, 3 - t] = 0.0
            x[..., i] -= (l[:, None] if batched else l) * x[..., j]
    for j in range(ny - 1, -1, -1):
        acc = x[..., j]
        for cc in range(1, 4):
            if j + cc < ny:
                u = T[..., j, 3 + cc]
                acc = acc - (u[:, None] if batched else u) * x[..., j + cc]
        d = T[..., j, 3]
        x[..., j] = acc / (d[:, None] if batched else d)
    return x


def d1(A1, B1, f):
    """First derivative along the last axis: solve A1 g = B1 f (DESIGN.md step 1 notation 'D1')."""
    rhs = band_matvec(B1, f)
    shp = rhs.shape
    return banded_solve(A1, rhs.reshape(-1, shp[-1])).reshape(shp)
