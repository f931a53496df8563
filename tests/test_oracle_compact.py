"""Pins for oracle/compact_fd.py (no GPU): closed forms, polynomial exactness, dense solves, analytic Helmholtz."""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import compact_fd as cfd
from paper_1808_06461_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold():
    out = {}
    for line in open(os.path.join(GOLD, "compact_uniform.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        out[k] = [float(Fraction(s)) for s in v]
    return out


def test_uniform_mesh_closed_forms():
    """Lele's maximal-order Pade schemes (PAPER.md ref [23]) are reproduced on a uniform mesh."""
    g = _gold()
    ny, h = 17, 2.0 / 16
    y = np.linspace(-1, 1, ny)
    A1, B1, A2, B2 = cfd.build_operators(y)
    for s, j in ((1, 1), (2, 2), (3, 8)):
        lhs, rhs = g[f"D1s{s}_lhs"], g[f"D1s{s}_rhs"]
        for m in range(1, s + 1):
            assert A1[j, 3 + m] == pytest.approx(lhs[m - 1], rel=1e-13)
            assert A1[j, 3 - m] == pytest.approx(lhs[m - 1], rel=1e-13)
            assert B1[j, 3 + m] * h == pytest.approx(rhs[m - 1], rel=1e-13)
            assert B1[j, 3 - m] * h == pytest.approx(-rhs[m - 1], rel=1e-13)
        assert abs(B1[j, 3]) * h < 1e-13
    for s, j in ((1, 1), (2, 2)):
        lhs, rhs = g[f"D2s{s}_lhs"], g[f"D2s{s}_rhs"]
        for m in range(1, s + 1):
            assert A2[j, 3 + m] == pytest.approx(lhs[m - 1], rel=1e-12)
            assert B2[j, 3 - m] * h * h == pytest.approx(rhs[m - 1], rel=1e-12)
        assert B2[j, 3] * h * h == pytest.approx(-2 * sum(rhs), rel=1e-12)
    # interior twelfth-order second-derivative row: symmetric, consistent (sum b = 0)
    assert A2[8, 4] == pytest.approx(A2[8, 2], rel=1e-13) and abs(B2[8].sum()) * h * h < 1e-12
    # wall rows of D1
    assert A1[0, 4] == pytest.approx(g["D1wall_lhs"][0], rel=1e-13)
    assert np.allclose(B1[0, 3:7] * h, g["D1wall_rhs"], rtol=1e-13)
    assert A1[-1, 2] == pytest.approx(3.0, rel=1e-13)
    assert np.allclose(B1[-1, 0:4][::-1] * h, [-x for x in g["D1wall_rhs"]], rtol=1e-13)


@pytest.mark.parametrize("mesh", ["cos", "tanh"])
def test_polynomial_exactness(mesh):
    """Row j is exact for all polynomials of degree <= 4 s_j on the actual (stretched) mesh (reading R4)."""
    ny = 33
    y = inputs.mesh_cosine(ny, 0.7) if mesh == "cos" else inputs.mesh_tanh(ny, 2.5)
    A1, B1, A2, B2 = cfd.build_operators(y)
    for j in range(ny):
        s = min(3, j, ny - 1 - j)
        deg1 = 4 if s == 0 else 4 * s
        t = y - y[j]
        scale = np.abs(t[max(0, j - 3):j + 4]).max()
        t = t / scale
        for k in range(deg1 + 1):
            f = t ** k
            df = k * t ** (k - 1) / scale if k else 0 * t
            lhs = sum(A1[j, 3 + m] * df[j + m] for m in range(-3, 4) if 0 <= j + m < ny)
            rhs = sum(B1[j, 3 + m] * f[j + m] for m in range(-3, 4) if 0 <= j + m < ny)
            assert abs(lhs - rhs) * scale < 2e-11, (j, k)
        if s == 0:
            continue
        for k in range(4 * s + 1):
            f = t ** k
            d2f = k * (k - 1) * t ** (k - 2) / scale ** 2 if k > 1 else 0 * t
            lhs = sum(A2[j, 3 + m] * d2f[j + m] for m in range(-3, 4) if 0 <= j + m < ny)
            rhs = sum(B2[j, 3 + m] * f[j + m] for m in range(-3, 4) if 0 <= j + m < ny)
            assert abs(lhs - rhs) * scale ** 2 < 2e-10, (j, k)
        # and NOT exact one degree higher in the interior (the row is maximal order, not accidental)
    j = ny // 2
    t = (y - y[j])
    f, d2f = t ** 14, 14 * 13 * t ** 12
    lhs = sum(A2[j, 3 + m] * d2f[j + m] for m in range(-3, 4))
    rhs = sum(B2[j, 3 + m] * f[j + m] for m in range(-3, 4))
    assert abs(lhs - rhs) > 1e-18


def test_banded_solve_and_matvec_match_dense():
    rng = np.random.default_rng(0)
    ny = 19
    T = rng.standard_normal((5, ny, 7))
    T[:, :, 3] += 6.0
    for j in range(3):  # zero the entries that fall outside the matrix
        T[:, j, : 3 - j] = 0.0
        T[:, ny - 1 - j, 4 + j:] = 0.0
    r = rng.standard_normal((5, 4, ny))
    x = cfd.banded_solve(T, r)
    for b in range(5):
        D = cfd.band_to_dense(T[b])
        assert np.allclose(x[b].T, np.linalg.solve(D, r[b].T), rtol=1e-12, atol=1e-13)
        assert np.allclose(cfd.band_matvec(T[b], r[b]), r[b] @ D.T, rtol=1e-13, atol=1e-13)
    # unbatched table, complex right-hand sides, arbitrary leading axes
    rc = rng.standard_normal((2, 3, ny)) + 1j * rng.standard_normal((2, 3, ny))
    xc = cfd.banded_solve(T[0], rc)
    assert np.allclose(np.einsum("ij,abj->abi", cfd.band_to_dense(T[0]), xc), rc, atol=1e-12)
    # batched band_matvec with a per-batch table
    f = rng.standard_normal((5, ny))
    mv = cfd.band_matvec(T, f)
    for b in range(5):
        assert np.allclose(mv[b], cfd.band_to_dense(T[b]) @ f[b])


def test_d1_on_smooth_function():
    y = inputs.mesh_tanh(65, 2.0)
    A1, B1, _, _ = cfd.build_operators(y)
    g = cfd.d1(A1, B1, np.sin(2 * y)[None, :])[0]
    assert np.abs(g - 2 * np.cos(2 * y)).max() < 5e-9  # wall rows are 4th order


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "mid", "cfg3", "cfg4", "cfg5"])
def test_d2_dirichlet_spectrum_admissible(name):
    """PAPER.md section 2.3 (L100-102): wide stencils are only usable on a mesh they were checked on (every mesh
    bench.py times is checked here: SURVEY.md Appendix A "harness obligation").
    Generalised eigenvalues of (B2, A2) with Dirichlet walls must be real, negative, -> -(n pi/2)^2."""
    import scipy.linalg as sla
    c = inputs.config(name)
    _, _, A2, B2 = cfd.build_operators(c["y"])
    a = cfd.band_to_dense(A2)[1:-1, 1:-1]
    b = cfd.band_to_dense(B2)[1:-1, 1:-1]
    ev = sla.eigvals(b, a)
    assert np.abs(ev.imag).max() < 1e-6 * np.abs(ev.real).max()
    assert ev.real.max() < 0
    lead = np.sort(ev.real)[::-1][:3]
    exact = -(np.arange(1, 4) * np.pi / 2) ** 2
    tol = 1e-6 if c["ny"] >= 65 else 2e-3
    assert np.allclose(lead, exact, rtol=tol)


@pytest.mark.parametrize("lam", [1e2, 1e4, 1e6])
def test_helmholtz_homogeneous_solution_matches_analytic(lam):
    """The paper's own numerical test (Fig. 2.3, L94, L100-102): phi'' - lam phi = 0, phi(-1)=1, phi(1)=0."""
    y = inputs.mesh_tanh(129, 2.5)
    _, _, A2, B2 = cfd.build_operators(y)
    M = B2 - lam * A2
    M[0] = M[-1] = 0.0
    M[0, 3] = M[-1, 3] = 1.0
    r = np.zeros(129)
    r[0] = 1.0
    phi = cfd.banded_solve(M, r)
    k = np.sqrt(lam)
    exact = np.exp(-k * (1 + y)) * (1 - np.exp(-2 * k * (1 - y))) / (1 - np.exp(-4 * k))
    tol = {1e2: 1e-10, 1e4: 1e-7, 1e6: 5e-3}[lam]
    assert np.abs(phi - exact).max() < tol
