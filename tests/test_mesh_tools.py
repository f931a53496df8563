"""NEXT-4 (section 2.3): the wall-layer error of the homogeneous Helmholtz solutions and the mesh remedy.
Host-only library calls (no GPU) against oracle/mesh_error.py."""
import numpy as np
import pytest

import __graft_entry__ as entry
from oracle import compact_fd as cfd
from oracle.mesh_error import exact_wall_layer, helmholtz_wall_error
from paper_1808_06461_b200 import inputs


@pytest.fixture(scope="module")
def B():
    entry.build()
    from paper_1808_06461_b200 import binding
    binding.load()
    return binding


def test_exact_wall_layer_is_the_sinh_solution():
    """Closed form: phi = sinh(k(2-d))/sinh(2k) solves phi'' = k^2 phi, phi(0) = 1, phi(2) = 0."""
    d = np.linspace(0, 2, 41)
    for lam in (0.5, 9.0, 400.0):
        k = np.sqrt(lam)
        assert np.allclose(exact_wall_layer(d, lam), np.sinh(k * (2 - d)) / np.sinh(2 * k), rtol=1e-12, atol=1e-300)
    assert exact_wall_layer(np.array([0.0, 2.0]), 1e8)[0] == pytest.approx(1.0, abs=1e-15) and exact_wall_layer(np.array([2.0]), 1e8)[0] == 0.0


def test_wall_error_grows_with_lambda_and_vanishes_when_resolved():
    """The effect the paper describes (L100): resolved layers are exact to rounding, thin ones are not."""
    y = inputs.mesh_tanh(129, 2.5)
    T = cfd.build_operators(y)[2:]
    e = [max(helmholtz_wall_error(y, lam, 23, T)) for lam in (1e2, 1e4, 1e6, 1e8)]
    assert e[0] < 1e-10 and e[1] < 1e-7 and 1e-6 < e[2] < 1e-2 and e[3] > 1e-3 and e[0] < e[1] < e[2] < e[3]
    a, b = helmholtz_wall_error(y, 1e6, 23, T)
    assert a == pytest.approx(b, rel=1e-9)                      # symmetric mesh: the two walls are mirror images


@pytest.mark.parametrize("lam", [1e4, 1e6, 1e8])
def test_library_error_matches_the_oracle(B, lam):
    y = inputs.mesh_tanh(129, 2.5)
    ref = helmholtz_wall_error(y, lam, 23)
    got = B.mesh_helmholtz_error(y, lam, 23)
    assert np.allclose(got, ref, rtol=1e-6, atol=1e-14)


def test_optimised_mesh_reduces_the_worst_case_error_within_its_bounds(B):
    """L102: "slightly displacing the first 20 grid points in order to minimize the error of the most dangerous
    solutions without affecting too much the individual grid spacing".  The oracle evaluates both meshes independently
    (exact-rational rows); the optimised one must be better by the factor the library reports, stay monotone and
    symmetric, keep every point within max_shift of its original spacing, leave the other points alone, and stay
    admissible (real negative D2-Dirichlet spectrum)."""
    import scipy.linalg as sla
    c = inputs.config("cfg3")            # 251 points, tanh 2.5
    y = c["y"]
    lam = (2 * np.pi * (c["nx"] // 2 - 1) / c["lx"]) ** 2 + (2 * np.pi * (c["nz"] // 2 - 1) / c["lz"]) ** 2 + 6.0 * c["re"] / c["dt"]
    npts, shift = 20, 0.1
    y2, eb, ea = B.mesh_optimize(y, npts, lam, shift, 8)
    assert ea.max() < 0.2 * eb.max() and np.all(ea <= eb)         # measured: 9.3e-3 -> 5.3e-4
    ob, oa = helmholtz_wall_error(y, lam, npts + 3), helmholtz_wall_error(y2, lam, npts + 3)
    assert np.allclose(eb, ob, rtol=1e-6) and np.allclose(ea, oa, rtol=1e-6)
    assert y2[0] == -1.0 and y2[-1] == 1.0 and np.all(np.diff(y2) > 0)
    assert np.array_equal(y2[npts + 1: -npts - 1], y[npts + 1: -npts - 1])
    assert np.abs(y2 + y2[::-1]).max() < 1e-15                   # symmetric in, symmetric out (the walls are optimised alike)
    h = np.minimum(np.diff(y)[:-1], np.diff(y)[1:])
    assert np.all(np.abs(y2 - y)[1:-1] <= shift * h * (1 + 1e-12))
    assert np.abs(np.diff(y2) / np.diff(y) - 1).max() <= 2 * shift + 1e-12
    assert not np.array_equal(y2, y)
    _, _, A2, B2 = cfd.build_operators(y2)
    ev = sla.eigvals(cfd.band_to_dense(B2)[1:-1, 1:-1], cfd.band_to_dense(A2)[1:-1, 1:-1])
    assert np.abs(ev.imag).max() < 1e-6 * np.abs(ev.real).max() and ev.real.max() < 0
    # the library accepts the optimised mesh like any other
    ch = B.Channel(32, c["ny"], 16, c["lx"], c["lz"], y2, c["re"], c["dt"])
    ch.close()


def test_mesh_tool_argument_validation(B):
    y = inputs.mesh_cosine(33, 0.7)
    lib = B.load()
    out = np.zeros(2)
    assert lib.chan_mesh_helmholtz_error(33, y.ctypes.data, -1.0, 5, out.ctypes.data) == B.EINVAL
    assert lib.chan_mesh_helmholtz_error(33, y.ctypes.data, 1e4, 0, out.ctypes.data) == B.EINVAL
    yb = y.copy(); yb[4] = yb[3]
    assert lib.chan_mesh_helmholtz_error(33, yb.ctypes.data, 1e4, 5, out.ctypes.data) == B.EINVAL
    assert lib.chan_mesh_optimize(33, y.copy().ctypes.data, 5, 1e4, 0.5, 4, None, None) == B.EINVAL      # max_shift must be < 1/2
    assert lib.chan_mesh_optimize(33, y.copy().ctypes.data, 20, 1e4, 0.1, 4, None, None) == B.EINVAL     # 2 (20 + 4) > 33
    assert lib.chan_mesh_optimize(33, y.copy().ctypes.data, 5, 1e4, 0.1, 4, None, None) == B.OK          # optional outputs
    bad = inputs.mesh_cosine(33, 1.0)                     # Chebyshev-Gauss-Lobatto: not admissible for these rows
    assert lib.chan_mesh_optimize(33, bad.ctypes.data, 5, 1e4, 0.1, 4, None, None) == B.EINVAL
