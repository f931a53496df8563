"""Pins for three oracle branches that nothing outside the oracle fixed before:
the trapezoid weights of the mass flux (reading R8), the constant-pressure-gradient forcing option
(forcing = 1: a chan_opts_t option of SURVEY 8(b), not the paper's constant-mass-flux case of PAPER.md
L61) and the row map of the filtered products (reading R11)."""
import math

import numpy as np
import pytest

from oracle.channel import ChannelOracle, trapezoid_weights
from paper_1808_06461_b200 import inputs


# ---------------------------------------------------------------------------------- trapezoid weights
@pytest.mark.parametrize("mesh", ["cos33", "tanh129", "ragged"])
def test_trapezoid_weights_are_the_trapezoid_rule(mesh):
    """Q = sum_j w_j U_j (R8).  Closed forms: sum w = 2 (length of [-1,1]); exact on every function that is linear
    between mesh points, in particular on |y - y_k| with the kink AT a mesh point, whose integral is
    ((y_k+1)^2 + (1-y_k)^2)/2 -- a rectangle (left or right) rule gets neither this nor the linear
    function y right on a stretched mesh; and second-order convergence (not exactness) on y^2."""
    if mesh == "cos33":
        y = inputs.mesh_cosine(33, 0.7)
    elif mesh == "tanh129":
        y = inputs.mesh_tanh(129, 2.5)
    else:   # not symmetric, irregular spacing
        rng = np.random.default_rng(3)
        y = np.sort(np.concatenate([[-1.0, 1.0], rng.uniform(-1, 1, 21)]))
    w = trapezoid_weights(y)
    assert w.shape == y.shape and np.all(w > 0)
    assert abs(w.sum() - 2.0) < 4e-16 * y.size
    assert abs(w @ y) < 1e-15                                     # int y dy = 0 exactly for any mesh containing +-1
    assert abs(w @ (3.0 * y + 0.5) - 1.0) < 1e-14                 # linear functions are integrated exactly
    for k in (1, y.size // 3, y.size // 2, y.size - 2):
        exact = 0.5 * ((y[k] + 1.0) ** 2 + (1.0 - y[k]) ** 2)
        assert abs(w @ np.abs(y - y[k]) - exact) < 1e-14, k       # kink at a mesh point: still exact
    # end weights are HALF intervals (a rectangle rule would carry a full interval at one end and none at the other)
    assert w[0] == pytest.approx(0.5 * (y[1] - y[0]), rel=1e-15) and w[-1] == pytest.approx(0.5 * (y[-1] - y[-2]), rel=1e-15)
    assert w[5] == pytest.approx(0.5 * (y[6] - y[4]), rel=1e-14)
    # y^2: error of the trapezoid rule is +sum h^3/6 > 0, not zero, and bounded by h_max^2/6 * 2
    err = w @ (y * y) - 2.0 / 3.0
    assert 0.0 < err <= np.diff(y).max() ** 2 / 3.0 + 1e-15


# ---------------------------------------------------------------------------------- forcing = 1
def test_forcing1_poiseuille_is_steady_under_the_matching_pressure_gradient():
    """U = Ucl (1 - y^2) with prescribed -dP/dx = 2 nu Ucl is an exact steady solution of
    dU/dt = -dP/dx + nu U'' (the compact rows are exact on a parabola); with 1.5x that gradient the mean flow
    accelerates at exactly 0.5 * 2 nu Ucl per unit time, uniformly in y away from the walls at early times."""
    c = inputs.config("cfg1")
    o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"], forcing=1)
    z = np.zeros(o.v.shape, complex)
    o.set_state(z, z, z, c["U"], c["W"])
    G = 2.0 * o.nu * 90.0
    o.pgrad = G
    for _ in range(5):
        o.step()
    assert np.abs(o.U - c["U"]).max() < 1e-10 * 90.0
    assert o.pgrad == G                                           # prescribed, never recomputed
    assert np.abs(o.W).max() == 0.0
    o2 = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"], forcing=1)
    o2.set_state(z, z, z, c["U"], c["W"])
    o2.pgrad = 1.5 * G
    o2.step()
    # the diffusive wall layer sqrt(nu dt) ~ 2e-3 is under-resolved on this mesh: its grid-scale oscillation (the
    # effect PAPER.md L100 describes) decays geometrically away from the wall and is 2e-8 at the centre
    mid = slice(o.ny // 2 - 1, o.ny // 2 + 2)
    assert np.allclose((o2.U - c["U"])[mid], 0.5 * G * c["dt"], rtol=1e-6, atol=0)


def _startup_series(y, t, G, nu, nterms=400):
    """Start-up of plane Poiseuille flow from rest under a constant pressure gradient (textbook Fourier series):
    U = G/(2 nu) (1-y^2) - sum_n 16 G (-1)^n / (nu (2n+1)^3 pi^3) cos((2n+1) pi y/2) exp(-nu (2n+1)^2 pi^2 t/4)."""
    U = G / (2.0 * nu) * (1.0 - y * y)
    for n in range(nterms):
        m = 2 * n + 1
        U = U - 16.0 * G * (-1.0) ** n / (nu * m ** 3 * math.pi ** 3) * np.cos(m * math.pi * y / 2.0) * math.exp(-nu * m * m * math.pi ** 2 * t / 4.0)
    return U


def test_forcing1_startup_from_rest_matches_the_series_at_second_order():
    """forcing = 1 from rest: the mean flow follows the start-up series; the error of the semi-implicit scheme [34]
    is second order in dt (reading R3) on top of a spatial error that is negligible on this mesh.  A wrong sign or a
    wrong (gamma_i + zeta_i) dt weight of the forcing fails at O(1)."""
    y = inputs.mesh_tanh(65, 1.5)
    nu, G, T = 1.0 / 20.0, 0.7, 2.0
    errs = []
    for dt in (0.1, 0.05, 0.025):
        o = ChannelOracle(8, 65, 8, 2 * math.pi, 2 * math.pi, y, 1.0 / nu, dt, forcing=1)
        z = np.zeros(o.v.shape, complex)
        o.set_state(z, z, z, np.zeros(65), np.zeros(65))
        o.pgrad = G
        for _ in range(int(round(T / dt))):
            o.step()
        ex = _startup_series(y, T, G, nu)
        errs.append(np.abs(o.U - ex).max() / np.abs(ex).max())
        assert o.U[0] == 0.0 and o.U[-1] == 0.0
    assert errs[0] < 2e-4 and errs[2] < 2e-5, errs
    assert 3.0 < errs[0] / errs[1] < 5.5 and 3.0 < errs[1] / errs[2] < 5.5, errs
    # a flow that has not reached the steady parabola yet: the test is about the transient
    assert 0.1 < ex.max() / (G / (2 * nu)) < 0.5


# ---------------------------------------------------------------------------------- filtered products: row map
def test_filtered_products_are_the_full_transform_restricted_by_the_integer_predicate():
    """PAPER.md L124 / R11-R12: out[3..9] of filter_store must be the retained-mode transform of the products
    -- the plain to_spectral() that tests/test_oracle_fft.py pins against brute-force trigonometric sums --
    restricted to 0 <= p <= Kx, |q| <= Kz with rows ordered q = 0..Kz, -Kz..-1, bit for bit.  A +-q mix-up, a
    shifted row or a transposed cutoff changes entries and fails array_equal.  Cutoffs differ in x and z and the
    spectrum is not symmetric in q (random phases), so such mistakes cannot cancel."""
    c = inputs.config("cfg1")
    o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    v, phi, omy = (t.numpy() * 50 for t in inputs.fluctuations(c))
    o.set_state(v, phi, omy, c["U"], c["W"])
    for kxc, kzc in ((5, 3), (o.nx // 2 - 1, o.nz // 2 - 1), (0, 0), (2, 9)):
        out = o.filter_store(kxc, kzc)
        pu, pv, pw, pox, poy, poz = (o.to_physical(f) for f in o.velocities_vorticities())
        prods = (pu * pu, pu * pv, pu * pw, pv * pv, pv * pw, pw * pw, pox * pox + poy * poy + poz * poz)
        qs = list(range(0, kzc + 1)) + list(range(-kzc, 0))
        for n, pr in enumerate(prods):
            full = o.to_spectral(pr)                               # [nz][nx/2][ny], retained modes, FFT slot order
            for r, q in enumerate(qs):
                slot = q if q >= 0 else o.nz + q
                for p in range(kxc + 1):
                    assert np.array_equal(out[3 + n, :, r, p], full[slot, p, :]), (n, q, p)
        # q and -q rows are genuinely different data (the test would be vacuous otherwise)
        if kzc >= 1:
            assert not np.array_equal(out[4, :, 1, 1], out[4, :, 2 * kzc, 1])
