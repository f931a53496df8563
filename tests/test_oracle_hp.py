"""The extended-precision yardstick (oracle/channel_hp.py) checked against EXACT rational arithmetic.

ChannelHP repeats the oracle's steps 5-7 in 80-bit long double.  It is used by the GPU parity tests to decide how
much of |gpu - oracle| on phi^ is fp64 rounding of an ill-conditioned step.  Here: on one
Fourier mode of config 1 the Helmholtz/Poisson/influence-matrix chain is redone with python Fractions (exact:
every double is a rational) from the same double inputs; the long-double result must sit orders of magnitude
closer to the exact one than the fp64 oracle does."""
from fractions import Fraction

import numpy as np

from oracle import channel_hp as hp
from oracle.channel import RK_ALPHA, RK_BETA, RK_GAMMA, RK_ZETA, ChannelOracle
from paper_1808_06461_b200 import inputs


def _exact_band_solve(T, r):
    """Gaussian elimination without pivoting over the rationals; T [ny][7] Fractions, r [ny] Fractions."""
    ny = len(T)
    T = [row[:] for row in T]
    x = r[:]
    for j in range(ny - 1):
        for t in range(1, 4):
            i = j + t
            if i >= ny:
                break
            l = T[i][3 - t] / T[j][3]
            if l == 0:
                continue
            for cc in range(1, 4):
                if 3 - t + cc <= 6:
                    T[i][3 - t + cc] -= l * T[j][3 + cc]
            T[i][3 - t] = Fraction(0)
            x[i] -= l * x[j]
    for j in range(ny - 1, -1, -1):
        acc = x[j]
        for cc in range(1, 4):
            if j + cc < ny:
                acc -= T[j][3 + cc] * x[j + cc]
        x[j] = acc / T[j][3]
    return x


def _fr(a):
    return [Fraction(float(v)) for v in a]


def _matvec(T, f):
    ny = len(f)
    return [sum((T[j][3 + m] * f[j + m] for m in range(-3, 4) if 0 <= j + m < ny), Fraction(0)) for j in range(ny)]


def test_long_double_substep_is_far_closer_to_exact_than_fp64():
    c = inputs.config("cfg1")
    o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    v, phi, omy = (t.numpy() * 10 for t in inputs.fluctuations(c))
    rng = np.random.default_rng(5)
    shp = o.v.shape
    H = [1e2 * (rng.standard_normal(shp) + 1j * rng.standard_normal(shp)) for _ in range(3)]
    hvp = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)
    isub = 1
    o.set_state(v, phi, omy, c["U"], c["W"])
    h = hp.ChannelHP(o)
    h.set_state(v, phi, omy, c["U"], c["W"])
    for orc in (o, h):
        orc.isub = isub
        orc.hv_prev = hvp.copy() if orc is o else hvp.astype(hp.CLD)
    o.nonlinear = lambda fields: tuple(x.copy() for x in H)
    h.nonlinear_override = lambda fields: H
    phi_old = o.phi.copy()
    o.substep()
    h.substep()
    assert h.phi.dtype == hp.CLD and h.v.dtype == hp.CLD and h.U.dtype == hp.LD
    # exact phi^, v^ of one mode (real parts only: the problems are real) from the same doubles
    s, p = 3, 5
    ny = o.ny
    al, be, ga, ze = RK_ALPHA[isub], RK_BETA[isub], RK_GAMMA[isub], RK_ZETA[isub]
    cc = Fraction(1.0 / (be * o.nu * o.dt))
    g = Fraction(al * o.nu * o.dt)
    k2 = Fraction(float(o.k2[s, p]))
    lam = Fraction(float(o.k2[s, p] + 1.0 / (be * o.nu * o.dt)))
    A1, B1, A2, B2 = ([_fr(row) for row in T] for T in (o.A1, o.B1, o.A2, o.B2))
    kx, kz = Fraction(float(o.kx[p])), Fraction(float(o.kz[s]))
    # h_v = -k2 H2 - D1(i kx H1 + i kz H3), real part: -k2 Re H2 - D1(-kx Im H1 - kz Im H3)
    d = [-kx * a - kz * b for a, b in zip(_fr(H[0][s, p].imag), _fr(H[2][s, p].imag))]
    dd = _exact_band_solve(A1, _matvec(B1, d))
    hv = [-k2 * a - b for a, b in zip(_fr(H[1][s, p].real), dd)]
    x = _fr(phi_old[s, p].real)
    t = [a + Fraction(o.dt) * (Fraction(ga) * b + Fraction(ze) * e) for a, b, e in zip(x, hv, _fr(hvp[s, p].real))]
    a2t, b2x, a2x = _matvec(A2, t), _matvec(B2, x), _matvec(A2, x)
    R = [-cc * (a + g * (b - k2 * e)) for a, b, e in zip(a2t, b2x, a2x)]
    R[0] = R[-1] = Fraction(0)

    def helm(l):
        M = [[B2[j][k] - l * A2[j][k] for k in range(7)] for j in range(ny)]
        for j in (0, ny - 1):
            M[j] = [Fraction(int(k == 3)) for k in range(7)]
        return M

    MH, MP = helm(lam), helm(k2)
    e0 = [Fraction(int(j == 0)) for j in range(ny)]
    e1 = [Fraction(int(j == ny - 1)) for j in range(ny)]
    php, pha, phb = (_exact_band_solve(MH, r) for r in (R, e0, e1))

    def poisson(ph):
        r = _matvec(A2, ph)
        r[0] = r[-1] = Fraction(0)
        return _exact_band_solve(MP, r)

    vp, va, vb = poisson(php), poisson(pha), poisson(phb)
    dvp, dva, dvb = (_exact_band_solve(A1, _matvec(B1, f)) for f in (vp, va, vb))
    det = dva[0] * dvb[-1] - dvb[0] * dva[-1]
    ca = (dvb[-1] * (-dvp[0]) - dvb[0] * (-dvp[-1])) / det
    cb = (-dva[-1] * (-dvp[0]) + dva[0] * (-dvp[-1])) / det
    phi_ex = np.array([float(a + ca * b + cb * e) for a, b, e in zip(php, pha, phb)])
    v_ex = np.array([float(a + ca * b + cb * e) for a, b, e in zip(vp, va, vb)])

    def rel(a, b):
        return float(np.linalg.norm(np.asarray(a, float) - b) / np.linalg.norm(b))

    e_hp_phi, e_or_phi = rel(h.phi[s, p].real, phi_ex), rel(o.phi[s, p].real, phi_ex)
    e_hp_v, e_or_v = rel(h.v[s, p].real, v_ex), rel(o.v[s, p].real, v_ex)
    # the long-double result is exact to fp64 printing precision; the fp64 oracle is visibly off on phi
    assert e_hp_phi < 5e-15 and e_hp_v < 5e-15, (e_hp_phi, e_hp_v)
    assert e_or_phi < 1e-9 and e_or_v < 1e-11, (e_or_phi, e_or_v)
    # whole field: oracle and yardstick agree to the fp64 error of the oracle (v, om_y: ~1e-14; phi: ~1e-11)
    assert rel(o.v.real, h.v.real.astype(float)) < 1e-12
    assert rel(o.omy.real, h.omy.real.astype(float)) < 1e-12
    assert rel(o.phi.real, h.phi.real.astype(float)) < 1e-9
    assert rel(o.U, h.U.astype(float)) < 1e-13


def test_long_double_plane_transforms_round_trip():
    """numpy's FFT keeps long double (no silent fp64 detour): spectral -> physical -> spectral returns the input
    to 1e-17, and the physical field matches the fp64 oracle's to fp64 accuracy."""
    c = inputs.config("cfg1")
    o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"])
    h = hp.ChannelHP(o)
    rng = np.random.default_rng(2)
    f = rng.standard_normal(o.v.shape) + 1j * rng.standard_normal(o.v.shape)
    nz = o.nz
    for q in range(1, nz // 2):
        f[nz - q, 0] = np.conj(f[q, 0])
    f[0, 0] = f[0, 0].real
    f[nz // 2] = 0
    ph = h.to_physical(f.astype(hp.CLD))
    assert ph.dtype == hp.LD
    back = h.to_spectral(ph)
    assert np.abs(back - f).max() < 1e-16 * np.abs(f).max() * 10
    assert np.abs(ph.astype(float) - o.to_physical(f)).max() < 1e-13 * np.abs(ph).max()
