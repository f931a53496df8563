"""Pins for the substep (steps 1, 5-9): analytic solutions and an independent nonlinear-term evaluation."""
import os

import numpy as np
import pytest
from numpy.polynomial import polynomial as npoly

from oracle.channel import ChannelOracle
from oracle.os_mode import discrete_os_mode
from paper_1808_06461_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _oracle(name, **kw):
    c = inputs.config(name)
    o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"], **kw)
    return c, o


def _os_gold():
    vals = [l for l in open(os.path.join(GOLD, "os_re7500_alpha1.txt")) if not l.startswith("#")][0].split()
    return float(vals[0]) + 1j * float(vals[1])


def test_poiseuille_is_steady_and_pressure_gradient_is_2nu():
    """laminar flow U = Ucl(1-y^2) under constant mass flux is an exact steady solution,
    and the recovered mean pressure gradient is -dP/dx = 2 nu Ucl."""
    c, o = _oracle("cfg1")
    z = np.zeros(o.v.shape, complex)
    o.set_state(z, z, z, c["U"], c["W"])
    for _ in range(5):
        o.step()
    assert np.abs(o.U - c["U"]).max() < 1e-10
    assert np.abs(o.W).max() == 0.0
    assert o.pgrad == pytest.approx(2.0 * o.nu * 90.0, rel=1e-7)
    assert abs(o.w @ o.U - o.Q0) < 1e-11


def test_divergence_stays_at_roundoff_and_hermitian_symmetry_holds():
    c, o = _oracle("cfg1")
    v, phi, omy = (t.numpy() for t in inputs.fluctuations(c))
    o.set_state(v, phi, omy, c["U"], c["W"])
    scale = np.abs(o.D1(o.v)).max()
    assert np.abs(o.divergence()).max() < 1e-13 * scale
    for _ in range(10):
        o.substep()
    assert np.abs(o.divergence()).max() < 1e-13 * scale
    nz = o.nz
    for q in range(1, nz // 2):  # reading R14: p = 0 column stays Hermitian to roundoff
        assert np.abs(o.v[nz - q, 0] - np.conj(o.v[q, 0])).max() < 1e-11 * np.abs(o.v).max()
    # wall conditions v = dv/dy = 0, om_y = 0
    assert np.abs(o.v[:, :, [0, -1]]).max() == 0.0
    assert np.abs(o.D1(o.v)[:, :, [0, -1]]).max() < 1e-9 * scale
    assert np.abs(o.omy[:, :, [0, -1]]).max() == 0.0


def test_os_golden_matches_chebyshev():
    """Independent textbook pin of the golden eigenvalue: Chebyshev collocation Orr-Sommerfeld solve."""
    import scipy.linalg as sla
    N, Re, al = 120, 7500.0, 1.0
    x = np.cos(np.pi * np.arange(N + 1) / N)
    cc = np.r_[2.0, np.ones(N - 1), 2.0] * (-1.0) ** np.arange(N + 1)
    X = np.tile(x, (N + 1, 1)).T
    D = np.outer(cc, 1 / cc) / (X - X.T + np.eye(N + 1))
    D -= np.diag(D.sum(axis=1))
    D2 = (D @ D)[1:N, 1:N]
    S = np.diag(np.r_[0.0, 1 / (1 - x[1:N] ** 2), 0.0])
    D4 = (np.diag(1 - x ** 2) @ np.linalg.matrix_power(D, 4) - 8 * np.diag(x) @ np.linalg.matrix_power(D, 3)
          - 12 * D @ D) @ S
    D4 = D4[1:N, 1:N]
    I = np.eye(N - 1)
    U = np.diag(1 - x[1:N] ** 2)
    A = U @ (D2 - al ** 2 * I) + 2 * I - (D4 - 2 * al ** 2 * D2 + al ** 4 * I) / (1j * al * Re)
    B = D2 - al ** 2 * I
    ev = sla.eigvals(A, B)
    ev = ev[np.isfinite(ev)]
    gold = _os_gold()
    assert np.abs(ev - gold).min() < 2e-8


def test_orr_sommerfeld_growth_rate():
    """north_star: the alpha=1 eigenmode at Re=7500 grows at the known rate.  40 full steps of the complete
    nonlinear path (config 2); gates: 1e-6 vs the discrete eigenvalue, 1e-4 vs the closed-form one."""
    c, o = _oracle("cfg2")
    gold = _os_gold()
    sig, v, phi = discrete_os_mode(o.y, o.A1, o.B1, o.A2, o.B2, c["U"], o.kx[1], o.nu, gold)
    assert abs(1j * sig / o.kx[1] - gold) < 1e-6
    V = np.zeros(o.v.shape, complex)
    P = np.zeros(o.v.shape, complex)
    V[0, 1], P[0, 1] = 1e-6 * v, 1e-6 * phi
    o.set_state(V, P, 0 * V, c["U"], c["W"])
    a0 = o.v[0, 1].copy()
    nst = 40
    for _ in range(nst):
        o.step()
    r = np.vdot(a0, o.v[0, 1]) / np.vdot(a0, a0)
    sig_num = np.log(r) / (nst * c["dt"])
    assert abs(sig_num - sig) / abs(sig) < 1e-6
    assert abs(sig_num.real - gold.imag) / gold.imag < 1e-4
    assert abs(sig_num.imag + gold.real) / gold.real < 1e-4
    assert np.abs(o.U - c["U"]).max() < 1e-9  # perturbation is 1e-6: mean flow unchanged to O(1e-12)


def test_stokes_mode_decay_and_second_order_in_time():
    """Viscous decay of one om_y mode with no mean flow: the exact semi-discrete rate is the generalised
    eigenvalue nu*(mu - k^2) of (B2, A2); the implicit part of [34] is second order in dt (reading R3)."""
    import scipy.linalg as sla
    from oracle import compact_fd as cfd
    errs = []
    for dt in (4e-2, 2e-2):
        c = inputs.config("cfg1")
        o = ChannelOracle(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], 20.0, dt)
        a = cfd.band_to_dense(o.A2)[1:-1, 1:-1]
        b = cfd.band_to_dense(o.B2)[1:-1, 1:-1]
        mu, vec = sla.eig(b, a)
        n = np.argmax(mu.real)
        mode = np.r_[0.0, vec[:, n].real, 0.0]
        Om = np.zeros(o.v.shape, complex)
        Om[1, 2] = 1e-8 * mode
        z = np.zeros_like(Om)
        o.set_state(z, z, Om, 0 * c["U"], c["W"])
        nst = int(round(0.4 / dt))
        for _ in range(nst):
            o.step()
        rate = o.nu * (mu[n].real - o.k2[1, 2])
        ratio = np.vdot(Om[1, 2], o.omy[1, 2]).real / np.vdot(Om[1, 2], Om[1, 2]).real
        errs.append(abs(ratio - np.exp(rate * nst * dt)))
        assert errs[-1] < 1e-4
    assert 3.0 < errs[0] / errs[1] < 5.0


def test_nonlinear_terms_match_convective_form_on_polynomials():
    """Sign/index pin for steps 1-5.  For fields that are low-degree polynomials in y the compact rows are
    exact, so h_g and h_v from the rotational form u x omega (reading R1) must equal
    the curl-based right-hand sides of (2.1) written CONVECTIVELY, N = -(u.grad)u:
        h_g = d_z N_x - d_x N_z,    h_v = (d_xx + d_zz) N_y - d_y (d_x N_x + d_z N_z),
    evaluated here with exact polynomial algebra and a brute-force mode convolution
    (grad(|u|^2/2) drops out of both).  PAPER.md L65 (2.1), L78."""
    nx, ny, nz = 8, 17, 8
    y = inputs.mesh_cosine(ny, 0.5)
    o = ChannelOracle(nx, ny, nz, 2 * np.pi, 2 * np.pi, y, 100.0, 1e-3)
    rng = np.random.default_rng(11)
    # two modes + their conjugates; v^ quadratic, om_y^ linear in y (products stay within degree 4)
    modes = {(1, 1): None, (2, -1): None}
    V = np.zeros(o.v.shape, complex)
    Om = np.zeros(o.v.shape, complex)
    poly = {}
    for (p, q) in modes:
        cv = rng.standard_normal(3) + 1j * rng.standard_normal(3)
        cw = rng.standard_normal(2) + 1j * rng.standard_normal(2)
        kx, kz = o.kx[p], 2 * np.pi * q / o.lz
        k2 = kx * kx + kz * kz
        dv = npoly.polyder(cv)
        pu = 1j * (kx * np.r_[dv, 0] - kz * np.r_[cw, 0]) / k2
        pw = 1j * (kz * np.r_[dv, 0] + kx * np.r_[cw, 0]) / k2
        poly[(p, q)] = (kx, kz, pu, cv, pw)
        poly[(-p, -q)] = (-kx, -kz, np.conj(pu), np.conj(cv), np.conj(pw))
        V[q % nz, p] = npoly.polyval(y, cv)
        Om[q % nz, p] = npoly.polyval(y, cw)
    o.v[...] = V
    o.omy[...] = Om
    fields = o.velocities_vorticities()
    H1, H2, H3 = o.nonlinear(fields)
    ikx = 1j * o.kx[None, :, None]
    ikz = 1j * o.kz[:, None, None]
    hg = ikz * H1 - ikx * H3
    hv = -o.k2[:, :, None] * H2 - o.D1(ikx * H1 + ikz * H3)
    # exact: N_i^(k) = -sum_{k'+k''=k} [ (i k''_x u' + i k''_z w') u''_i + v' d_y u''_i ]
    N = {}
    for ka, (kxa, kza, ua, va, wa) in poly.items():
        for kb, (kxb, kzb, ub, vb, wb) in poly.items():
            key = (ka[0] + kb[0], ka[1] + kb[1])
            acc = N.setdefault(key, [np.zeros(1, complex)] * 3)
            new = []
            for comp, fb in enumerate((ub, vb, wb)):
                adv = npoly.polymul(1j * kxb * ua + 1j * kzb * wa, fb)
                adv = npoly.polyadd(adv, npoly.polymul(va, npoly.polyder(fb)))
                new.append(npoly.polyadd(acc[comp], -adv))
            N[key] = new
    checked = 0
    for (p, q), (Nx, Ny_, Nz_) in N.items():
        if p < 0 or (p == 0 and q < 0) or (p, q) == (0, 0) or p >= nx // 2 or abs(q) >= nz // 2:
            continue  # outside the retained set: dropped by the dealiased truncation
        kx, kz = o.kx[p], 2 * np.pi * q / o.lz
        hg_ex = npoly.polyval(y, 1j * kz * Nx - 1j * kx * Nz_)
        inner = npoly.polyadd(1j * kx * Nx, 1j * kz * Nz_)
        hv_ex = npoly.polyval(y, npoly.polyadd(-(kx * kx + kz * kz) * Ny_, -npoly.polyder(inner)))
        sc = max(np.abs(hv_ex).max(), np.abs(hg_ex).max())
        assert np.abs(hg[q % nz, p] - hg_ex).max() < 1e-9 * sc, (p, q)
        assert np.abs(hv[q % nz, p] - hv_ex).max() < 1e-9 * sc, (p, q)
        checked += 1
    assert checked >= 3
