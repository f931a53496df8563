"""Discrete Orr-Sommerfeld eigenmode of the oracle's own operators (test infrastructure).

BASELINE.json config 2 / north_star: "a single Orr-Sommerfeld eigenmode at Re=7500, alpha=1 grows at
the known rate".  The initial condition must be an eigenvector of the *discrete* linearised operator
(compact D1, A2/B2 of oracle.compact_fd; rotational form with om_z from D1 of u, readings R1, R7),
otherwise the measured growth is polluted by the other modes.  Linearising steps 1-7 of
oracle.channel about U(y), for a mode (kx, kz=0) with om_y = 0:

    u = i D1 v / kx,     om_z' = ikx v - D1 u = -(i/kx)(D1 D1 - kx^2) v,     Om_z = -D1 U
    H1 = v Om_z,   H2 = -U om_z' - u Om_z,   h_v = -kx^2 H2 - D1(ikx H1)
    sigma A2 phi = A2 h_v(v) + nu (B2 - kx^2 A2) phi      rows 1..ny-2
    0 = (B2 - kx^2 A2) v - A2 phi                         rows 1..ny-2
    v(+-1) = 0, (D1 v)(+-1) = 0

solved as a dense generalised eigenproblem (scipy.linalg.eig).  sigma = -i kx c.
"""
import numpy as np
import scipy.linalg as sla

from . import compact_fd as cfd


def discrete_os_mode(y, A1, B1, A2, B2, U, kx, nu, c_guess):
    ny = y.size
    a1, b1, a2, b2 = (cfd.band_to_dense(T) for T in (A1, B1, A2, B2))
    D1 = np.linalg.solve(a1, b1)
    dU = D1 @ U
    k2 = kx * kx
    lap1 = D1 @ D1 - k2 * np.eye(ny)
    H2 = (1j / kx) * (np.diag(U) @ lap1 + np.diag(dU) @ D1)
    H1 = -np.diag(dU)
    Nv = -k2 * H2 - D1 @ (1j * kx * H1)
    L = np.zeros((2 * ny, 2 * ny), complex)
    M = np.zeros((2 * ny, 2 * ny), complex)
    P = b2 - k2 * a2
    r = 0
    for j in range(1, ny - 1):  # phi equation
        L[r, :ny] = (a2 @ Nv)[j]
        L[r, ny:] = nu * P[j]
        M[r, ny:] = a2[j]
        r += 1
    for j in range(1, ny - 1):  # Poisson rows
        L[r, :ny] = P[j]
        L[r, ny:] = -a2[j]
        r += 1
    L[r, 0] = 1.0; r += 1
    L[r, ny - 1] = 1.0; r += 1
    L[r, :ny] = D1[0]; r += 1
    L[r, :ny] = D1[ny - 1]; r += 1
    assert r == 2 * ny
    sig, vec = sla.eig(L, M)
    ok = np.isfinite(sig)
    sig, vec = sig[ok], vec[:, ok]
    target = -1j * kx * c_guess
    n = int(np.argmin(np.abs(sig - target)))
    v, phi = vec[:ny, n], vec[ny:, n]
    s = v[np.argmax(np.abs(v))]
    return sig[n], v / s, phi / s
