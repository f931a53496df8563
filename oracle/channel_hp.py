"""Extended-precision evaluation of the oracle's substep: the yardstick for fp64 rounding error.

TEST INFRASTRUCTURE (see oracle/__init__.py).  The same discrete problem as ``oracle/channel.py`` --
same band tables, wavenumbers and RK constants, all taken as the DOUBLES the oracle holds (a double is
an exact extended-precision number) -- with every array operation carried out in numpy ``longdouble``
(x87 80-bit: 64-bit mantissa, eps = 1.1e-19) instead of fp64, including the plane transforms
(numpy's pocketfft works natively in long double).  Steps and notation are those of DESIGN.md
"What one substep computes"; nothing here is tuned.

What it is for (SURVEY.md section 7 "hard part 4"): phi^ = lap(v^) is obtained from
Helmholtz problems whose condition number grows like 1/dy_min^2 and from the 2x2 influence matrix, so the
fp64 oracle and the fp64 CUDA path both carry a rounding error on phi^ that can exceed north_star's
1e-11 per substep.  |oracle - hp| measures the oracle's own rounding error on the given data and
|gpu - hp| the kernel's: a parity gate may be widened to a small multiple of the former, never by
comparing two fp64 evaluations with each other.

The scalar problem parameters nu, dt, c = 1/(beta nu dt), lam = k^2 + c, alpha nu dt are formed in fp64
exactly as the oracle (and the library) form them, so that all three evaluations solve the same
discrete systems; only the array arithmetic differs.
"""
import numpy as np

from .channel import RK_ALPHA, RK_BETA, RK_GAMMA, RK_ZETA

LD = np.longdouble
CLD = np.clongdouble


def band_matvec(T, f):
    """(T f)_j = sum_m T[j,3+m] f_{j+m}, y last, in the dtype of the operands."""
    ny = f.shape[-1]
    out = np.zeros(np.broadcast_shapes(f.shape, T.shape[:-1]), dtype=np.result_type(f, T))
    for m in range(-3, 4):
        lo, hi = max(0, -m), min(ny, ny - m)
        out[..., lo:hi] += T[..., lo:hi, 3 + m] * f[..., lo + m:hi + m]
    return out


def banded_solve(T, r):
    """Unpivoted heptadiagonal elimination, rows ascending; T (ny,7) or (batch,ny,7); r (..., ny) or
    (batch, k, ny).  Same algorithm as oracle.compact_fd.banded_solve, dtype preserved."""
    T = np.array(T, dtype=LD, copy=True)
    ny = T.shape[-2]
    batched = T.ndim == 3
    x = np.array(r, copy=True)
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


class ChannelHP:
    """Long-double twin of a ChannelOracle ``o``: copies its tables and parameters, holds its own state."""

    def __init__(self, o):
        self.nx, self.ny, self.nz, self.mx, self.mz = o.nx, o.ny, o.nz, o.mx, o.mz
        self.nu, self.dt, self.forcing = o.nu, o.dt, o.forcing
        self.A1, self.B1, self.A2, self.B2 = (np.asarray(t, dtype=LD) for t in (o.A1, o.B1, o.A2, o.B2))
        self.kx, self.kz = o.kx.astype(LD), o.kz.astype(LD)
        self.k2d = o.k2.copy()                   # fp64, as the oracle forms it
        self.k2 = self.k2d.astype(LD)
        self.w = o.w.astype(LD)
        shp = (o.nz, o.nx // 2, o.ny)
        self.v, self.phi, self.omy = (np.zeros(shp, CLD) for _ in range(3))
        self.U, self.W = np.zeros(o.ny, LD), np.zeros(o.ny, LD)
        self.hv_prev, self.hg_prev = np.zeros(shp, CLD), np.zeros(shp, CLD)
        self.H1m_prev, self.H3m_prev = np.zeros(o.ny, LD), np.zeros(o.ny, LD)
        self.isub, self.Q0, self.pgrad = 0, LD(0), LD(o.pgrad)
        self.nonlinear_override = None           # callable(fields) -> (H1,H2,H3): seeded H of the stage tests

    def set_state(self, v, phi, omy, U, W):
        self.v[...] = v
        self.phi[...] = phi
        self.omy[...] = omy
        self.U[...] = U
        self.W[...] = W
        nzh = self.nz // 2
        for f in (self.v, self.phi, self.omy):
            f[nzh, :, :] = 0.0
            f[0, 0, :] = 0.0
        self.Q0 = self.w @ self.U
        self.isub = 0

    def D1(self, f):
        rhs = band_matvec(self.B1, f)
        shp = rhs.shape
        return banded_solve(self.A1, rhs.reshape(-1, shp[-1])).reshape(shp)

    def velocities_vorticities(self):
        ikx = 1j * self.kx[None, :, None]
        ikz = 1j * self.kz[:, None, None]
        k2 = self.k2.copy()
        k2[0, 0] = 1.0
        k2[self.nz // 2, :] = 1.0
        dv = self.D1(self.v)
        u = (ikx * dv - ikz * self.omy) / k2[:, :, None]
        w = (ikz * dv + ikx * self.omy) / k2[:, :, None]
        v, omy = self.v.copy(), self.omy.copy()
        u[0, 0, :] = self.U
        w[0, 0, :] = self.W
        v[0, 0, :] = 0.0
        omy[0, 0, :] = 0.0
        nzh = self.nz // 2
        for f in (u, v, w, omy):
            f[nzh] = 0.0
        omx = self.D1(w) - ikz * v
        omz = ikx * v - self.D1(u)
        omx[nzh] = 0.0
        omz[nzh] = 0.0
        return u, v, w, omx, omy, omz

    def to_physical(self, f):
        nx, nz, mx, mz, ny = self.nx, self.nz, self.mx, self.mz, self.ny
        pad = np.zeros((ny, mz, mx // 2 + 1), CLD)
        g = np.transpose(f, (2, 0, 1))
        pad[:, : nz // 2, : nx // 2] = g[:, : nz // 2, :]
        pad[:, mz - (nz // 2 - 1):, : nx // 2] = g[:, nz // 2 + 1:, :]
        pz = np.fft.ifft(pad, axis=1) * LD(mz)
        return np.fft.irfft(pz, n=mx, axis=2) * LD(mx)

    def to_spectral(self, r):
        nx, nz, mx, mz = self.nx, self.nz, self.mx, self.mz
        s = np.fft.fft(np.fft.rfft(r, axis=2), axis=1) / LD(mx * mz)
        out = np.zeros((self.ny, nz, nx // 2), CLD)
        out[:, : nz // 2, :] = s[:, : nz // 2, : nx // 2]
        out[:, nz // 2 + 1:, :] = s[:, mz - (nz // 2 - 1):, : nx // 2]
        return np.ascontiguousarray(np.transpose(out, (1, 2, 0)))

    def nonlinear(self, fields):
        if self.nonlinear_override is not None:
            return tuple(np.asarray(h, dtype=CLD) for h in self.nonlinear_override(fields))
        u, v, w, ox, oy, oz = (self.to_physical(f) for f in fields)
        assert u.dtype == LD
        return self.to_spectral(v * oz - w * oy), self.to_spectral(w * ox - u * oz), self.to_spectral(u * oy - v * ox)

    def _helmholtz_matrix(self, lam):
        lam = np.asarray(lam, dtype=LD).reshape(-1)
        M = self.B2[None] - lam[:, None, None] * self.A2[None]
        M[:, 0, :] = 0.0
        M[:, -1, :] = 0.0
        M[:, 0, 3] = 1.0
        M[:, -1, 3] = 1.0
        return M

    def substep(self):
        i = self.isub
        al, be, ga, ze = RK_ALPHA[i], RK_BETA[i], RK_GAMMA[i], RK_ZETA[i]
        nu, dt, ny = self.nu, self.dt, self.ny
        c = 1.0 / (be * nu * dt)                 # fp64 scalars, as in the oracle and the library
        g = al * nu * dt
        nmodes = self.nz * (self.nx // 2)
        ikx = 1j * self.kx[None, :, None]
        ikz = 1j * self.kz[:, None, None]
        k2 = self.k2[:, :, None]
        A2, B2 = self.A2, self.B2
        fields = self.velocities_vorticities()
        H1, H2, H3 = self.nonlinear(fields)
        hg = ikz * H1 - ikx * H3
        hv = -k2 * H2 - self.D1(ikx * H1 + ikz * H3)
        lamd = self.k2d.reshape(-1) + c           # fp64 sum, as in the oracle and the library
        MH = self._helmholtz_matrix(lamd)

        def rhs(x, h, hprev):
            t = x + LD(dt) * (LD(ga) * h + LD(ze) * hprev)
            R = -LD(c) * (band_matvec(A2, t) + LD(g) * (band_matvec(B2, x) - k2 * band_matvec(A2, x)))
            R[..., 0] = 0.0
            R[..., -1] = 0.0
            return R.reshape(nmodes, ny)

        R_om = rhs(self.omy, hg, self.hg_prev)
        R_ph = rhs(self.phi, hv, self.hv_prev)
        ea = np.zeros((nmodes, ny), LD)
        ea[:, 0] = 1.0
        eb = np.zeros((nmodes, ny), LD)
        eb[:, -1] = 1.0
        sol = banded_solve(MH, np.stack([R_om.real, R_om.imag, R_ph.real, R_ph.imag, ea, eb], axis=1))
        omy_new = sol[:, 0] + 1j * sol[:, 1]
        phi_p = sol[:, 2] + 1j * sol[:, 3]
        phi_a, phi_b = sol[:, 4], sol[:, 5]
        MP = self._helmholtz_matrix(self.k2d.reshape(-1))

        def prhs(ph):
            r = band_matvec(A2, ph)
            r[..., 0] = 0.0
            r[..., -1] = 0.0
            return r

        sol = banded_solve(MP, np.stack([prhs(phi_p.real), prhs(phi_p.imag), prhs(phi_a), prhs(phi_b)], axis=1))
        v_p = sol[:, 0] + 1j * sol[:, 1]
        v_a, v_b = sol[:, 2], sol[:, 3]
        dvp, dva, dvb = self.D1(v_p), self.D1(v_a), self.D1(v_b)
        g11, g12, g21, g22 = dva[:, 0], dvb[:, 0], dva[:, -1], dvb[:, -1]
        det = g11 * g22 - g12 * g21
        r1, r2 = -dvp[:, 0], -dvp[:, -1]
        with np.errstate(all="ignore"):
            ca = (g22 * r1 - g12 * r2) / det
            cb = (-g21 * r1 + g11 * r2) / det
        phi_new = phi_p + ca[:, None] * phi_a + cb[:, None] * phi_b
        v_new = v_p + ca[:, None] * v_a + cb[:, None] * v_b

        H1m, H3m = H1[0, 0].real.copy(), H3[0, 0].real.copy()
        Mm = self._helmholtz_matrix(np.array([c]))[0]

        def mean_rhs(X, Hm, Hp):
            R = -LD(c) * (band_matvec(A2, X + LD(dt) * (LD(ga) * Hm + LD(ze) * Hp)) + LD(g) * band_matvec(B2, X))
            R[0] = R[-1] = 0.0
            return R

        Up = banded_solve(Mm, mean_rhs(self.U, H1m, self.H1m_prev))
        one = -LD(c) * band_matvec(A2, np.ones(ny, LD))
        one[0] = one[-1] = 0.0
        Uh = banded_solve(Mm, one)
        if self.forcing == 0:
            Pi = (self.Q0 - self.w @ Up) / (self.w @ Uh)
            self.pgrad = Pi / LD((ga + ze) * dt)
        else:
            Pi = self.pgrad * LD((ga + ze) * dt)
        self.U = Up + Pi * Uh
        self.W = banded_solve(Mm, mean_rhs(self.W, H3m, self.H3m_prev))
        shp = self.v.shape
        self.omy, self.phi, self.v = omy_new.reshape(shp), phi_new.reshape(shp), v_new.reshape(shp)
        nzh = self.nz // 2
        for f in (self.omy, self.phi, self.v):
            f[0, 0, :] = 0.0
            f[nzh] = 0.0
        self.hv_prev, self.hg_prev = hv, hg
        self.H1m_prev, self.H3m_prev = H1m, H3m
        self.isub = (i + 1) % 3

    def step(self):
        assert self.isub == 0
        for _ in range(3):
            self.substep()
