"""Oracle of one semi-implicit RK3 substep, the low-storage filter and the plane statistics.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Follows PAPER.md section 2.1 (L61-80: plane channel,
periodic x,z, walls at y=+-1, constant mass flux; (omega_y, lap v) formulation of [20]; Fourier x,z
with zero-padding dealiasing; compact finite differences in y; semi-implicit low-storage RK3 [34])
and section 3.2 (L124: sharp Fourier cutoff, ten stored variables), step by step in the order and
notation of DESIGN.md "What one substep computes" (steps 1-9), with the readings R1-R17 listed there.

Layouts (same as the C ABI): spectral fields are complex128 ``[nz][nx/2][ny]`` (y fastest),
k_z in FFT order (0..nz/2-1, nz/2 (always zero), -nz/2+1..-1), k_x index p = 0..nx/2-1.
"""
import numpy as np

from . import compact_fd as cfd

# Reading R3 -- constants of the three-substep scheme of [34] (PAPER.md L80 cites it, prints none).
RK_GAMMA = (8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0)
RK_ZETA = (0.0, -17.0 / 60.0, -5.0 / 12.0)
RK_ALPHA = (29.0 / 96.0, -3.0 / 40.0, 1.0 / 6.0)
RK_BETA = (37.0 / 160.0, 5.0 / 24.0, 1.0 / 6.0)


def wavenumbers(nx, nz, lx, lz):
    """k_x[p], k_z[slot], and the integer q of every k_z slot (reading R2)."""
    p = np.arange(nx // 2)
    q = np.concatenate([np.arange(nz // 2), [0], np.arange(-nz // 2 + 1, 0)])
    return 2.0 * np.pi * p / lx, 2.0 * np.pi * q / lz, q


def trapezoid_weights(y):
    """Reading R8: Q = sum_j w_j U_j, trapezoid rule on the mesh."""
    w = np.zeros_like(y)
    dy = np.diff(y)
    w[:-1] += 0.5 * dy
    w[1:] += 0.5 * dy
    return w


class ChannelOracle:
    def __init__(self, nx, ny, nz, lx, lz, y, re_tau, dt, forcing=0, half_lhs=3, half_rhs=3):
        assert nx % 2 == 0 and nz % 2 == 0
        self.nx, self.ny, self.nz = nx, ny, nz
        self.mx, self.mz = 3 * nx // 2, 3 * nz // 2
        self.lx, self.lz = float(lx), float(lz)
        self.y = np.asarray(y, dtype=np.float64).copy()
        assert self.y.shape == (ny,)
        self.nu = 1.0 / re_tau  # reading R9
        self.dt = float(dt)
        self.forcing = forcing  # 0: constant mass flux; 1: constant pressure gradient
        self.A1, self.B1, self.A2, self.B2 = cfd.build_operators(self.y, half_lhs, half_rhs)
        self.kx, self.kz, self.q = wavenumbers(nx, nz, lx, lz)
        self.k2 = self.kz[:, None] ** 2 + self.kx[None, :] ** 2  # [nz][nx/2]
        self.w = trapezoid_weights(self.y)
        shp = (nz, nx // 2, ny)
        self.v = np.zeros(shp, complex)
        self.phi = np.zeros(shp, complex)
        self.omy = np.zeros(shp, complex)
        self.U = np.zeros(ny)
        self.W = np.zeros(ny)
        self.hv_prev = np.zeros(shp, complex)
        self.hg_prev = np.zeros(shp, complex)
        self.H1m_prev = np.zeros(ny)
        self.H3m_prev = np.zeros(ny)
        self.isub = 0
        self.Q0 = 0.0
        self.pgrad = 0.0  # forcing==1: prescribed -dP/dx; forcing==0: last recovered value
        self.stat_sum = np.zeros((10, ny))
        self.stat_n = 0

    # ------------------------------------------------------------------ state
    def set_state(self, v, phi, omy, U, W):
        self.v[...] = v
        self.phi[...] = phi
        self.omy[...] = omy
        self.U[...] = U
        self.W[...] = W
        nzh = self.nz // 2
        for f in (self.v, self.phi, self.omy):
            f[nzh, :, :] = 0.0  # z-Nyquist slot is always zero (reading R2)
            f[0, 0, :] = 0.0    # the (0,0) mode lives in U, W
        self.Q0 = float(self.w @ self.U)
        self.isub = 0

    # ------------------------------------------------------------------ step 1
    def D1(self, f):
        return cfd.d1(self.A1, self.B1, f)

    def velocities_vorticities(self):
        """Step 1: (u,v,w,om_x,om_y,om_z) spectral, line layout, from the state (readings R1, R7)."""
        ikx = 1j * self.kx[None, :, None]
        ikz = 1j * self.kz[:, None, None]
        k2 = self.k2.copy()
        k2[0, 0] = 1.0  # placeholder, overwritten below
        k2[self.nz // 2, :] = 1.0  # Nyquist slot holds zeros; avoid 0/0 at p = 0 only cosmetically
        dv = self.D1(self.v)
        u = (ikx * dv - ikz * self.omy) / k2[:, :, None]
        w = (ikz * dv + ikx * self.omy) / k2[:, :, None]
        v = self.v.copy()
        omy = self.omy.copy()
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

    # ------------------------------------------------------------------ steps 2-4
    def to_physical(self, f):
        """Step 2: zero-pad to (mz, mx/2+1), inverse DFT in z then real inverse in x, no normalisation.

        Input ``[nz][nx/2][ny]``; output real ``[ny][mz][mx]``.
        """
        nx, nz, mx, mz, ny = self.nx, self.nz, self.mx, self.mz, self.ny
        pad = np.zeros((ny, mz, mx // 2 + 1), complex)
        g = np.transpose(f, (2, 0, 1))  # [y][kz slot][p]
        pad[:, : nz // 2, : nx // 2] = g[:, : nz // 2, :]
        pad[:, mz - (nz // 2 - 1):, : nx // 2] = g[:, nz // 2 + 1:, :]
        pz = np.fft.ifft(pad, axis=1) * mz
        return np.fft.irfft(pz, n=mx, axis=2) * mx

    def to_spectral(self, r, kx_keep=None, kz_keep=None):
        """Step 4: F(p,q) = 1/(mx mz) sum_n sum_m r e^{-i(kx x_n + kz z_m)}, retained modes only.

        Input real ``[ny][mz][mx]``; output ``[nz][nx/2][ny]`` (default), or, with integer cutoffs,
        ``[ny][2 kz_keep + 1][kx_keep + 1]`` in the filter's layout (q = 0..Kz, -Kz..-1).
        """
        nx, nz, mx, mz = self.nx, self.nz, self.mx, self.mz
        s = np.fft.fft(np.fft.rfft(r, axis=2), axis=1) / (mx * mz)
        if kx_keep is None:
            out = np.zeros((self.ny, nz, nx // 2), complex)
            out[:, : nz // 2, :] = s[:, : nz // 2, : nx // 2]
            out[:, nz // 2 + 1:, :] = s[:, mz - (nz // 2 - 1):, : nx // 2]
            return np.ascontiguousarray(np.transpose(out, (1, 2, 0)))
        rows = [qq % mz for qq in list(range(0, kz_keep + 1)) + list(range(-kz_keep, 0))]
        return np.ascontiguousarray(s[:, rows, : kx_keep + 1])

    def nonlinear(self, fields):
        """Steps 2-4 (reading R1, rotational form): H = u x omega on the dealiased grid -> spectral."""
        u, v, w, ox, oy, oz = (self.to_physical(f) for f in fields)
        H1 = v * oz - w * oy
        H2 = w * ox - u * oz
        H3 = u * oy - v * ox
        return self.to_spectral(H1), self.to_spectral(H2), self.to_spectral(H3)

    # ------------------------------------------------------------------ steps 5-9
    def _helmholtz_matrix(self, lam):
        """Band table of B2 - lam*A2 (rows 1..ny-2) with identity Dirichlet rows 0, ny-1 (step 6)."""
        lam = np.asarray(lam, dtype=np.float64).reshape(-1)
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
        c = 1.0 / (be * nu * dt)
        nmodes = self.nz * (self.nx // 2)
        ikx = 1j * self.kx[None, :, None]
        ikz = 1j * self.kz[:, None, None]
        k2 = self.k2[:, :, None]
        A2, B2 = self.A2, self.B2

        # steps 1-4
        fields = self.velocities_vorticities()
        H1, H2, H3 = self.nonlinear(fields)
        # step 5
        hg = ikz * H1 - ikx * H3
        hv = -k2 * H2 - self.D1(ikx * H1 + ikz * H3)

        # step 6: Helmholtz problems, one real matrix per mode
        k2f = self.k2.reshape(-1)
        MH = self._helmholtz_matrix(k2f + c)

        def rhs(x, h, hprev):
            t = x + dt * (ga * h + ze * hprev)
            R = -c * (cfd.band_matvec(A2, t) + al * nu * dt * (cfd.band_matvec(B2, x) - k2 * cfd.band_matvec(A2, x)))
            R[..., 0] = 0.0
            R[..., -1] = 0.0
            return R.reshape(nmodes, ny)

        R_om = rhs(self.omy, hg, self.hg_prev)
        R_ph = rhs(self.phi, hv, self.hv_prev)
        ea = np.zeros((nmodes, ny))
        ea[:, 0] = 1.0
        eb = np.zeros((nmodes, ny))
        eb[:, -1] = 1.0
        stack = np.stack([R_om.real, R_om.imag, R_ph.real, R_ph.imag, ea, eb], axis=1)
        sol = cfd.banded_solve(MH, stack)
        omy_new = sol[:, 0] + 1j * sol[:, 1]
        phi_p = sol[:, 2] + 1j * sol[:, 3]
        phi_a, phi_b = sol[:, 4], sol[:, 5]

        # step 7: Poisson problems and the influence matrix
        MP = self._helmholtz_matrix(k2f)

        def prhs(ph):
            r = cfd.band_matvec(A2, ph)
            r[..., 0] = 0.0
            r[..., -1] = 0.0
            return r

        stack = np.stack([prhs(phi_p.real), prhs(phi_p.imag), prhs(phi_a), prhs(phi_b)], axis=1)
        sol = cfd.banded_solve(MP, stack)
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

        # step 8: mean mode (p,q) = (0,0)
        H1m, H3m = H1[0, 0].real.copy(), H3[0, 0].real.copy()
        Mm = self._helmholtz_matrix(np.array([c]))[0]

        def mean_rhs(X, Hm, Hp):
            R = -c * (cfd.band_matvec(A2, X + dt * (ga * Hm + ze * Hp)) + al * nu * dt * cfd.band_matvec(B2, X))
            R[0] = R[-1] = 0.0
            return R

        Up = cfd.banded_solve(Mm, mean_rhs(self.U, H1m, self.H1m_prev))
        one = -c * cfd.band_matvec(A2, np.ones(ny))
        one[0] = one[-1] = 0.0
        Uh = cfd.banded_solve(Mm, one)
        if self.forcing == 0:
            Pi = (self.Q0 - self.w @ Up) / (self.w @ Uh)
            self.pgrad = Pi / ((ga + ze) * dt)
        else:
            Pi = self.pgrad * (ga + ze) * dt
        U_new = Up + Pi * Uh
        W_new = cfd.banded_solve(Mm, mean_rhs(self.W, H3m, self.H3m_prev))

        # step 9 and state update
        shp = self.v.shape
        self.omy = omy_new.reshape(shp)
        self.phi = phi_new.reshape(shp)
        self.v = v_new.reshape(shp)
        nzh = self.nz // 2
        for f in (self.omy, self.phi, self.v):
            f[0, 0, :] = 0.0
            f[nzh] = 0.0
        self.U, self.W = U_new, W_new
        self.hv_prev, self.hg_prev = hv, hg
        self.H1m_prev, self.H3m_prev = H1m, H3m
        self.isub = (i + 1) % 3

    def step(self):
        assert self.isub == 0
        for _ in range(3):
            self.substep()

    # ------------------------------------------------------------------ filter and statistics
    def filter_store(self, kx_cut, kz_cut, single=False):
        """ten variables, sharp cutoff 0<=p<=kx_cut, |q|<=kz_cut (readings R11, R12).

        Returns ``[10][ny][2 kz_cut + 1][kx_cut + 1]`` complex: u,v,w, uu,uv,uw,vv,vw,ww, om_i om_i.
        Products are formed on the dealiased grid at full resolution and truncated afterwards.
        ``single``: the database as the paper stores it -- about four bytes per value (150 TB for
        3900 snapshots of ten 1024^3-point variables; reading R13) -- i.e. the fp64 result rounded ONCE, to nearest
        even, to IEEE binary32 per component (complex64).
        """
        assert 0 <= kx_cut <= self.nx // 2 - 1 and 0 <= kz_cut <= self.nz // 2 - 1
        u, v, w, ox, oy, oz = self.velocities_vorticities()
        slots = [qq % self.nz for qq in list(range(0, kz_cut + 1)) + list(range(-kz_cut, 0))]
        out = np.zeros((10, self.ny, 2 * kz_cut + 1, kx_cut + 1), complex)
        for n, f in enumerate((u, v, w)):
            out[n] = np.transpose(f[slots][:, : kx_cut + 1, :], (2, 0, 1))
        pu, pv, pw, pox, poy, poz = (self.to_physical(f) for f in (u, v, w, ox, oy, oz))
        prods = (pu * pu, pu * pv, pu * pw, pv * pv, pv * pw, pw * pw, pox * pox + poy * poy + poz * poz)
        for n, pr in enumerate(prods):
            out[3 + n] = self.to_spectral(pr, kx_cut, kz_cut)
        return out.astype(np.complex64) if single else out

    def run(self, nsteps, filter_every, stats_every, kx_cut, kz_cut, single=False):
        """Snapshot cadence (the filtered fields are stored every Delta t_e, a multiple of the time
        step; L47: statistics on the fly): ``nsteps`` full steps; before step n the filtered database of the current
        state is emitted when n % filter_every == 0 and the statistics are accumulated when n % stats_every == 0
        (0 = never).  Returns the list of emitted databases."""
        snaps = []
        for n in range(nsteps):
            if stats_every and n % stats_every == 0:
                self.stats_accumulate()
            if filter_every and n % filter_every == 0:
                snaps.append(self.filter_store(kx_cut, kz_cut, single))
            self.step()
        return snaps

    def stats_profiles(self):
        """<u_i>, <u_i u_j>, <om_i om_i> per y-plane by Parseval sums over the retained modes."""
        u, v, w, ox, oy, oz = self.velocities_vorticities()
        wp = np.full(self.nx // 2, 2.0)
        wp[0] = 1.0

        def mean(a, b):
            return np.einsum("p,qpy->y", wp, (a * np.conj(b)).real)

        prof = np.zeros((10, self.ny))
        prof[0], prof[1], prof[2] = u[0, 0].real, v[0, 0].real, w[0, 0].real
        pairs = ((u, u), (u, v), (u, w), (v, v), (v, w), (w, w))
        for n, (a, b) in enumerate(pairs):
            prof[3 + n] = mean(a, b)
        prof[9] = mean(ox, ox) + mean(oy, oy) + mean(oz, oz)
        return prof

    def spectra(self):
        """One-dimensional co-spectra of the seven second-order quantities uu,uv,uw,vv,vw,ww, om_i om_i at every y
        (Fig. 3.1, L163/L173 Fig. 3.3 show such spectra of the database): E_x[n][y][p] = w_p sum over k_z
        slots of Re(a conj b), E_z[n][y][slot] = sum over p of w_p Re(a conj b), w_0 = 1, w_p = 2.  Summed over their
        wavenumber both give the plane statistics <a b>(y)."""
        u, v, w, ox, oy, oz = self.velocities_vorticities()
        wp = np.full(self.nx // 2, 2.0)
        wp[0] = 1.0
        pairs = ((u, u), (u, v), (u, w), (v, v), (v, w), (w, w))
        dens = [(a * np.conj(b)).real for a, b in pairs]
        dens.append((ox * np.conj(ox)).real + (oy * np.conj(oy)).real + (oz * np.conj(oz)).real)
        ex = np.stack([np.transpose(wp[:, None] * d.sum(axis=0), (1, 0)) for d in dens])            # [7][ny][nx/2]
        ez = np.stack([np.transpose(np.einsum("p,qpy->qy", wp, d), (1, 0)) for d in dens])           # [7][ny][nz]
        return ex, ez

    def stats_accumulate(self):
        self.stat_sum += self.stats_profiles()
        self.stat_n += 1

    def stats_read(self):
        return self.stat_sum.copy(), self.stat_n

    def stats_reset(self):
        self.stat_sum[...] = 0.0
        self.stat_n = 0

    # ------------------------------------------------------------------ diagnostics used by the pins
    def divergence(self):
        u, v, w, *_ = self.velocities_vorticities()
        return 1j * self.kx[None, :, None] * u + self.D1(v) + 1j * self.kz[:, None, None] * w
