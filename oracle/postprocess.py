"""Oracle of the post-processing that the paper performs on the STORED database (NEXT-2).

TEST INFRASTRUCTURE (see oracle/__init__.py).  PAPER.md section 3.2 (L124-149): from the ten stored variables
u_i, u_i u_j, om_i om_i (filtered, on the retained modes 0 <= p <= Kx, |q| <= Kz, all y) one can compute

* the filtered pressure from the Poisson equation (3.2),  d_kk p = -d_ij(u_i u_j)   (L126-132),
* the norm of the filtered rate-of-strain tensor through the identity (3.3)           (L134, L145),
* the sub-grid stress tensor (3.4),  tau_ij = (u_i u_j) - u_i u_j                    (L149),
* the filtered vorticities om_i = eps_ijk d_j u_k and the kinetic energy E = u_i u_i / 2 (L124),

"without requiring extra information from the small scales" because the sharp cutoff commutes with every derivative.

Readings (R17-R20):
 R17  (3.3) and (3.4) are misprinted (L134: "-2 d_ij(u_i u_j) = S_ij S_ij - om_i om_i"; L149: "u_j u_j").  For a
      solenoidal field  d_ij(u_i u_j) = d_i u_j d_j u_i = S_ij S_ij - Om_ij Om_ij  with Om_ij Om_ij = om_i om_i / 2, so
          S_ij S_ij = d_ij(u_i u_j) + om_i om_i / 2      (and the same for the filtered quantities: all terms are
      linear in the stored variables);   tau_ij = (u_i u_j) - u_i u_j.
 R18  The wall boundary condition of (3.2) is not printed.  The wall-normal momentum equation at a no-slip wall reads
      d_y p = nu d_yy v, so every mode gets the Neumann data  d_y p(+-1) = nu (D1 D1 v)(+-1)  from the stored v.  The
      mode (0,0) is fixed by  p_00 = -(vv)_00 + (vv)_00(-1)  (the mean of (3.2) integrated twice; p_00(-1) = 0).
 R19  Discretisation in y: the same compact operators as the substep.  (D2 - k^2) p = r is multiplied through by A2
      (reading R6) and the Neumann data are imposed with the same three-solution superposition as the influence matrix
      of the substep (step 7): p = p_p + c_a p_a + c_b p_b, (c_a, c_b) from (D1 p)(+-1) = g_+-.  d_yy f = D1(D1 f)
      (the second-derivative rows have no wall closure).
 R20  The product u_i u_j of (3.4) is formed from the STORED (filtered) velocities on a dealiased grid
      (3/2 rule on the stored modes) and tau_ij is returned on the stored modes; modes of u_i u_j beyond the cutoff
      cannot be held by the database and are dropped.

Layout: db[10][ny][2Kz+1][Kx+1] complex, rows q = 0..Kz, -Kz..-1 (the filter's output); variables
0..2 = u,v,w; 3..8 = uu,uv,uw,vv,vw,ww; 9 = om_i om_i.
"""
import numpy as np

from . import compact_fd as cfd

UU, UV, UW, VV, VW, WW, ENS = 3, 4, 5, 6, 7, 8, 9


class DatabaseOracle:
    def __init__(self, y, lx, lz, kx_cut, kz_cut, nu, A1=None, B1=None, A2=None, B2=None):
        self.y = np.asarray(y, dtype=np.float64)
        self.ny = self.y.size
        self.Kx, self.Kz, self.nu = kx_cut, kz_cut, nu
        if A1 is None:
            A1, B1, A2, B2 = cfd.build_operators(self.y)
        self.A1, self.B1, self.A2, self.B2 = A1, B1, A2, B2
        self.q = np.array(list(range(0, kz_cut + 1)) + list(range(-kz_cut, 0)))
        self.kx = 2.0 * np.pi * np.arange(kx_cut + 1) / lx
        self.kz = 2.0 * np.pi * self.q / lz
        self.k2 = self.kz[:, None] ** 2 + self.kx[None, :] ** 2              # [2Kz+1][Kx+1]

    # fields here are [ny][2Kz+1][Kx+1]; the compact operators want y last
    def D1(self, f):
        g = np.moveaxis(f, 0, -1)
        return np.moveaxis(cfd.d1(self.A1, self.B1, np.ascontiguousarray(g)), -1, 0)

    def dx(self, f):
        return 1j * self.kx[None, None, :] * f

    def dz(self, f):
        return 1j * self.kz[None, :, None] * f

    # ------------------------------------------------------------------ (3.2)
    def div_div_stress(self, db):
        """d_ij(u_i u_j) = d_xx uu + d_yy vv + d_zz ww + 2 d_xy uv + 2 d_xz uw + 2 d_yz vw   (L128-132)."""
        return (self.dx(self.dx(db[UU])) + self.D1(self.D1(db[VV])) + self.dz(self.dz(db[WW]))
                + 2.0 * self.dx(self.D1(db[UV])) + 2.0 * self.dx(self.dz(db[UW])) + 2.0 * self.dz(self.D1(db[VW])))

    def wall_dpdy(self, db):
        """Reading R18: d_y p(+-1) = nu d_yy v(+-1); returns (g_minus, g_plus), each [2Kz+1][Kx+1]."""
        d2v = self.D1(self.D1(db[1]))
        return self.nu * d2v[0], self.nu * d2v[-1]

    def poisson_neumann(self, r, g_minus, g_plus):
        """Solve (D2 - k^2) p = r with d_y p(-1) = g_minus, d_y p(+1) = g_plus for every mode but (0,0) (reading R19).

        r: [ny][2Kz+1][Kx+1]; returns p of the same shape with p[:, 0, 0] = 0."""
        ny = self.ny
        nq, npx = self.k2.shape
        nm = nq * npx
        k2 = self.k2.reshape(-1).copy()
        k2[0] = 1.0                                    # placeholder: mode (0,0) is overwritten by the caller
        M = self.B2[None] - k2[:, None, None] * self.A2[None]
        M[:, 0, :] = 0.0
        M[:, -1, :] = 0.0
        M[:, 0, 3] = 1.0
        M[:, -1, 3] = 1.0
        rl = np.moveaxis(r, 0, -1).reshape(nm, ny)     # y last
        rhs = cfd.band_matvec(self.A2, rl)
        rhs[:, 0] = 0.0
        rhs[:, -1] = 0.0
        ea = np.zeros((nm, ny))
        ea[:, 0] = 1.0
        eb = np.zeros((nm, ny))
        eb[:, -1] = 1.0
        sol = cfd.banded_solve(M, np.stack([rhs.real, rhs.imag, ea, eb], axis=1))
        p_p = sol[:, 0] + 1j * sol[:, 1]
        p_a, p_b = sol[:, 2], sol[:, 3]
        dp, da, dbb = (cfd.d1(self.A1, self.B1, f) for f in (p_p, p_a, p_b))
        g11, g12, g21, g22 = da[:, 0], dbb[:, 0], da[:, -1], dbb[:, -1]
        det = g11 * g22 - g12 * g21
        r1 = g_minus.reshape(-1) - dp[:, 0]
        r2 = g_plus.reshape(-1) - dp[:, -1]
        ca = (g22 * r1 - g12 * r2) / det
        cb = (-g21 * r1 + g11 * r2) / det
        p = p_p + ca[:, None] * p_a + cb[:, None] * p_b
        p[0] = 0.0
        return np.moveaxis(p.reshape(nq, npx, ny), -1, 0)

    def filtered_pressure(self, db, wall=None):
        """(3.2): the filtered pressure on the stored modes, [ny][2Kz+1][Kx+1].  wall = (g_minus, g_plus) overrides the
        no-slip Neumann data of reading R18 (used by the pins with flows that are not no-slip)."""
        gm, gp = self.wall_dpdy(db) if wall is None else wall
        p = self.poisson_neumann(-self.div_div_stress(db), gm, gp)
        p[:, 0, 0] = -(db[VV][:, 0, 0] - db[VV][0, 0, 0])
        return p

    # ------------------------------------------------------------------ (3.3), re-derived
    def strain_norm(self, db):
        """Filtered S_ij S_ij = d_ij(u_i u_j) + om_i om_i / 2 (reading R17)."""
        return self.div_div_stress(db) + 0.5 * db[ENS]

    # ------------------------------------------------------------------ L124: trivially derived variables
    def vorticity(self, db):
        u, v, w = db[0], db[1], db[2]
        return self.D1(w) - self.dz(v), self.dz(u) - self.dx(w), self.dx(v) - self.D1(u)

    def kinetic_energy(self, db):
        return 0.5 * (db[UU] + db[VV] + db[WW])

    # ------------------------------------------------------------------ (3.4)
    def _phys(self, f):
        """Stored modes -> real field on the 3/2 grid of the stored modes, [ny][mzs][mxs] (mxs, mzs even)."""
        Kx, Kz = self.Kx, self.Kz
        mxs, mzs = self.sgs_grid()
        pad = np.zeros((self.ny, mzs, mxs // 2 + 1), complex)
        pad[:, : Kz + 1, : Kx + 1] = f[:, : Kz + 1, :]
        if Kz:
            pad[:, mzs - Kz:, : Kx + 1] = f[:, Kz + 1:, :]
        return np.fft.irfft(np.fft.ifft(pad, axis=1) * mzs, n=mxs, axis=2) * mxs

    def _spec(self, r):
        Kx, Kz = self.Kx, self.Kz
        mxs, mzs = self.sgs_grid()
        s = np.fft.fft(np.fft.rfft(r, axis=2), axis=1) / (mxs * mzs)
        rows = [qq % mzs for qq in self.q]
        return s[:, rows, : Kx + 1]

    def sgs_grid(self):
        """Smallest even grid that holds the product of two stored fields without aliasing into the stored modes:
        3 K + 1 points suffice for modes |k| <= K (3/2 rule); rounded up to an even number >= 4."""
        ev = lambda n: max(4, n + (n & 1))
        return ev(3 * self.Kx + 2), ev(3 * self.Kz + 2)

    def sgs_tensor(self, db):
        """(3.4) with reading R17/R20: tau[6][ny][2Kz+1][Kx+1] in the order uu,uv,uw,vv,vw,ww."""
        u, v, w = (self._phys(db[n]) for n in range(3))
        prods = (u * u, u * v, u * w, v * v, v * w, w * w)
        return np.stack([db[3 + n] - self._spec(pr) for n, pr in enumerate(prods)])
