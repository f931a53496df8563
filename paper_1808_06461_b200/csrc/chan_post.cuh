// Post-processing of the stored database (NEXT-2; section 3.2): filtered pressure from the
// Poisson equation (3.2), norm of the filtered rate of strain through the identity (3.3) as re-derived in DESIGN.md
// reading R17, sub-grid stresses (3.4).  Readings R17-R20 of DESIGN.md.
//
// The database is small (0 <= p <= Kx, |q| <= Kz: 1.5% of the modes at config 5) and this runs once per stored
// snapshot, off the time-stepping path: one thread per stored mode marches along y through global scratch arrays
// laid out [ny][modes] (consecutive lanes = consecutive modes: coalesced), with the same compact operators, the same
// unpivoted band elimination and the same three-solution superposition for the wall conditions as the substep.
#pragma once
#include <cuda_runtime.h>

#include "chan_ykernels.cuh"

namespace chn {

struct PostParams {
    int ny, nr, npk, kzc;      // database planes are [nr = 2 kzc + 1][npk = kxc + 1]
    int nz;                    // z slots of the handle (for the k_z table)
    const double* B1;          // [ny][8] orientation 0
    const double* lu1;         // [ny][8] LU of A1: l1,l2,l3,1/u,u1,u2,u3
    const double* A2;          // [ny][8]
    const double* B2;          // [ny][8]
    const double* kx;          // [nxh]
    const double* kz;          // [nz]
    const double* wm;          // [ny] (D1 f)(-1) = wm . f
    const double* wp;          // [ny]
    double nu;
};

__device__ __forceinline__ c2 cscale(double s, c2 a) { return mk(s * a.x, s * a.y); }

// g = D1 f = A1^-1 B1 f for one mode: f(j) is read through `get`, g is left in out[j * stride]
template <class Get>
__device__ void post_d1(const PostParams& P, Get get, double2* out, size_t stride) {
    const int ny = P.ny;
    c2 z1 = mk(0, 0), z2 = mk(0, 0), z3 = mk(0, 0);
    for (int j = 0; j < ny; ++j) {
        c2 r = mk(0, 0);
        for (int m = -3; m <= 3; ++m) {
            const int jj = j + m;
            if (jj >= 0 && jj < ny) r = r + cscale(__ldg(P.B1 + (size_t)j * 8 + 3 + m), get(jj));
        }
        const double* lu = P.lu1 + (size_t)j * 8;
        const c2 z = r - cscale(__ldg(lu + 0), z1) - cscale(__ldg(lu + 1), z2) - cscale(__ldg(lu + 2), z3);
        z3 = z2; z2 = z1; z1 = z;
        stc(out + (size_t)j * stride, z);
    }
    c2 g1 = mk(0, 0), g2 = mk(0, 0), g3 = mk(0, 0);
    for (int j = ny - 1; j >= 0; --j) {
        const double* lu = P.lu1 + (size_t)j * 8;
        const c2 z = ldc(out + (size_t)j * stride);
        const c2 g = cscale(__ldg(lu + 3), z - cscale(__ldg(lu + 4), g1) - cscale(__ldg(lu + 5), g2) - cscale(__ldg(lu + 6), g3));
        g3 = g2; g2 = g1; g1 = g;
        stc(out + (size_t)j * stride, g);
    }
}

// Mode m of the database -> (row rr, column p), wavenumbers.
__device__ __forceinline__ void post_mode(const PostParams& P, int m, int& rr, int& p, double& kx, double& kz) {
    rr = m / P.npk; p = m - rr * P.npk;
    const int s = (rr <= P.kzc) ? rr : P.nz - (P.nr - rr);
    kx = __ldg(P.kx + p); kz = __ldg(P.kz + s);
}

// R = d_ij(u_i u_j) = D1( D1(vv) + 2 i (kx uv + kz vw) ) - kx^2 uu - kz^2 ww - 2 kx kz uw   (3.2), into R[ny][modes].
// s0: scratch [ny][modes].  With ens != nullptr the output is the strain norm R + ens/2 instead (3.3, reading R17).
__global__ void __launch_bounds__(128) k_post_divdiv(PostParams P, const double2* __restrict__ db, double2* s0, double2* R, int add_half_ens) {
    const int nm = P.nr * P.npk;
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= nm) return;
    int rr, p; double kx, kz;
    post_mode(P, m, rr, p, kx, kz);
    const size_t per = (size_t)P.ny * nm, st = (size_t)nm;
    const double2* uu = db + 3 * per + m; const double2* uv = db + 4 * per + m; const double2* uw = db + 5 * per + m;
    const double2* vv = db + 6 * per + m; const double2* vw = db + 7 * per + m; const double2* ww = db + 8 * per + m;
    const double2* ens = db + 9 * per + m;
    post_d1(P, [&](int j) { return ldc(vv + (size_t)j * st); }, s0 + m, st);
    post_d1(P, [&](int j) {
        const c2 a = ldc(uv + (size_t)j * st), b = ldc(vw + (size_t)j * st), e = ldc(s0 + m + (size_t)j * st);
        const c2 c = mk(kx * a.x + kz * b.x, kx * a.y + kz * b.y);          // kx uv + kz vw
        return mk(e.x - 2.0 * c.y, e.y + 2.0 * c.x);                        // e + 2 i c
    }, R + m, st);
    for (int j = 0; j < P.ny; ++j) {
        const size_t o = (size_t)j * st;
        c2 r = ldc(R + m + o) - cscale(kx * kx, ldc(uu + o)) - cscale(kz * kz, ldc(ww + o)) - cscale(2.0 * kx * kz, ldc(uw + o));
        if (add_half_ens) r = r + cscale(0.5, ldc(ens + o));
        stc(R + m + o, r);
    }
}

// Pressure of one mode: (B2 - k^2 A2) p_s = A2 (-R) on the interior rows, p_s(+-1) Dirichlet (0,0), (1,0), (0,1);
// p = p_p + c_a p_a + c_b p_b with (D1 p)(+-1) = nu (D1 D1 v)(+-1)  (readings R18, R19).
// R: [ny][modes] from k_post_divdiv; scratch s0, s1 (complex), s2 (two reals), f0, f1 (factor rows), all [ny][modes];
// p: output [ny][modes].
__global__ void __launch_bounds__(128) k_post_pressure(PostParams P, const double2* __restrict__ db, const double2* __restrict__ R,
                                                       double2* s0, double2* s2, double2* f0, double2* f1, double2* __restrict__ p_out) {
    const int nm = P.nr * P.npk, ny = P.ny;
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= nm) return;
    int rr, p; double kx, kz;
    post_mode(P, m, rr, p, kx, kz);
    const size_t per = (size_t)ny * nm, st = (size_t)nm;
    if (m == 0) {        // mode (0,0): p = -(vv) + (vv)(-1)
        const double2* vv = db + 6 * per;
        const c2 v0 = ldc(vv);
        for (int j = 0; j < ny; ++j) { const c2 a = ldc(vv + (size_t)j * st); stc(p_out + (size_t)j * st, mk(v0.x - a.x, v0.y - a.y)); }
        return;
    }
    const double k2 = kx * kx + kz * kz;
    // wall data: g = nu (D1 D1 v)(+-1) = nu w . (D1 v)
    const double2* v = db + 1 * per + m;
    post_d1(P, [&](int j) { return ldc(v + (size_t)j * st); }, s0 + m, st);
    c2 gm = mk(0, 0), gp = mk(0, 0);
    for (int j = 0; j < ny; ++j) {
        const c2 d = ldc(s0 + m + (size_t)j * st);
        gm = gm + cscale(__ldg(P.wm + j), d); gp = gp + cscale(__ldg(P.wp + j), d);
    }
    gm = cscale(P.nu, gm); gp = cscale(P.nu, gp);
    // forward elimination of the three right-hand sides with the factorisation of B2 - k^2 A2
    double di[3] = {1, 1, 1}, u1[3] = {0, 0, 0}, u2[3] = {0, 0, 0}, u3[3] = {0, 0, 0};     // rows j-1, j-2, j-3
    c2 zp[3] = {mk(0, 0), mk(0, 0), mk(0, 0)};
    double za[3] = {0, 0, 0}, zb[3] = {0, 0, 0};
    for (int j = 0; j < ny; ++j) {
        double a[7];
        const bool wall = (j == 0 || j == ny - 1);
        for (int k = 0; k < 7; ++k) a[k] = wall ? (k == 3 ? 1.0 : 0.0) : __ldg(P.B2 + (size_t)j * 8 + k) - k2 * __ldg(P.A2 + (size_t)j * 8 + k);
        c2 r = mk(0, 0);
        if (!wall)
            for (int mm = -3; mm <= 3; ++mm) {
                const int jj = j + mm;
                if (jj >= 0 && jj < ny) r = r - cscale(__ldg(P.A2 + (size_t)j * 8 + 3 + mm), ldc(R + m + (size_t)jj * st));
            }
        const double l3 = a[0] * di[2];
        a[1] -= l3 * u1[2]; a[2] -= l3 * u2[2]; a[3] -= l3 * u3[2];
        const double l2 = a[1] * di[1];
        a[2] -= l2 * u1[1]; a[3] -= l2 * u2[1]; a[4] -= l2 * u3[1];
        const double l1 = a[2] * di[0];
        a[3] -= l1 * u1[0]; a[4] -= l1 * u2[0]; a[5] -= l1 * u3[0];
        const double d = 1.0 / a[3];
        const c2 z = r - cscale(l3, zp[2]) - cscale(l2, zp[1]) - cscale(l1, zp[0]);
        const double ea = (j == 0) ? 1.0 : 0.0, eb = (j == ny - 1) ? 1.0 : 0.0;
        const double ya = ea - l3 * za[2] - l2 * za[1] - l1 * za[0], yb = eb - l3 * zb[2] - l2 * zb[1] - l1 * zb[0];
        di[2] = di[1]; u1[2] = u1[1]; u2[2] = u2[1]; u3[2] = u3[1];
        di[1] = di[0]; u1[1] = u1[0]; u2[1] = u2[0]; u3[1] = u3[0];
        di[0] = d; u1[0] = a[4]; u2[0] = a[5]; u3[0] = a[6];
        zp[2] = zp[1]; zp[1] = zp[0]; zp[0] = z;
        za[2] = za[1]; za[1] = za[0]; za[0] = ya;
        zb[2] = zb[1]; zb[1] = zb[0]; zb[0] = yb;
        const size_t o = m + (size_t)j * st;
        stc(s0 + o, z); s2[o] = make_double2(ya, yb);
        f0[o] = make_double2(d, a[4]); f1[o] = make_double2(a[5], a[6]);
    }
    // back substitution; wall derivatives through the functionals wm, wp
    c2 xp[3] = {mk(0, 0), mk(0, 0), mk(0, 0)};
    double xa[3] = {0, 0, 0}, xb[3] = {0, 0, 0};
    c2 dpm = mk(0, 0), dpp = mk(0, 0);
    double dam = 0, dap = 0, dbm = 0, dbp = 0;
    for (int j = ny - 1; j >= 0; --j) {
        const size_t o = m + (size_t)j * st;
        const double2 fa = f0[o], fb = f1[o];
        const c2 z = ldc(s0 + o); const double2 zab = s2[o];
        const c2 x = cscale(fa.x, z - cscale(fa.y, xp[0]) - cscale(fb.x, xp[1]) - cscale(fb.y, xp[2]));
        const double ya = (zab.x - fa.y * xa[0] - fb.x * xa[1] - fb.y * xa[2]) * fa.x;
        const double yb = (zab.y - fa.y * xb[0] - fb.x * xb[1] - fb.y * xb[2]) * fa.x;
        xp[2] = xp[1]; xp[1] = xp[0]; xp[0] = x;
        xa[2] = xa[1]; xa[1] = xa[0]; xa[0] = ya;
        xb[2] = xb[1]; xb[1] = xb[0]; xb[0] = yb;
        const double wmj = __ldg(P.wm + j), wpj = __ldg(P.wp + j);
        dpm = dpm + cscale(wmj, x); dpp = dpp + cscale(wpj, x);
        dam += wmj * ya; dap += wpj * ya; dbm += wmj * yb; dbp += wpj * yb;
        stc(s0 + o, x); s2[o] = make_double2(ya, yb);
    }
    const double det = dam * dbp - dbm * dap;
    const c2 r1 = gm - dpm, r2 = gp - dpp;
    const c2 ca = cscale(1.0 / det, cscale(dbp, r1) - cscale(dbm, r2));
    const c2 cb = cscale(1.0 / det, cscale(dam, r2) - cscale(dap, r1));
    for (int j = 0; j < ny; ++j) {
        const size_t o = m + (size_t)j * st;
        const c2 x = ldc(s0 + o); const double2 ab = s2[o];
        stc(p_out + o, x + cscale(ab.x, ca) + cscale(ab.y, cb));
    }
}

// (3.4), first half: the stored velocities into the plane-layout fields u, v, w of a handle (zeros elsewhere; the
// fields were cleared by the caller); [ny][nr][npk] -> [ny][nz][nxh]
__global__ void k_post_scatter(PostParams P, int nxh, const double2* __restrict__ db, double2* __restrict__ u, double2* __restrict__ v, double2* __restrict__ w) {
    const size_t nmf = (size_t)P.nr * P.npk, per = (size_t)P.ny * nmf, nm = (size_t)P.nz * nxh;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < per; e += (size_t)gridDim.x * blockDim.x) {
        const int j = (int)(e / nmf);
        const size_t rem = e - (size_t)j * nmf;
        const int rr = (int)(rem / P.npk), p = (int)(rem - (size_t)rr * P.npk);
        const int s = (rr <= P.kzc) ? rr : P.nz - (P.nr - rr);
        const size_t o = (size_t)j * nm + (size_t)s * nxh + p;
        u[o] = db[e]; v[o] = db[per + e]; w[o] = db[2 * per + e];
    }
}
// (3.4), second half: tau = stored products - products of the stored velocities, six planes sets [ny][nr][npk]
__global__ void k_post_sub(size_t n, const double2* __restrict__ a, const double2* __restrict__ b, double2* __restrict__ out) {
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const double2 x = a[e], y = b[e];
        out[e] = make_double2(x.x - y.x, x.y - y.y);
    }
}

}  // namespace chn
