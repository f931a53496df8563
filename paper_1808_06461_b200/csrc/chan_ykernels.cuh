// Wall-normal (y) phase: one thread per Fourier mode marching along y in PLANE layout [ny][nz][nxh]
// (consecutive threads = consecutive k_x, so every load and store is a coalesced 16-byte-per-lane
// access).  Steps a1, a9-a11 of DESIGN.md; PAPER.md L78-80 (formulation, compact differences, RK3),
// L84 ("operations in the y direction (mostly banded-matrix solvers)"), L100 (influence matrix).
//
// Banded systems are solved by unpivoted elimination in ascending row order of an ORIENTATION:
// orientation 0 is the natural order j = 0..ny-1, orientation 1 the flipped order i = ny-1-j (the
// same system with rows and columns reversed).  A sweep that walks physical rows downwards can
// therefore back-substitute an orientation-0 system and forward-eliminate an orientation-1 system in
// the same pass, and vice versa, which is what chains the sweeps Y1..Y4 without extra passes.
#pragma once
#include <cuda_runtime.h>

namespace chn {

#define CHAN_HD __host__ __device__ __forceinline__
struct c2 { double x, y; };
CHAN_HD c2 mk(double a, double b) { c2 r; r.x = a; r.y = b; return r; }
CHAN_HD c2 operator+(c2 a, c2 b) { return mk(a.x + b.x, a.y + b.y); }
CHAN_HD c2 operator-(c2 a, c2 b) { return mk(a.x - b.x, a.y - b.y); }
CHAN_HD c2 operator*(double s, c2 a) { return mk(s * a.x, s * a.y); }
CHAN_HD c2 cmul(c2 a, c2 b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
CHAN_HD c2 muli(c2 a) { return mk(-a.y, a.x); }  // i * a
CHAN_HD c2 ldc(const double2* p) { double2 v = *p; return mk(v.x, v.y); }
CHAN_HD void stc(double2* p, c2 v) { *p = make_double2(v.x, v.y); }

// L2 prefetch of a row that a marching sweep will read CHAN_PF iterations later: the sweeps are bound by
// the latency of one dependent global round trip per row, not by bandwidth, at the occupancy their
// register windows allow.
#ifndef CHAN_PF
#define CHAN_PF 6
#endif
__device__ __forceinline__ void pf2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

struct YTab {               // device pointers to the row tables of one orientation
    const double* B1;       // [ny][8]
    const double* A2;       // [ny][8]
    const double* B2;       // [ny][8]
    const double* lu1;      // [ny][8]
};

struct YParams {
    int ny, nz, nxh, nzh;
    long long nm;           // modes per plane = nz*nxh
    YTab t[2];
    const double* kx;       // [nxh]
    const double* kz;       // [nz]
    const double* wm;       // [ny]
    const double* wp;       // [ny]
    double nu, dt;          // dt = full step
    double alpha, beta, gamma, zeta;  // of the current substep
};

__device__ __forceinline__ void load8(const double* tab, int row, double (&r)[8]) {
    const double2* p = reinterpret_cast<const double2*>(tab + (size_t)row * 8);
    double2 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2), d = __ldg(p + 3);
    r[0] = a.x; r[1] = a.y; r[2] = b.x; r[3] = b.y; r[4] = c.x; r[5] = c.y; r[6] = d.x; r[7] = d.y;
}

// Sliding 7-wide window; w[6] is the newest entry.
template <typename T> __device__ __forceinline__ void push(T (&w)[7], T v) {
#pragma unroll
    for (int k = 0; k < 6; ++k) w[k] = w[k + 1];
    w[6] = v;
}
__device__ __forceinline__ c2 band7(const double (&c)[8], const c2 (&w)[7]) {
    c2 s = c[0] * w[0];
#pragma unroll
    for (int k = 1; k < 7; ++k) { s.x += c[k] * w[k].x; s.y += c[k] * w[k].y; }
    return s;
}
__device__ __forceinline__ double band7(const double (&c)[8], const double (&w)[7]) {
    double s = c[0] * w[0];
#pragma unroll
    for (int k = 1; k < 7; ++k) s += c[k] * w[k];
    return s;
}

// ---- constant-LU first derivative ------------------------------------------------------------------
struct D1Fwd {   // forward elimination state: z_{i-1}, z_{i-2}, z_{i-3}
    c2 z1, z2, z3;
    __device__ __forceinline__ void init() { z1 = z2 = z3 = mk(0, 0); }
    __device__ __forceinline__ c2 step(const double (&lu)[8], c2 r) {
        c2 z = mk(r.x - lu[0] * z1.x - lu[1] * z2.x - lu[2] * z3.x, r.y - lu[0] * z1.y - lu[1] * z2.y - lu[2] * z3.y);
        z3 = z2; z2 = z1; z1 = z;
        return z;
    }
};
struct D1Bwd {   // back substitution state: g_{i+1}, g_{i+2}, g_{i+3}
    c2 g1, g2, g3;
    __device__ __forceinline__ void init() { g1 = g2 = g3 = mk(0, 0); }
    __device__ __forceinline__ c2 step(const double (&lu)[8], c2 z) {
        c2 g = mk((z.x - lu[4] * g1.x - lu[5] * g2.x - lu[6] * g3.x) * lu[3],
                  (z.y - lu[4] * g1.y - lu[5] * g2.y - lu[6] * g3.y) * lu[3]);
        g3 = g2; g2 = g1; g1 = g;
        return g;
    }
};

// ---- per-mode heptadiagonal factorisation ------------------------------------------------------------
// Row i of M (entries a[0..6] at columns i-3..i+3) is reduced against the three previous pivot rows.
// Stored factor row: {1/d_i, U_{i,i+1}, U_{i,i+2}, U_{i,i+3}}.
struct HeptaFac {
    double d1i, u11, u12, u13;   // row i-1
    double d2i, u21, u22, u23;   // row i-2
    double d3i, u31, u32, u33;   // row i-3
    double l1, l2, l3;           // multipliers of the row being reduced
    __device__ __forceinline__ void init() {
        d1i = d2i = d3i = 1.0; u11 = u12 = u13 = u21 = u22 = u23 = u31 = u32 = u33 = 0.0; l1 = l2 = l3 = 0.0;
    }
    // reduce row; returns {1/d, u1, u2, u3} and keeps l1..l3 for the right-hand sides
    __device__ __forceinline__ double4 reduce(double (&a)[7]) {
        l3 = a[0] * d3i;
        a[1] -= l3 * u31; a[2] -= l3 * u32; a[3] -= l3 * u33;
        l2 = a[1] * d2i;
        a[2] -= l2 * u21; a[3] -= l2 * u22; a[4] -= l2 * u23;
        l1 = a[2] * d1i;
        a[3] -= l1 * u11; a[4] -= l1 * u12; a[5] -= l1 * u13;
        const double di = 1.0 / a[3];
        d3i = d2i; u31 = u21; u32 = u22; u33 = u23;
        d2i = d1i; u21 = u11; u22 = u12; u23 = u13;
        d1i = di; u11 = a[4]; u12 = a[5]; u13 = a[6];
        return make_double4(di, a[4], a[5], a[6]);
    }
};
template <typename T> struct RhsFwd {   // forward substitution of one right-hand side with HeptaFac multipliers
    T z1, z2, z3;
    __device__ __forceinline__ T step(const HeptaFac& f, T r);
};
template <> __device__ __forceinline__ c2 RhsFwd<c2>::step(const HeptaFac& f, c2 r) {
    c2 z = mk(r.x - f.l3 * z3.x - f.l2 * z2.x - f.l1 * z1.x, r.y - f.l3 * z3.y - f.l2 * z2.y - f.l1 * z1.y);
    z3 = z2; z2 = z1; z1 = z;
    return z;
}
template <> __device__ __forceinline__ double RhsFwd<double>::step(const HeptaFac& f, double r) {
    double z = r - f.l3 * z3 - f.l2 * z2 - f.l1 * z1;
    z3 = z2; z2 = z1; z1 = z;
    return z;
}
// A factor row {1/d, u1, u2, u3} is stored as two double2 halves in two separate arrays (facA = {1/d, u1},
// facB = {u2, u3}) so that each half can live in a different dead field buffer.
__device__ __forceinline__ void st_fac(double2* fa, double2* fb, size_t o, double4 f) {
    fa[o] = make_double2(f.x, f.y); fb[o] = make_double2(f.z, f.w);
}
__device__ __forceinline__ double4 ld_fac(const double2* fa, const double2* fb, size_t o) {
    const double2 a = fa[o], b = fb[o];
    return make_double4(a.x, a.y, b.x, b.y);
}
template <typename T> struct RhsBwd {   // back substitution with a stored factor row
    T x1, x2, x3;
    __device__ __forceinline__ T step(double4 f, T z);
};
template <> __device__ __forceinline__ c2 RhsBwd<c2>::step(double4 f, c2 z) {
    c2 x = mk((z.x - f.y * x1.x - f.z * x2.x - f.w * x3.x) * f.x, (z.y - f.y * x1.y - f.z * x2.y - f.w * x3.y) * f.x);
    x3 = x2; x2 = x1; x1 = x;
    return x;
}
template <> __device__ __forceinline__ double RhsBwd<double>::step(double4 f, double z) {
    double x = (z - f.y * x1 - f.z * x2 - f.w * x3) * f.x;
    x3 = x2; x2 = x1; x1 = x;
    return x;
}

__device__ __forceinline__ bool mode_setup(const YParams& P, long long& m, int& s, int& p, double& kx, double& kz) {
    m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= P.nm) return false;
    s = (int)(m / P.nxh);
    p = (int)(m - (long long)s * P.nxh);
    kx = __ldg(P.kx + p);
    kz = __ldg(P.kz + s);
    return true;
}

// =====================================================================================================
// K1a: z = forward elimination (orientation 0) of B1 f.        reads f, writes z
// =====================================================================================================
__global__ void __launch_bounds__(128) k_d1_forward(YParams P, const double2* __restrict__ f, double2* __restrict__ z) {
    long long m; int s, p; double kx, kz;
    if (!mode_setup(P, m, s, p, kx, kz)) return;
    if (s == P.nzh) return;
    const int ny = P.ny;
    c2 w[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) w[k] = mk(0, 0);
    D1Fwd fw; fw.init();
    double b1[8], lu[8];
    for (int jj = 0; jj < ny + 3; ++jj) {
        if (jj + CHAN_PF < ny) pf2(f + (size_t)(jj + CHAN_PF) * P.nm + m);
        push(w, jj < ny ? ldc(f + (size_t)jj * P.nm + m) : mk(0, 0));
        const int j = jj - 3;
        if (j >= 0) {
            load8(P.t[0].B1, j, b1); load8(P.t[0].lu1, j, lu);
            stc(z + (size_t)j * P.nm + m, fw.step(lu, band7(b1, w)));
        }
    }
}

// =====================================================================================================
// K1b (physical rows descending): dv = backsub(zv); u,w from (dv, om_y) [mode 0: U,W]; store u,w;
// forward-eliminate (orientation 1) B1 u and B1 w -> zu, zw.
// =====================================================================================================
__global__ void __launch_bounds__(128) k_derive_down(YParams P, const double2* zv, const double2* __restrict__ omy,
                                                     const double* __restrict__ U, const double* __restrict__ W,
                                                     double2* __restrict__ u, double2* __restrict__ w_,
                                                     double2* zu /* may alias zv */, double2* __restrict__ zw) {
    long long m; int s, p; double kx, kz;
    if (!mode_setup(P, m, s, p, kx, kz)) return;
    const int ny = P.ny;
    if (s == P.nzh) {   // z-Nyquist slot: always zero (the buffers double as y-phase scratch)
        for (int j = 0; j < ny; ++j) { stc(u + (size_t)j * P.nm + m, mk(0, 0)); stc(w_ + (size_t)j * P.nm + m, mk(0, 0)); }
        return;
    }
    const bool mean = (m == 0);
    const double k2 = kx * kx + kz * kz;
    const double ik2 = mean ? 0.0 : 1.0 / k2;
    D1Bwd bs; bs.init();
    D1Fwd fu, fw; fu.init(); fw.init();
    c2 wu[7], ww[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wu[k] = ww[k] = mk(0, 0);
    double lu[8], b1[8], luf[8];
    for (int ii = 0; ii < ny + 3; ++ii) {       // ii: virtual (flipped) index of the row being produced
        const int j = ny - 1 - ii;             // physical row
        c2 uj = mk(0, 0), wj = mk(0, 0);
        if (j - CHAN_PF >= 0) { pf2(zv + (size_t)(j - CHAN_PF) * P.nm + m); pf2(omy + (size_t)(j - CHAN_PF) * P.nm + m); }
        if (ii < ny) {
            load8(P.t[0].lu1, j, lu);
            c2 dv = bs.step(lu, ldc(zv + (size_t)j * P.nm + m));
            if (mean) { uj = mk(__ldg(U + j), 0.0); wj = mk(__ldg(W + j), 0.0); }
            else {
                c2 oy = ldc(omy + (size_t)j * P.nm + m);
                // u = i (kx dv - kz om_y)/k2 ; w = i (kz dv + kx om_y)/k2
                c2 a = mk(kx * dv.x - kz * oy.x, kx * dv.y - kz * oy.y);
                c2 b = mk(kz * dv.x + kx * oy.x, kz * dv.y + kx * oy.y);
                uj = mk(-a.y / k2, a.x / k2);
                wj = mk(-b.y / k2, b.x / k2);
                (void)ik2;
            }
            stc(u + (size_t)j * P.nm + m, uj);
            stc(w_ + (size_t)j * P.nm + m, wj);
        }
        push(wu, uj); push(ww, wj);
        const int i = ii - 3;                  // virtual row whose window is complete
        if (i >= 0) {
            load8(P.t[1].B1, i, b1); load8(P.t[1].lu1, i, luf);
            const size_t o = (size_t)(ny - 1 - i) * P.nm + m;
            stc(zu + o, fu.step(luf, band7(b1, wu)));
            stc(zw + o, fw.step(luf, band7(b1, ww)));
        }
    }
}

// =====================================================================================================
// K1c (physical rows ascending): du, dw = backsub (orientation 1) of zu, zw;
// om_x = dw - i kz v, om_z = i kx v - du.
// =====================================================================================================
__global__ void __launch_bounds__(128) k_derive_up(YParams P, const double2* __restrict__ zu, const double2* zw /* may alias oz */,
                                                   const double2* __restrict__ v, double2* __restrict__ ox, double2* oz) {
    long long m; int s, p; double kx, kz;
    if (!mode_setup(P, m, s, p, kx, kz)) return;
    const int ny = P.ny;
    if (s == P.nzh) {
        for (int j = 0; j < ny; ++j) { stc(ox + (size_t)j * P.nm + m, mk(0, 0)); stc(oz + (size_t)j * P.nm + m, mk(0, 0)); }
        return;
    }
    D1Bwd bu, bw; bu.init(); bw.init();
    double luf[8];
    for (int j = 0; j < ny; ++j) {
        const int i = ny - 1 - j;
        load8(P.t[1].lu1, i, luf);
        const size_t o = (size_t)j * P.nm + m;
        c2 du = bu.step(luf, ldc(zu + o));
        c2 dw = bw.step(luf, ldc(zw + o));
        c2 vj = (m == 0) ? mk(0, 0) : ldc(v + o);
        // -i kz v = (kz v.y, -kz v.x);  i kx v = (-kx v.y, kx v.x)
        stc(ox + o, mk(dw.x + kz * vj.y, dw.y - kz * vj.x));
        stc(oz + o, mk(-kx * vj.y - du.x, kx * vj.x - du.y));
    }
}

// Helmholtz / Poisson matrix row in orientation o: interior rows B2 - lam*A2, wall rows identity.
__device__ __forceinline__ void helm_row(const YParams& P, int o, int i, double lam, const double (&a2)[8], const double (&b2)[8],
                                         double (&a)[7]) {
    if (i == 0 || i == P.ny - 1) {
#pragma unroll
        for (int k = 0; k < 7; ++k) a[k] = 0.0;
        a[3] = 1.0;
    } else {
#pragma unroll
        for (int k = 0; k < 7; ++k) a[k] = b2[k] - lam * a2[k];
    }
}

// Right-hand side row of step 6: -c [ A2 t + alpha nu dt (B2 x - k2 A2 x) ], zero at the wall rows.
__device__ __forceinline__ c2 helm_rhs(const YParams& P, int i, double c, double k2, const double (&a2)[8], const double (&b2)[8],
                                       const c2 (&t)[7], const c2 (&x)[7]) {
    if (i == 0 || i == P.ny - 1) return mk(0, 0);
    c2 at = band7(a2, t), bx = band7(b2, x), ax = band7(a2, x);
    const double g = P.alpha * P.nu * P.dt;
    return mk(-c * (at.x + g * (bx.x - k2 * ax.x)), -c * (at.y + g * (bx.y - k2 * ax.y)));
}

// =====================================================================================================
// Y1 (ascending): h_g = i kz H1 - i kx H3 (stored over hg_prev), d = i kx H1 + i kz H3,
//   zd  = D1-forward(orientation 0) of d,
//   om_y Helmholtz (B2 - lam A2) x = R_om, forward elimination in orientation 0 -> fac, z_om.
// =====================================================================================================
__global__ void __launch_bounds__(128) k_y1(YParams P, const double2* H1, const double2* __restrict__ H3,
                                            const double2* __restrict__ omy, double2* __restrict__ hg,
                                            double2* __restrict__ zd, double2* __restrict__ facA, double2* __restrict__ facB, double2* zom) {
    long long m; int s, p; double kx, kz;
    if (!mode_setup(P, m, s, p, kx, kz)) return;
    if (s == P.nzh || m == 0) return;
    const int ny = P.ny;
    const double k2 = kx * kx + kz * kz;
    const double c = 1.0 / (P.beta * P.nu * P.dt), lam = k2 + c;
    c2 wd[7], wt[7], wx[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wd[k] = wt[k] = wx[k] = mk(0, 0);
    D1Fwd fd; fd.init();
    HeptaFac hf; hf.init();
    RhsFwd<c2> rz; rz.z1 = rz.z2 = rz.z3 = mk(0, 0);
    double b1[8], lu[8], a2[8], b2[8], a[7];
    for (int jj = 0; jj < ny + 3; ++jj) {
        if (jj + CHAN_PF < ny) { const size_t op = (size_t)(jj + CHAN_PF) * P.nm + m; pf2(H1 + op); pf2(H3 + op); pf2(omy + op); pf2(hg + op); }
        if (jj < ny) {
            const size_t o = (size_t)jj * P.nm + m;
            c2 h1 = ldc(H1 + o), h3 = ldc(H3 + o), x = ldc(omy + o), gp = ldc(hg + o);
            // i kz h1 - i kx h3 ; i kx h1 + i kz h3
            c2 g = mk(-kz * h1.y + kx * h3.y, kz * h1.x - kx * h3.x);
            c2 d = mk(-kx * h1.y - kz * h3.y, kx * h1.x + kz * h3.x);
            stc(hg + o, g);
            push(wd, d);
            push(wx, x);
            push(wt, mk(x.x + P.dt * (P.gamma * g.x + P.zeta * gp.x), x.y + P.dt * (P.gamma * g.y + P.zeta * gp.y)));
        } else { push(wd, mk(0, 0)); push(wx, mk(0, 0)); push(wt, mk(0, 0)); }
        const int j = jj - 3;
        if (j >= 0) {
            const size_t o = (size_t)j * P.nm + m;
            load8(P.t[0].B1, j, b1); load8(P.t[0].lu1, j, lu);
            stc(zd + o, fd.step(lu, band7(b1, wd)));
            load8(P.t[0].A2, j, a2); load8(P.t[0].B2, j, b2);
            helm_row(P, 0, j, lam, a2, b2, a);
            c2 r = helm_rhs(P, j, c, k2, a2, b2, wt, wx);
            st_fac(facA, facB, o, hf.reduce(a));
            stc(zom + o, rz.step(hf, r));
        }
    }
}

// =====================================================================================================
// Y2 (descending): om_y^new = backsub(fac, z_om);  dd = D1-backsub(zd);  h_v = -k2 H2 - dd (over hv_prev);
//   phi Helmholtz in orientation 1: forward elimination -> fac (overwritten), z_phi, z_b
//   (z of the homogeneous problem with phi(+1)=1; the one with phi(-1)=1 has z = unit vector, not stored).
// =====================================================================================================
__global__ void __launch_bounds__(128) k_y2(YParams P, const double2* __restrict__ H2, const double2* zd,
                                            const double2* __restrict__ zom, double2* facA, double2* facB,
                                            const double2* __restrict__ phi, double2* __restrict__ hv, double2* __restrict__ omy,
                                            double2* zphi, double* __restrict__ zb) {
    long long m; int s, p; double kx, kz;
    if (!mode_setup(P, m, s, p, kx, kz)) return;
    if (s == P.nzh || m == 0) return;
    const int ny = P.ny;
    const double k2 = kx * kx + kz * kz;
    const double c = 1.0 / (P.beta * P.nu * P.dt), lam = k2 + c;
    c2 wt[7], wx[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wt[k] = wx[k] = mk(0, 0);
    D1Bwd bd; bd.init();
    RhsBwd<c2> bo; bo.x1 = bo.x2 = bo.x3 = mk(0, 0);
    HeptaFac hf; hf.init();
    RhsFwd<c2> rz; rz.z1 = rz.z2 = rz.z3 = mk(0, 0);
    RhsFwd<double> rb; rb.z1 = rb.z2 = rb.z3 = 0.0;
    double lu[8], a2[8], b2[8], a[7];
    for (int ii = 0; ii < ny + 3; ++ii) {
        const int j = ny - 1 - ii;
        if (j - CHAN_PF >= 0) {
            const size_t op = (size_t)(j - CHAN_PF) * P.nm + m;
            pf2(facA + op); pf2(facB + op); pf2(zom + op); pf2(zd + op); pf2(H2 + op); pf2(phi + op); pf2(hv + op);
        }
        if (ii < ny) {
            const size_t o = (size_t)j * P.nm + m;
            stc(omy + o, bo.step(ld_fac(facA, facB, o), ldc(zom + o)));
            load8(P.t[0].lu1, j, lu);
            c2 dd = bd.step(lu, ldc(zd + o));
            c2 h2 = ldc(H2 + o), x = ldc(phi + o), hp = ldc(hv + o);
            c2 h = mk(-k2 * h2.x - dd.x, -k2 * h2.y - dd.y);
            stc(hv + o, h);
            push(wx, x);
            push(wt, mk(x.x + P.dt * (P.gamma * h.x + P.zeta * hp.x), x.y + P.dt * (P.gamma * h.y + P.zeta * hp.y)));
        } else { push(wx, mk(0, 0)); push(wt, mk(0, 0)); }
        const int i = ii - 3;
        if (i >= 0) {
            const size_t o = (size_t)(ny - 1 - i) * P.nm + m;
            load8(P.t[1].A2, i, a2); load8(P.t[1].B2, i, b2);
            helm_row(P, 1, i, lam, a2, b2, a);
            c2 r = helm_rhs(P, i, c, k2, a2, b2, wt, wx);
            st_fac(facA, facB, o, hf.reduce(a));
            stc(zphi + o, rz.step(hf, r));
            zb[o] = rb.step(hf, i == 0 ? 1.0 : 0.0);   // virtual row 0 = physical wall y=+1
        }
    }
}

// =====================================================================================================
// Y3 (ascending): phi_p, phi_a, phi_b = backsub (orientation 1);  Poisson (B2 - k2 A2) v_s = A2 phi_s,
//   forward elimination in orientation 0 -> fac (overwritten), z_vp, z_va, z_vb.
// =====================================================================================================
__global__ void __launch_bounds__(128) k_y3(YParams P, double2* facA, double2* facB, double2* __restrict__ zphi /* -> phi_p */,
                                            double* __restrict__ zb /* -> phi_b */, double* __restrict__ phia,
                                            double2* __restrict__ zvp, double* __restrict__ zva, double* __restrict__ zvb) {
    long long m; int s, p; double kx, kz;
    if (!mode_setup(P, m, s, p, kx, kz)) return;
    if (s == P.nzh || m == 0) return;
    const int ny = P.ny;
    const double k2 = kx * kx + kz * kz;
    c2 wp_[7]; double wa[7], wb[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) { wp_[k] = mk(0, 0); wa[k] = wb[k] = 0.0; }
    RhsBwd<c2> bp; bp.x1 = bp.x2 = bp.x3 = mk(0, 0);
    RhsBwd<double> ba, bb; ba.x1 = ba.x2 = ba.x3 = 0.0; bb.x1 = bb.x2 = bb.x3 = 0.0;
    HeptaFac hf; hf.init();
    RhsFwd<c2> rp; rp.z1 = rp.z2 = rp.z3 = mk(0, 0);
    RhsFwd<double> ra, rb; ra.z1 = ra.z2 = ra.z3 = 0.0; rb.z1 = rb.z2 = rb.z3 = 0.0;
    double a2[8], b2[8], a[7];
    for (int jj = 0; jj < ny + 3; ++jj) {
        if (jj + CHAN_PF < ny) { const size_t op = (size_t)(jj + CHAN_PF) * P.nm + m; pf2(facA + op); pf2(facB + op); pf2(zphi + op); pf2(zb + op); }
        if (jj < ny) {
            const size_t o = (size_t)jj * P.nm + m;
            const double4 f = ld_fac(facA, facB, o);
            c2 pp = bp.step(f, ldc(zphi + o));
            double pb = bb.step(f, zb[o]);
            double pa = ba.step(f, jj == 0 ? 1.0 : 0.0);   // z of the phi(-1)=1 problem: unit vector at the last virtual row
            stc(zphi + o, pp); zb[o] = pb; phia[o] = pa;
            push(wp_, pp); push(wa, pa); push(wb, pb);
        } else { push(wp_, mk(0, 0)); push(wa, 0.0); push(wb, 0.0); }
        const int j = jj - 3;
        if (j >= 0) {
            const size_t o = (size_t)j * P.nm + m;
            load8(P.t[0].A2, j, a2); load8(P.t[0].B2, j, b2);
            helm_row(P, 0, j, k2, a2, b2, a);
            const bool wall = (j == 0 || j == ny - 1);
            c2 r = wall ? mk(0, 0) : band7(a2, wp_);
            double rra = wall ? 0.0 : band7(a2, wa), rrb = wall ? 0.0 : band7(a2, wb);
            st_fac(facA, facB, o, hf.reduce(a));
            stc(zvp + o, rp.step(hf, r));
            zva[o] = ra.step(hf, rra);
            zvb[o] = rb.step(hf, rrb);
        }
    }
}

// =====================================================================================================
// Y4 (descending): v_p, v_a, v_b = backsub (orientation 0); wall derivatives as weighted sums;
//   influence matrix (step 7) -> coef[m] = (c_a, c_b).
// =====================================================================================================
__global__ void __launch_bounds__(128) k_y4(YParams P, const double2* __restrict__ facA, const double2* __restrict__ facB, double2* __restrict__ zvp,
                                            double* __restrict__ zva, double* __restrict__ zvb, double4* __restrict__ coef) {
    long long m; int s, p; double kx, kz;
    if (!mode_setup(P, m, s, p, kx, kz)) return;
    if (s == P.nzh || m == 0) return;
    const int ny = P.ny;
    RhsBwd<c2> bp; bp.x1 = bp.x2 = bp.x3 = mk(0, 0);
    RhsBwd<double> ba, bb; ba.x1 = ba.x2 = ba.x3 = 0.0; bb.x1 = bb.x2 = bb.x3 = 0.0;
    c2 dpm = mk(0, 0), dpp = mk(0, 0);
    double dam = 0, dap = 0, dbm = 0, dbp = 0;
    for (int j = ny - 1; j >= 0; --j) {
        const size_t o = (size_t)j * P.nm + m;
        const double4 f = ld_fac(facA, facB, o);
        c2 vp = bp.step(f, ldc(zvp + o));
        double va = ba.step(f, zva[o]), vb = bb.step(f, zvb[o]);
        stc(zvp + o, vp); zva[o] = va; zvb[o] = vb;
        const double wm = __ldg(P.wm + j), wp = __ldg(P.wp + j);
        dpm.x += wm * vp.x; dpm.y += wm * vp.y; dpp.x += wp * vp.x; dpp.y += wp * vp.y;
        dam += wm * va; dap += wp * va; dbm += wm * vb; dbp += wp * vb;
    }
    // G = [[dam, dbm],[dap, dbp]];  (ca, cb) = -G^{-1} (dpm, dpp)
    const double det = dam * dbp - dbm * dap;
    c2 ca = mk((dbp * (-dpm.x) - dbm * (-dpp.x)) / det, (dbp * (-dpm.y) - dbm * (-dpp.y)) / det);
    c2 cb = mk((-dap * (-dpm.x) + dam * (-dpp.x)) / det, (-dap * (-dpm.y) + dam * (-dpp.y)) / det);
    coef[m] = make_double4(ca.x, ca.y, cb.x, cb.y);
}

// =====================================================================================================
// Y5: phi = phi_p + ca phi_a + cb phi_b, v likewise.
// =====================================================================================================
__global__ void __launch_bounds__(128) k_y5(YParams P, const double4* __restrict__ coef, const double2* __restrict__ phip,
                                            const double* __restrict__ phia, const double* __restrict__ phib,
                                            const double2* __restrict__ vp, const double* __restrict__ va, const double* __restrict__ vb,
                                            double2* __restrict__ phi, double2* __restrict__ v) {
    long long m; int s, p; double kx, kz;
    if (!mode_setup(P, m, s, p, kx, kz)) return;
    if (s == P.nzh || m == 0) return;
    const double4 cc = coef[m];
    for (int j = blockIdx.y; j < P.ny; j += gridDim.y) {
        const size_t o = (size_t)j * P.nm + m;
        c2 pp = ldc(phip + o), vv = ldc(vp + o);
        const double pa = phia[o], pb = phib[o], a = va[o], b = vb[o];
        stc(phi + o, mk(pp.x + cc.x * pa + cc.z * pb, pp.y + cc.y * pa + cc.w * pb));
        stc(v + o, mk(vv.x + cc.x * a + cc.z * b, vv.y + cc.y * a + cc.w * b));
    }
}

// =====================================================================================================
// Mean mode (step 8), one thread: U, W Helmholtz with c; constant mass flux.  Arrays in global scratch.
// scal: [0] -dP/dx, [1] Q0, [2] nu dU/dy(-1), [3] -nu dU/dy(+1)
// =====================================================================================================
struct MeanParams {
    int ny; long long nm;
    const double *A2, *B2;     // orientation 0 [ny][8]
    const double *wq, *wm, *wp;
    double nu, dt, alpha, beta, gamma, zeta;
    int forcing;
};
// One CTA; dynamic shared memory 15*ny doubles: the matrix rows and right-hand sides are built by all threads,
// the (serial) factorisation and substitutions run in thread 0 out of shared memory.
__global__ void __launch_bounds__(256) k_mean(MeanParams M, const double2* __restrict__ H1, const double2* __restrict__ H3,
                                              double* __restrict__ U, double* __restrict__ W, double* __restrict__ H1p,
                                              double* __restrict__ H3p, double* __restrict__ scal) {
    extern __shared__ double sh[];
    const int ny = M.ny;
    double* Mt = sh;                  // [ny][8] rows of B2 - c A2 (Dirichlet rows at the walls)
    double* zu = sh + (size_t)8 * ny; double* zh = zu + ny; double* zw = zh + ny;
    double* f1 = zw + ny; double* f2 = f1 + ny; double* f3 = f2 + ny; double* fd = f3 + ny;
    const double c = 1.0 / (M.beta * M.nu * M.dt);
    const double g = M.alpha * M.nu * M.dt;
    // explicit parts t = X + dt (gamma H + zeta Hprev), kept in f1 (U) and f2 (W); old U, W in f3, fd
    for (int j = threadIdx.x; j < ny; j += blockDim.x) {
        const double h1 = H1[(size_t)j * M.nm].x, h3 = H3[(size_t)j * M.nm].x;
        f1[j] = U[j] + M.dt * (M.gamma * h1 + M.zeta * H1p[j]);
        f2[j] = W[j] + M.dt * (M.gamma * h3 + M.zeta * H3p[j]);
        f3[j] = U[j]; fd[j] = W[j];
        H1p[j] = h1; H3p[j] = h3;
    }
    __syncthreads();
    // r_u = -c (A2 t_u + g B2 U), r_h = -c (A2 1), r_w = -c (A2 t_w + g B2 W); matrix rows
    for (int j = threadIdx.x; j < ny; j += blockDim.x) {
        double su = 0, sh_ = 0, sw = 0;
        const bool wall = (j == 0 || j == ny - 1);
        for (int k = 0; k < 7; ++k) {
            const double a2 = M.A2[(size_t)j * 8 + k], b2 = M.B2[(size_t)j * 8 + k];
            Mt[(size_t)j * 8 + k] = wall ? (k == 3 ? 1.0 : 0.0) : b2 - c * a2;
            const int jj = j + k - 3;
            if (wall || jj < 0 || jj >= ny) continue;
            su += a2 * f1[jj] + g * b2 * f3[jj];
            sw += a2 * f2[jj] + g * b2 * fd[jj];
            sh_ += a2;
        }
        zu[j] = -c * su; zh[j] = -c * sh_; zw[j] = -c * sw;
        if (wall) { zu[j] = 0.0; zh[j] = 0.0; zw[j] = 0.0; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double d1 = 1, u11 = 0, u12 = 0, u13 = 0, d2 = 1, u21 = 0, u22 = 0, u23 = 0, d3 = 1, u31 = 0, u32 = 0, u33 = 0;
        double* zs[3] = {zu, zh, zw};
        for (int j = 0; j < ny; ++j) {
            double a[7];
            for (int k = 0; k < 7; ++k) a[k] = Mt[(size_t)j * 8 + k];
            const double l3 = a[0] * d3; a[1] -= l3 * u31; a[2] -= l3 * u32; a[3] -= l3 * u33;
            const double l2 = a[1] * d2; a[2] -= l2 * u21; a[3] -= l2 * u22; a[4] -= l2 * u23;
            const double l1 = a[2] * d1; a[3] -= l1 * u11; a[4] -= l1 * u12; a[5] -= l1 * u13;
            const double di = 1.0 / a[3];
            d3 = d2; u31 = u21; u32 = u22; u33 = u23; d2 = d1; u21 = u11; u22 = u12; u23 = u13;
            d1 = di; u11 = a[4]; u12 = a[5]; u13 = a[6];
            for (int q = 0; q < 3; ++q) {
                double z = zs[q][j];
                if (j >= 3) z -= l3 * zs[q][j - 3];
                if (j >= 2) z -= l2 * zs[q][j - 2];
                if (j >= 1) z -= l1 * zs[q][j - 1];
                zs[q][j] = z;
            }
            fd[j] = di; f1[j] = a[4]; f2[j] = a[5]; f3[j] = a[6];
        }
        for (int j = ny - 1; j >= 0; --j) {
            for (int q = 0; q < 3; ++q) {
                double x = zs[q][j];
                if (j + 1 < ny) x -= f1[j] * zs[q][j + 1];
                if (j + 2 < ny) x -= f2[j] * zs[q][j + 2];
                if (j + 3 < ny) x -= f3[j] * zs[q][j + 3];
                zs[q][j] = x * fd[j];
            }
        }
        double qp = 0, qh = 0;
        for (int j = 0; j < ny; ++j) { qp += M.wq[j] * zu[j]; qh += M.wq[j] * zh[j]; }
        double Pi;
        if (M.forcing == 0) { Pi = (scal[1] - qp) / qh; scal[0] = Pi / ((M.gamma + M.zeta) * M.dt); }
        else Pi = scal[0] * (M.gamma + M.zeta) * M.dt;
        double sm = 0, sp = 0;
        for (int j = 0; j < ny; ++j) {
            const double un = zu[j] + Pi * zh[j];
            U[j] = un; W[j] = zw[j];
            sm += M.wm[j] * un; sp += M.wp[j] * un;
        }
        scal[2] = M.nu * sm; scal[3] = -M.nu * sp;
    }
}

__global__ void k_flux(int ny, const double* __restrict__ wq, const double* __restrict__ U, double* __restrict__ scal) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    double q = 0;
    for (int j = 0; j < ny; ++j) q += wq[j] * U[j];
    scal[1] = q;
}

}  // namespace chn
