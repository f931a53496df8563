// Wall-normal (y) phase, second generation: six marching sweeps in PLANE layout [ny][nz][nxh] with TWO
// threads per Fourier mode.  Steps a1, a9-a11 of DESIGN.md; PAPER.md L78-80 (formulation, compact
// differences, RK3), L84 ("operations in the y direction (mostly banded-matrix solvers)"), L100
// (influence matrix).
//
// Every banded matrix of the y-phase is REAL and acts on complex data, so the real and the imaginary part
// of a mode are independent problems with the same factorisation: thread 2m carries Re, thread 2m+1 carries
// Im (each repeats the cheap real factorisation; of the two real homogeneous problems "a" and "b" the even
// thread carries a, the odd one b).  That halves the register windows per thread and doubles the number of
// threads in flight, which is what these latency-bound sweeps need.  Consecutive lanes touch consecutive
// doubles, so all traffic stays coalesced.
//
// Orientations as in chan_ykernels.cuh: orientation 0 is the natural row order, orientation 1 the flipped
// one; a sweep walking physical rows downwards back-substitutes an orientation-0 system and
// forward-eliminates an orientation-1 system in the same pass, and vice versa.
//
//   SA (up)  : h_g, d = i kx H1 + i kz H3, forward D1(d) [o0], Helmholtz right-hand side R_om
//   SB (down): back D1(d) -> h_v; ONE Helmholtz factorisation [o1] shared by om_y, phi_p and phi_b: forward
//   SC (up)  : back -> om_y^new, phi_p, phi_a, phi_b; Poisson factorisation [o0], forward v_p, v_a, v_b; the
//              wall derivatives D1 v_s(+-1) = w . U^-1 z_s = (U^-T w) . z_s are accumulated in the SAME
//              sweep through the adjoint recurrence U^T g = w, so the influence matrix (step 7) is solved
//              before the back substitution
//   SD (down): v = back(z_p + c_a z_a + c_b z_b), phi = phi_p + c_a phi_a + c_b phi_b, forward D1(v) [o1]
//   SE (up)  : back D1(v) -> u, w; forward D1(u), D1(w) [o0]
//   SF (down): back -> om_x, om_z
// Row tables are staged through shared memory in chunks of YCH iterations.
#pragma once
#include <cuda_runtime.h>

#include "chan_ykernels.cuh"

namespace chn {

constexpr int YCH = 32;     // iterations per shared-memory table chunk
constexpr int YNT = 128;    // threads per CTA = 64 modes

struct YS {                 // per-thread identity
    long long m;            // mode
    int part;               // 0: real part / problem a, 1: imaginary part / problem b
    bool act;               // has work (not the mean mode, not the z-Nyquist slot, inside the plane)
    bool inplane, nyq;
    double kx, kz, k2;
};
__device__ __forceinline__ YS ys_setup(const YParams& P) {
    YS S;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    S.m = t >> 1; S.part = (int)(t & 1);
    S.inplane = S.m < P.nm;
    const long long mm = S.inplane ? S.m : 0;
    const int s = (int)(mm / P.nxh), p = (int)(mm - (long long)s * P.nxh);
    S.nyq = (s == P.nzh);
    S.kx = __ldg(P.kx + p); S.kz = __ldg(P.kz + s);
    S.k2 = S.kx * S.kx + S.kz * S.kz;
    S.act = S.inplane && !S.nyq && S.m != 0;
    return S;
}

// rows r(it) = a + b*it, it = it0 .. it0+YCH-1, of an [ny][8] table -> dst[YCH][8] (zeros outside)
__device__ __forceinline__ void stage8(double* dst, const double* tab, int ny, int it0, int a, int b) {
    for (int e = threadIdx.x; e < YCH * 8; e += blockDim.x) {
        const int r = a + b * (it0 + (e >> 3));
        dst[e] = (r >= 0 && r < ny) ? __ldg(tab + (size_t)r * 8 + (e & 7)) : 0.0;
    }
}
__device__ __forceinline__ void stage1(double* dst, const double* vec, int ny, int it0, int a, int b) {
    for (int e = threadIdx.x; e < YCH; e += blockDim.x) {
        const int r = a + b * (it0 + e);
        dst[e] = (r >= 0 && r < ny) ? __ldg(vec + r) : 0.0;
    }
}
// element 6 of rows of an [ny][8] table
__device__ __forceinline__ void stage_col6(double* dst, const double* tab, int ny, int it0, int a, int b) {
    for (int e = threadIdx.x; e < YCH; e += blockDim.x) {
        const int r = a + b * (it0 + e);
        dst[e] = (r >= 0 && r < ny) ? __ldg(tab + (size_t)r * 8 + 6) : 0.0;
    }
}

__device__ __forceinline__ double band7s(const double* c, const double (&w)[7]) {
    double s = c[0] * w[0];
#pragma unroll
    for (int k = 1; k < 7; ++k) s += c[k] * w[k];
    return s;
}
struct D1FwdR {
    double z1, z2, z3;
    __device__ __forceinline__ void init() { z1 = z2 = z3 = 0.0; }
    __device__ __forceinline__ double step(const double* lu, double r) {
        const double z = r - lu[0] * z1 - lu[1] * z2 - lu[2] * z3;
        z3 = z2; z2 = z1; z1 = z;
        return z;
    }
};
struct D1BwdR {
    double g1, g2, g3;
    __device__ __forceinline__ void init() { g1 = g2 = g3 = 0.0; }
    __device__ __forceinline__ double step(const double* lu, double z) {
        const double g = (z - lu[4] * g1 - lu[5] * g2 - lu[6] * g3) * lu[3];
        g3 = g2; g2 = g1; g1 = g;
        return g;
    }
};
// matrix row of B2 - lam A2 (identity at the walls) from staged table rows
__device__ __forceinline__ void helm_row_s(int ny, int i, double lam, const double* a2, const double* b2, double (&a)[7]) {
    if (i == 0 || i == ny - 1) {
#pragma unroll
        for (int k = 0; k < 7; ++k) a[k] = 0.0;
        a[3] = 1.0;
    } else {
#pragma unroll
        for (int k = 0; k < 7; ++k) a[k] = b2[k] - lam * a2[k];
    }
}
// -c [ A2 t + alpha nu dt (B2 x - k2 A2 x) ], zero at the walls (step 6)
__device__ __forceinline__ double helm_rhs_s(const YParams& P, int i, double c, double k2, const double* a2, const double* b2,
                                             const double (&t)[7], const double (&x)[7]) {
    if (i == 0 || i == P.ny - 1) return 0.0;
    const double at = band7s(a2, t), bx = band7s(b2, x), ax = band7s(a2, x);
    const double g = P.alpha * P.nu * P.dt;
    return -c * (at + g * (bx - k2 * ax));
}

__device__ __forceinline__ const double* cpart(const double2* a, size_t o, int part) { return reinterpret_cast<const double*>(a + o) + part; }
__device__ __forceinline__ double* wpart(double2* a, size_t o, int part) { return reinterpret_cast<double*>(a + o) + part; }

// =====================================================================================================
// SA (ascending).  reads H1, H3, om_y, h_g^prev; writes h_g (in place), zd, R_om.
// =====================================================================================================
__global__ void __launch_bounds__(YNT) k_sa(YParams P, const double2* __restrict__ H1, const double2* __restrict__ H3,
                                            const double2* __restrict__ omy, double2* __restrict__ hg,
                                            double2* __restrict__ zd, double2* __restrict__ rom) {
    __shared__ double sB1[YCH * 8], sLU[YCH * 8], sA2[YCH * 8], sB2[YCH * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    const double c = 1.0 / (P.beta * P.nu * P.dt);
    double wd[7], wt[7], wx[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wd[k] = wt[k] = wx[k] = 0.0;
    D1FwdR fd; fd.init();
    const int nit = ny + 3;
    for (int it0 = 0; it0 < nit; it0 += YCH) {
        __syncthreads();
        stage8(sB1, P.t[0].B1, ny, it0, -3, 1); stage8(sLU, P.t[0].lu1, ny, it0, -3, 1);
        stage8(sA2, P.t[0].A2, ny, it0, -3, 1); stage8(sB2, P.t[0].B2, ny, it0, -3, 1);
        __syncthreads();
        const int ite = min(it0 + YCH, nit);
        for (int jj = it0; jj < ite; ++jj) {
            double d = 0.0, x = 0.0, t = 0.0;
            if (S.act && jj < ny) {
                const size_t o = (size_t)jj * P.nm + S.m;
                if (jj + CHAN_PF < ny) { const size_t op = o + (size_t)CHAN_PF * P.nm; pf2(H1 + op); pf2(H3 + op); pf2(omy + op); pf2(hg + op); }
                const c2 h1 = ldc(H1 + o), h3 = ldc(H3 + o);
                x = *cpart(omy, o, part);
                const double gp = *cpart(hg, o, part);
                // h_g = i kz h1 - i kx h3 ; d = i kx h1 + i kz h3
                const double g = part ? (S.kz * h1.x - S.kx * h3.x) : (-S.kz * h1.y + S.kx * h3.y);
                d = part ? (S.kx * h1.x + S.kz * h3.x) : (-S.kx * h1.y - S.kz * h3.y);
                *wpart(hg, o, part) = g;
                t = x + P.dt * (P.gamma * g + P.zeta * gp);
            }
            push(wd, d); push(wx, x); push(wt, t);
            const int j = jj - 3;
            if (S.act && j >= 0) {
                const size_t o = (size_t)j * P.nm + S.m;
                const int e = (jj - it0) * 8;
                *wpart(zd, o, part) = fd.step(sLU + e, band7s(sB1 + e, wd));
                *wpart(rom, o, part) = helm_rhs_s(P, j, c, S.k2, sA2 + e, sB2 + e, wt, wx);
            }
        }
    }
}

// =====================================================================================================
// SB (descending).  reads zd, H2, phi, h_v^prev, R_om; writes h_v (in place), facA = {1/d, u1},
// facB = {u2, z_b}, z_phi (over zd), z_om (over R_om).  Helmholtz matrix B2 - lam A2 in orientation 1.
// =====================================================================================================
__global__ void __launch_bounds__(YNT) k_sb(YParams P, const double2* __restrict__ H2, const double2* __restrict__ phi,
                                            double2* __restrict__ hv, double2* zd_zphi, double2* rom_zom,
                                            double2* __restrict__ facA, double2* __restrict__ facB) {
    __shared__ double sLU[YCH * 8], sA2[YCH * 8], sB2[YCH * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    const double c = 1.0 / (P.beta * P.nu * P.dt), lam = S.k2 + c;
    double wt[7], wx[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wt[k] = wx[k] = 0.0;
    D1BwdR bd; bd.init();
    HeptaFac hf; hf.init();
    RhsFwd<double> rz, ro, rb;
    rz.z1 = rz.z2 = rz.z3 = 0.0; ro.z1 = ro.z2 = ro.z3 = 0.0; rb.z1 = rb.z2 = rb.z3 = 0.0;
    const int nit = ny + 3;
    for (int it0 = 0; it0 < nit; it0 += YCH) {
        __syncthreads();
        stage8(sLU, P.t[0].lu1, ny, it0, ny - 1, -1);          // orientation-0 LU of A1 at physical row j = ny-1-ii
        stage8(sA2, P.t[1].A2, ny, it0, -3, 1); stage8(sB2, P.t[1].B2, ny, it0, -3, 1);   // orientation 1, virtual row i = ii-3
        __syncthreads();
        const int ite = min(it0 + YCH, nit);
        for (int ii = it0; ii < ite; ++ii) {
            const int j = ny - 1 - ii;
            double x = 0.0, t = 0.0;
            if (S.act && j >= 0) {
                const size_t o = (size_t)j * P.nm + S.m;
                if (j - CHAN_PF >= 0) { const size_t op = o - (size_t)CHAN_PF * P.nm; pf2(zd_zphi + op); pf2(H2 + op); pf2(phi + op); pf2(hv + op); pf2(rom_zom + op); }
                const double dd = bd.step(sLU + (ii - it0) * 8, *cpart(zd_zphi, o, part));
                const double h2 = *cpart(H2, o, part), hp = *cpart(hv, o, part);
                x = *cpart(phi, o, part);
                const double h = -S.k2 * h2 - dd;
                *wpart(hv, o, part) = h;
                t = x + P.dt * (P.gamma * h + P.zeta * hp);
            }
            push(wx, x); push(wt, t);
            const int i = ii - 3;
            if (S.act && i >= 0) {
                const size_t o = (size_t)(ny - 1 - i) * P.nm + S.m;
                const int e = (ii - it0) * 8;
                double a[7];
                const double romv = *cpart(rom_zom, o, part);
                helm_row_s(ny, i, lam, sA2 + e, sB2 + e, a);
                const double r = helm_rhs_s(P, i, c, S.k2, sA2 + e, sB2 + e, wt, wx);
                const double4 f = hf.reduce(a);
                *wpart(zd_zphi, o, part) = rz.step(hf, r);
                *wpart(rom_zom, o, part) = ro.step(hf, romv);
                if (part == 0) facA[o] = make_double2(f.x, f.y);
                else facB[o] = make_double2(f.z, rb.step(hf, i == 0 ? 1.0 : 0.0));   // virtual row 0 = wall y=+1
            }
        }
    }
}

// =====================================================================================================
// SC (ascending).  reads facA, facB, z_om, z_phi; writes om_y^new, phi_p (over z_phi), phi_ab = {phi_a, phi_b},
// the Poisson factor rows (over facA, facB), z_vp, z_vab = {z_va, z_vb} (over z_om), coef = (c_a, c_b).
// u3 of the Helmholtz factor is not stored (its slot carries z_b): it is the band entry b2[6] - lam a2[6]
// of the orientation-1 row, recomputed here.
// =====================================================================================================
__global__ void __launch_bounds__(YNT) k_sc(YParams P, double2* facA, double2* facB, double2* zom_zvab, double2* zphi_phip,
                                            double2* __restrict__ omy, double2* __restrict__ phiab, double2* __restrict__ zvp,
                                            double4* __restrict__ coef) {
    __shared__ double sA2[YCH * 8], sB2[YCH * 8], sWm[YCH], sWp[YCH], sA6[YCH], sB6[YCH];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    const double c = 1.0 / (P.beta * P.nu * P.dt), lam = S.k2 + c;
    double wp_[7], wab[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wp_[k] = wab[k] = 0.0;
    RhsBwd<double> bo, bp, bab;
    bo.x1 = bo.x2 = bo.x3 = 0.0; bp.x1 = bp.x2 = bp.x3 = 0.0; bab.x1 = bab.x2 = bab.x3 = 0.0;
    HeptaFac hf; hf.init();
    RhsFwd<double> rp, rab;
    rp.z1 = rp.z2 = rp.z3 = 0.0; rab.z1 = rab.z2 = rab.z3 = 0.0;
    double gm1 = 0, gm2 = 0, gm3 = 0, gp1 = 0, gp2 = 0, gp3 = 0;      // adjoint solution U^T g = w at rows j-1..j-3
    double spm = 0, spp = 0, sabm = 0, sabp = 0;                      // w- . v_p, w+ . v_p, w- . v_ab, w+ . v_ab
    const int nit = ny + 3;
    for (int it0 = 0; it0 < nit; it0 += YCH) {
        __syncthreads();
        stage8(sA2, P.t[0].A2, ny, it0, -3, 1); stage8(sB2, P.t[0].B2, ny, it0, -3, 1);
        stage1(sWm, P.wm, ny, it0, -3, 1); stage1(sWp, P.wp, ny, it0, -3, 1);
        stage_col6(sA6, P.t[1].A2, ny, it0, ny - 1, -1); stage_col6(sB6, P.t[1].B2, ny, it0, ny - 1, -1);   // virtual row ny-1-jj
        __syncthreads();
        const int ite = min(it0 + YCH, nit);
        for (int jj = it0; jj < ite; ++jj) {
            double pp = 0.0, pab = 0.0;
            if (S.act && jj < ny) {
                const size_t o = (size_t)jj * P.nm + S.m;
                if (jj + CHAN_PF < ny) { const size_t op = o + (size_t)CHAN_PF * P.nm; pf2(facA + op); pf2(facB + op); pf2(zom_zvab + op); pf2(zphi_phip + op); }
                const double2 fa = facA[o], fb = facB[o];
                const int iv = ny - 1 - jj;
                const double u3 = (iv == 0 || iv == ny - 1) ? 0.0 : sB6[jj - it0] - lam * sA6[jj - it0];
                const double4 f = make_double4(fa.x, fa.y, fb.x, u3);
                *wpart(omy, o, part) = bo.step(f, *cpart(zom_zvab, o, part));
                pp = bp.step(f, *cpart(zphi_phip, o, part));
                // problem a: phi(-1) = 1, its forward-eliminated right-hand side is the unit vector at the last
                // virtual row (physical row 0); problem b: phi(+1) = 1, z_b from SB
                pab = bab.step(f, part ? fb.y : (jj == 0 ? 1.0 : 0.0));
                *wpart(zphi_phip, o, part) = pp;
                *wpart(phiab, o, part) = pab;
            }
            push(wp_, pp); push(wab, pab);
            const int j = jj - 3;
            if (S.act && j >= 0) {
                const size_t o = (size_t)j * P.nm + S.m;
                const int e = (jj - it0) * 8;
                double a[7];
                helm_row_s(ny, j, S.k2, sA2 + e, sB2 + e, a);
                const bool wall = (j == 0 || j == ny - 1);
                const double r = wall ? 0.0 : band7s(sA2 + e, wp_), rr = wall ? 0.0 : band7s(sA2 + e, wab);
                // adjoint recurrence with the rows j-1, j-2, j-3 of U still in hf
                const double tm = sWm[jj - it0] - hf.u11 * gm1 - hf.u22 * gm2 - hf.u33 * gm3;
                const double tp = sWp[jj - it0] - hf.u11 * gp1 - hf.u22 * gp2 - hf.u33 * gp3;
                const double4 f = hf.reduce(a);
                const double gm = tm * f.x, gp = tp * f.x;
                gm3 = gm2; gm2 = gm1; gm1 = gm; gp3 = gp2; gp2 = gp1; gp1 = gp;
                const double zp = rp.step(hf, r), zab = rab.step(hf, rr);
                spm += gm * zp; spp += gp * zp; sabm += gm * zab; sabp += gp * zab;
                *wpart(zvp, o, part) = zp;
                *wpart(zom_zvab, o, part) = zab;
                if (part == 0) facA[o] = make_double2(f.x, f.y); else facB[o] = make_double2(f.z, f.w);
            }
        }
    }
    // influence matrix (step 7): G = [[w-.v_a, w-.v_b],[w+.v_a, w+.v_b]], (c_a, c_b) = -G^-1 (w-.v_p, w+.v_p)
    const double oabm = __shfl_xor_sync(0xffffffffu, sabm, 1), oabp = __shfl_xor_sync(0xffffffffu, sabp, 1);
    if (S.act) {
        const double dam = part ? oabm : sabm, dap = part ? oabp : sabp, dbm = part ? sabm : oabm, dbp = part ? sabp : oabp;
        const double det = dam * dbp - dbm * dap;
        const double ca = (dbp * (-spm) - dbm * (-spp)) / det;
        const double cb = (-dap * (-spm) + dam * (-spp)) / det;
        double* cf = reinterpret_cast<double*>(coef + S.m);
        cf[part] = ca; cf[2 + part] = cb;
    }
}

// =====================================================================================================
// SD (descending).  reads Poisson factor rows, z_vp, z_vab, phi_p, phi_ab, coef; writes v (over phi_ab),
// phi, zv = forward D1(v) in orientation 1 (over phi_p).
// =====================================================================================================
__global__ void __launch_bounds__(YNT) k_sd(YParams P, const double2* __restrict__ facA, const double2* __restrict__ facB,
                                            const double2* __restrict__ zvp, const double2* __restrict__ zvab,
                                            double2* phip_zv, double2* phiab_v, const double4* __restrict__ coef,
                                            double2* __restrict__ phi) {
    __shared__ double sB1[YCH * 8], sLU[YCH * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    double ca = 0.0, cb = 0.0;
    if (S.act) { const double* cf = reinterpret_cast<const double*>(coef + S.m); ca = cf[part]; cb = cf[2 + part]; }
    double wv[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wv[k] = 0.0;
    RhsBwd<double> bv; bv.x1 = bv.x2 = bv.x3 = 0.0;
    D1FwdR fw; fw.init();
    const int nit = ny + 3;
    for (int it0 = 0; it0 < nit; it0 += YCH) {
        __syncthreads();
        stage8(sB1, P.t[1].B1, ny, it0, -3, 1); stage8(sLU, P.t[1].lu1, ny, it0, -3, 1);
        __syncthreads();
        const int ite = min(it0 + YCH, nit);
        for (int ii = it0; ii < ite; ++ii) {
            const int j = ny - 1 - ii;
            double v = 0.0;
            // each lane reads only the slot of phi_ab / z_vab it owns (and later overwrites); the partner's
            // value comes by shuffle, so the in-place update of phi_ab by v is free of read/write hazards
            const bool on = S.act && j >= 0;
            const size_t o = on ? (size_t)j * P.nm + S.m : 0;
            double myz = 0.0, myp = 0.0, zp = 0.0, pp = 0.0;
            double2 fa = make_double2(1.0, 0.0), fb = make_double2(0.0, 0.0);
            if (on) {
                if (j - CHAN_PF >= 0) { const size_t op = o - (size_t)CHAN_PF * P.nm; pf2(facA + op); pf2(facB + op); pf2(zvp + op); pf2(zvab + op); pf2(phip_zv + op); pf2(phiab_v + op); }
                myz = *cpart(zvab, o, part); myp = *cpart(phiab_v, o, part);
                fa = facA[o]; fb = facB[o];
                zp = *cpart(zvp, o, part); pp = *cpart(phip_zv, o, part);
            }
            const double otz = __shfl_xor_sync(0xffffffffu, myz, 1), otp = __shfl_xor_sync(0xffffffffu, myp, 1);
            if (on) {
                const double za = part ? otz : myz, zb = part ? myz : otz, pa = part ? otp : myp, pb = part ? myp : otp;
                v = bv.step(make_double4(fa.x, fa.y, fb.x, fb.y), zp + ca * za + cb * zb);
                *wpart(phiab_v, o, part) = v;
                *wpart(phi, o, part) = pp + ca * pa + cb * pb;
            }
            push(wv, v);
            const int i = ii - 3;
            if (S.act && i >= 0) {
                const int e = (ii - it0) * 8;
                *wpart(phip_zv, (size_t)(ny - 1 - i) * P.nm + S.m, part) = fw.step(sLU + e, band7s(sB1 + e, wv));
            }
        }
    }
}

// =====================================================================================================
// SD0 (descending): zv = forward D1(v) in orientation 1 alone -- the entry of the a1 chain when the state comes
// from chan_set_state instead of from SD.
// =====================================================================================================
__global__ void __launch_bounds__(YNT) k_sd0(YParams P, const double2* __restrict__ v, double2* __restrict__ zv) {
    __shared__ double sB1[YCH * 8], sLU[YCH * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    double wv[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wv[k] = 0.0;
    D1FwdR fw; fw.init();
    const int nit = ny + 3;
    for (int it0 = 0; it0 < nit; it0 += YCH) {
        __syncthreads();
        stage8(sB1, P.t[1].B1, ny, it0, -3, 1); stage8(sLU, P.t[1].lu1, ny, it0, -3, 1);
        __syncthreads();
        const int ite = min(it0 + YCH, nit);
        for (int ii = it0; ii < ite; ++ii) {
            const int j = ny - 1 - ii;
            push(wv, (S.act && j >= 0) ? *cpart(v, (size_t)j * P.nm + S.m, part) : 0.0);
            const int i = ii - 3;
            if (S.act && i >= 0) {
                const int e = (ii - it0) * 8;
                *wpart(zv, (size_t)(ny - 1 - i) * P.nm + S.m, part) = fw.step(sLU + e, band7s(sB1 + e, wv));
            }
        }
    }
}

// =====================================================================================================
// SE (ascending, step a1).  reads zv, om_y (mean mode: U, W); writes u, w, zu = forward D1(u) (over zv),
// zw = forward D1(w), both in orientation 0.  u = i (kx dv - kz om_y)/k2, w = i (kz dv + kx om_y)/k2.
// The z-Nyquist slot is written as zeros (the buffers double as y-phase scratch).
// =====================================================================================================
__global__ void __launch_bounds__(YNT) k_se(YParams P, double2* zv_zu, const double2* __restrict__ omy,
                                            const double* __restrict__ U, const double* __restrict__ W,
                                            double2* __restrict__ u, double2* __restrict__ w_, double2* __restrict__ zw) {
    __shared__ double sLUb[YCH * 8], sB1[YCH * 8], sLU[YCH * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    const bool mean = S.inplane && S.m == 0;
    const bool wr = S.inplane;                  // every in-plane slot is written (zeros where there is no mode)
    double wu[7], ww[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wu[k] = ww[k] = 0.0;
    D1BwdR bs; bs.init();
    D1FwdR fu, fw; fu.init(); fw.init();
    const int nit = ny + 3;
    for (int it0 = 0; it0 < nit; it0 += YCH) {
        __syncthreads();
        stage8(sLUb, P.t[1].lu1, ny, it0, ny - 1, -1);      // back substitution of the orientation-1 system: virtual row ny-1-jj
        stage8(sB1, P.t[0].B1, ny, it0, -3, 1); stage8(sLU, P.t[0].lu1, ny, it0, -3, 1);
        __syncthreads();
        const int ite = min(it0 + YCH, nit);
        for (int jj = it0; jj < ite; ++jj) {
            double a = 0.0, b = 0.0;
            const bool ld = S.act && jj < ny;
            const size_t o = (size_t)min(jj, ny - 1) * P.nm + (S.inplane ? S.m : 0);
            if (ld) {
                if (jj + CHAN_PF < ny) { const size_t op = o + (size_t)CHAN_PF * P.nm; pf2(zv_zu + op); pf2(omy + op); }
                const double dv = bs.step(sLUb + (jj - it0) * 8, *cpart(zv_zu, o, part));
                const double oy = *cpart(omy, o, part);
                a = S.kx * dv - S.kz * oy;
                b = S.kz * dv + S.kx * oy;
            }
            // i * (a_re + i a_im) = -a_im + i a_re: each lane needs its partner's component
            const double oa = __shfl_xor_sync(0xffffffffu, a, 1), ob = __shfl_xor_sync(0xffffffffu, b, 1);
            double uj = 0.0, wj = 0.0;
            if (ld) { uj = (part ? oa : -oa) / S.k2; wj = (part ? ob : -ob) / S.k2; }
            if (mean && jj < ny && part == 0) { uj = __ldg(U + jj); wj = __ldg(W + jj); }
            if (wr && jj < ny) { *wpart(u, o, part) = uj; *wpart(w_, o, part) = wj; }
            push(wu, uj); push(ww, wj);
            const int j = jj - 3;
            if (wr && j >= 0) {
                const size_t oc = (size_t)j * P.nm + S.m;
                const int e = (jj - it0) * 8;
                *wpart(zv_zu, oc, part) = fu.step(sLU + e, band7s(sB1 + e, wu));
                *wpart(zw, oc, part) = fw.step(sLU + e, band7s(sB1 + e, ww));
            }
        }
    }
}

// =====================================================================================================
// SF (descending, step a1).  reads zu, zw, v; writes om_x = D1 w - i kz v, om_z = i kx v - D1 u (om_z over zw).
// =====================================================================================================
__global__ void __launch_bounds__(YNT) k_sf(YParams P, const double2* __restrict__ zu, double2* zw_oz, const double2* __restrict__ v,
                                            double2* __restrict__ ox) {
    __shared__ double sLU[YCH * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    const bool wr = S.inplane;
    const bool hasv = S.act;                    // v of the mean mode and of the Nyquist slot counts as zero
    D1BwdR bu, bw; bu.init(); bw.init();
    for (int it0 = 0; it0 < ny; it0 += YCH) {
        __syncthreads();
        stage8(sLU, P.t[0].lu1, ny, it0, ny - 1, -1);
        __syncthreads();
        const int ite = min(it0 + YCH, ny);
        for (int ii = it0; ii < ite; ++ii) {
            const int j = ny - 1 - ii;
            if (!wr) continue;
            const size_t o = (size_t)j * P.nm + S.m;
            if (j - CHAN_PF >= 0) { const size_t op = o - (size_t)CHAN_PF * P.nm; pf2(zu + op); pf2(zw_oz + op); pf2(v + op); }
            const double* lu = sLU + (ii - it0) * 8;
            const double du = bu.step(lu, *cpart(zu, o, part));
            const double dw = bw.step(lu, *cpart(zw_oz, o, part));
            const c2 vj = hasv ? ldc(v + o) : mk(0, 0);
            // -i kz v = (kz v.y, -kz v.x);  i kx v = (-kx v.y, kx v.x)
            *wpart(ox, o, part) = part ? dw - S.kz * vj.x : dw + S.kz * vj.y;
            *wpart(zw_oz, o, part) = part ? S.kx * vj.x - du : -S.kx * vj.y - du;
        }
    }
}

}  // namespace chn
