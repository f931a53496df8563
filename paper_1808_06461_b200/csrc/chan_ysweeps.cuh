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
// Row tables are staged through shared memory in chunks of YR = 21 iterations; the inputs of the next row are
// loaded one step ahead of their use, and the rows needed CHAN_PF steps later are prefetched into L2.
#pragma once
#include <cuda_runtime.h>

#include <type_traits>
#include <utility>

#include "chan_ykernels.cuh"

namespace chn {

#ifndef CHAN_YNT
#define CHAN_YNT 128
#endif
constexpr int YNT = CHAN_YNT;    // threads per CTA (two per mode): 128 = 64 modes

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

// rows r(it) = a + b*it, it = it0 .. it0+n-1, of an [ny][8] table -> dst[n][8] (zeros outside)
__device__ __forceinline__ void stage8n(double* dst, const double* tab, int ny, int it0, int a, int b, int n) {
    for (int e = threadIdx.x; e < n * 8; e += blockDim.x) {
        const int r = a + b * (it0 + (e >> 3));
        dst[e] = (r >= 0 && r < ny) ? __ldg(tab + (size_t)r * 8 + (e & 7)) : 0.0;
    }
}
// the same for column col of a table with row pitch `pitch`
__device__ __forceinline__ void stage1n(double* dst, const double* vec, int ny, int it0, int a, int b, int n, int col, int pitch) {
    for (int e = threadIdx.x; e < n; e += blockDim.x) {
        const int r = a + b * (it0 + e);
        dst[e] = (r >= 0 && r < ny) ? __ldg(vec + (size_t)r * pitch + col) : 0.0;
    }
}

// ---- rotation-free state ------------------------------------------------------------------------------
// The row loops are unrolled by YR = 21 = lcm(7, 3) so that the 7-wide band windows and the 3-deep recurrence
// histories are register files indexed by compile-time constants: slot R%7 (R%3) is overwritten by the newest
// entry instead of shifting every entry every row (the shifts were ~40% of the instructions of a sweep).
constexpr int YR = 21;
template <class F, int... I> __device__ __forceinline__ void static_for_impl(F&& f, std::integer_sequence<int, I...>) {
    (f(std::integral_constant<int, I>{}), ...);
}
template <int N, class F> __device__ __forceinline__ void static_for(F&& f) { static_for_impl(f, std::make_integer_sequence<int, N>{}); }

// window: entry written at step R sits in slot R%7; the band product at step R sees the entries of steps
// R-6 .. R in coefficient order 0 .. 6
template <int R> __device__ __forceinline__ double band7r(const double* c, const double (&w)[7]) {
    double s = c[0] * w[(R + 1) % 7];
#pragma unroll
    for (int k = 1; k < 7; ++k) s += c[k] * w[(R + 1 + k) % 7];
    return s;
}
// a chunk of YR iterations it0 .. it0+YR-1 whose rows are all interior for every index a sweep forms from them: the trailing
// row (iteration - 3) is past the first wall, and the row CHAN_PF ahead of the last iteration still exists
__device__ __forceinline__ bool interior_chunk(int it0, int ny) { return it0 >= YR && it0 + YR + CHAN_PF <= ny; }
struct Rec3 { double x[3]; __device__ __forceinline__ void init() { x[0] = x[1] = x[2] = 0.0; } };
// back substitution with a factor row f = {1/d, u1, u2, u3}
template <int R> __device__ __forceinline__ double bwd3(Rec3& s, double4 f, double z) {
    const double x = (z - f.y * s.x[(R + 2) % 3] - f.z * s.x[(R + 1) % 3] - f.w * s.x[R % 3]) * f.x;
    s.x[R % 3] = x;
    return x;
}
// constant-LU first derivative rows {l1,l2,l3,1/u,u1,u2,u3,0}
template <int R> __device__ __forceinline__ double d1fwd3(Rec3& s, const double* lu, double r) {
    const double z = r - lu[0] * s.x[(R + 2) % 3] - lu[1] * s.x[(R + 1) % 3] - lu[2] * s.x[R % 3];
    s.x[R % 3] = z;
    return z;
}
template <int R> __device__ __forceinline__ double d1bwd3(Rec3& s, const double* lu, double z) {
    const double g = (z - lu[4] * s.x[(R + 2) % 3] - lu[5] * s.x[(R + 1) % 3] - lu[6] * s.x[R % 3]) * lu[3];
    s.x[R % 3] = g;
    return g;
}
// per-mode heptadiagonal elimination: rows i-1, i-2, i-3 of U live in slots (R+2)%3, (R+1)%3, R%3
struct Hepta3 {
    double di[3], u1[3], u2[3], u3[3];
    double l1, l2, l3;
    __device__ __forceinline__ void init() {
#pragma unroll
        for (int k = 0; k < 3; ++k) { di[k] = 1.0; u1[k] = u2[k] = u3[k] = 0.0; }
        l1 = l2 = l3 = 0.0;
    }
    template <int R> __device__ __forceinline__ double4 reduce(double (&a)[7]) {
        constexpr int s1 = (R + 2) % 3, s2 = (R + 1) % 3, s3 = R % 3;
        l3 = a[0] * di[s3];
        a[1] -= l3 * u1[s3]; a[2] -= l3 * u2[s3]; a[3] -= l3 * u3[s3];
        l2 = a[1] * di[s2];
        a[2] -= l2 * u1[s2]; a[3] -= l2 * u2[s2]; a[4] -= l2 * u3[s2];
        l1 = a[2] * di[s1];
        a[3] -= l1 * u1[s1]; a[4] -= l1 * u2[s1]; a[5] -= l1 * u3[s1];
        const double d = 1.0 / a[3];
        di[s3] = d; u1[s3] = a[4]; u2[s3] = a[5]; u3[s3] = a[6];
        return make_double4(d, a[4], a[5], a[6]);
    }
    // forward substitution of a right-hand side with the multipliers of the row just reduced
    template <int R> __device__ __forceinline__ double fwd(Rec3& s, double r) const {
        const double z = r - l3 * s.x[R % 3] - l2 * s.x[(R + 1) % 3] - l1 * s.x[(R + 2) % 3];
        s.x[R % 3] = z;
        return z;
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

template <bool IN> __device__ __forceinline__ void helm_row_t(int ny, int i, double lam, const double* a2, const double* b2, double (&a)[7]) {
    if constexpr (IN) {
#pragma unroll
        for (int k = 0; k < 7; ++k) a[k] = b2[k] - lam * a2[k];
    } else helm_row_s(ny, i, lam, a2, b2, a);
}
__device__ __forceinline__ const double* cpart(const double2* a, size_t o, int part) { return reinterpret_cast<const double*>(a + o) + part; }
__device__ __forceinline__ double* wpart(double2* a, size_t o, int part) { return reinterpret_cast<double*>(a + o) + part; }

// =====================================================================================================
// SA (ascending).  reads H1, H3, om_y, h_g^prev; writes h_g (in place), zd, R_om.
// =====================================================================================================
__global__ void __launch_bounds__(YNT) k_sa(YParams P, const double2* __restrict__ H1, const double2* __restrict__ H3,
                                            const double2* __restrict__ omy, double2* __restrict__ hg,
                                            double2* __restrict__ zd, double2* __restrict__ rom) {
    __shared__ __align__(16) double sB1[YR * 8], sLU[YR * 8], sA2[YR * 8], sB2[YR * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    const double c = 1.0 / (P.beta * P.nu * P.dt);
    const bool hist = (P.zeta != 0.0);
    double wd[7], wt[7], wx[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wd[k] = wt[k] = wx[k] = 0.0;
    Rec3 fd; fd.init();
    const int nit = ny + 3;
    size_t ol = S.inplane ? (size_t)S.m : 0;
    const size_t nm = (size_t)P.nm;
    for (int it0 = 0; it0 < nit; it0 += YR) {
        __syncthreads();
        stage8n(sB1, P.t[0].B1, ny, it0, -3, 1, YR); stage8n(sLU, P.t[0].lu1, ny, it0, -3, 1, YR);
        stage8n(sA2, P.t[0].A2, ny, it0, -3, 1, YR); stage8n(sB2, P.t[0].B2, ny, it0, -3, 1, YR);
        __syncthreads();
        auto row = [&](auto ic, auto interior) {      // IN: a chunk of interior rows, the range checks fold (see k_se)
            constexpr int R = decltype(ic)::value;
            constexpr bool IN = decltype(interior)::value;
            const int jj = it0 + R;
            if (IN || jj < nit) {
                double d = 0.0, x = 0.0, t = 0.0;
                if (S.act && (IN || jj < ny)) {
                    if (IN || jj + CHAN_PF < ny) { const size_t op = ol + (size_t)CHAN_PF * nm; pf2(H1 + op); pf2(H3 + op); pf2(omy + op); if (hist) pf2(hg + op); }
                    const c2 h1 = ldc(H1 + ol), h3 = ldc(H3 + ol);
                    x = *cpart(omy, ol, part);
                    const double gp = hist ? *cpart(hg, ol, part) : 0.0;     // zeta_1 = 0: the first substep reads no history
                    // h_g = i kz h1 - i kx h3 ; d = i kx h1 + i kz h3
                    const double g = part ? (S.kz * h1.x - S.kx * h3.x) : (-S.kz * h1.y + S.kx * h3.y);
                    d = part ? (S.kx * h1.x + S.kz * h3.x) : (-S.kx * h1.y - S.kz * h3.y);
                    *wpart(hg, ol, part) = g;
                    t = x + P.dt * (P.gamma * g + P.zeta * gp);
                }
                wd[R % 7] = d; wx[R % 7] = x; wt[R % 7] = t;
                const int j = jj - 3;
                if (S.act && (IN || j >= 0)) {
                    const size_t oc = ol - 3 * nm;
                    *wpart(zd, oc, part) = d1fwd3<R>(fd, sLU + R * 8, band7r<R>(sB1 + R * 8, wd));
                    double r = 0.0;
                    if (IN || (j != 0 && j != ny - 1)) {
                        const double at = band7r<R>(sA2 + R * 8, wt), bx = band7r<R>(sB2 + R * 8, wx), ax = band7r<R>(sA2 + R * 8, wx);
                        r = -c * (at + P.alpha * P.nu * P.dt * (bx - S.k2 * ax));
                    }
                    *wpart(rom, oc, part) = r;
                }
                ol += nm;
            }
        };
        // (the interior-chunk variant cost this sweep 20 registers and a CTA per SM: measured slower, not dispatched)
        static_for<YR>([&](auto ic) { row(ic, std::false_type{}); });
    }
}

// =====================================================================================================
// SB (descending).  reads zd, H2, phi, h_v^prev, R_om; writes h_v (in place), facA = {1/d, u1},
// facB = {u2, z_b}, z_phi (over zd), z_om (over R_om).  Helmholtz matrix B2 - lam A2 in orientation 1.
// =====================================================================================================
__global__ void __launch_bounds__(YNT, 4) k_sb(YParams P, const double2* __restrict__ H2, const double2* __restrict__ phi,
                                            double2* __restrict__ hv, double2* zd_zphi, double2* rom_zom,
                                            double2* __restrict__ facA, double2* __restrict__ facB) {
    __shared__ __align__(16) double sLU[YR * 8], sA2[YR * 8], sB2[YR * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    const double c = 1.0 / (P.beta * P.nu * P.dt), lam = S.k2 + c;
    const bool hist = (P.zeta != 0.0);
    double wt[7], wx[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wt[k] = wx[k] = 0.0;
    Rec3 bd, rz, ro, rb;
    bd.init(); rz.init(); ro.init(); rb.init();
    Hepta3 hf; hf.init();
    const int nit = ny + 3;
    const size_t nm = (size_t)P.nm;
    // offset of (row j = ny-1-ii, mode m); runs below zero for the three trailing iterations: signed
    long long ol = (long long)(ny - 1) * P.nm + (S.inplane ? S.m : 0);
    double nzd = 0.0, nh2 = 0.0, nhp = 0.0, nph = 0.0;                    // inputs of the next row, loaded one step ahead
    if (S.act) { nzd = *cpart(zd_zphi, (size_t)ol, part); nh2 = *cpart(H2, (size_t)ol, part); nhp = hist ? *cpart(hv, (size_t)ol, part) : 0.0; nph = *cpart(phi, (size_t)ol, part); }
    for (int it0 = 0; it0 < nit; it0 += YR) {
        __syncthreads();
        stage8n(sLU, P.t[0].lu1, ny, it0, ny - 1, -1, YR);        // orientation-0 LU of A1 at physical row j = ny-1-ii
        stage8n(sA2, P.t[1].A2, ny, it0, -3, 1, YR); stage8n(sB2, P.t[1].B2, ny, it0, -3, 1, YR);   // orientation 1, virtual row i = ii-3
        __syncthreads();
        auto row = [&](auto ic, auto interior) {      // IN: a chunk of interior rows, the range checks fold (see k_se)
            constexpr int R = decltype(ic)::value;
            constexpr bool IN = decltype(interior)::value;
            const int ii = it0 + R;
            if (IN || ii < nit) {
                const int j = ny - 1 - ii;
                const int i = ii - 3;
                double x = 0.0, t = 0.0, romv = 0.0;
                const size_t oc = (size_t)(ol + 3 * (long long)nm);     // row ny-1-i = j+3
                if (S.act && (IN || i >= 0)) romv = *cpart(rom_zom, oc, part);
                if (S.act && (IN || j >= 0)) {
                    const size_t o = (size_t)ol;
                    if (IN || j - CHAN_PF >= 0) { const size_t op = o - (size_t)CHAN_PF * nm; pf2(zd_zphi + op); pf2(H2 + op); pf2(phi + op); if (hist) pf2(hv + op); pf2(rom_zom + op); }
                    const double zdv = nzd, h2 = nh2, hp = nhp;
                    x = nph;
                    if (IN || j > 0) { const size_t o1 = o - nm; nzd = *cpart(zd_zphi, o1, part); nh2 = *cpart(H2, o1, part); nhp = hist ? *cpart(hv, o1, part) : 0.0; nph = *cpart(phi, o1, part); }
                    const double dd = d1bwd3<R>(bd, sLU + R * 8, zdv);
                    const double h = -S.k2 * h2 - dd;
                    *wpart(hv, o, part) = h;
                    t = x + P.dt * (P.gamma * h + P.zeta * hp);
                }
                wx[R % 7] = x; wt[R % 7] = t;
                if (S.act && (IN || i >= 0)) {
                    const double* a2 = sA2 + R * 8; const double* b2 = sB2 + R * 8;
                    double a[7];
                    helm_row_t<IN>(ny, i, lam, a2, b2, a);
                    double r = 0.0;
                    if (IN || (i != 0 && i != ny - 1)) {
                        const double at = band7r<R>(a2, wt), bx = band7r<R>(b2, wx), ax = band7r<R>(a2, wx);
                        r = -c * (at + P.alpha * P.nu * P.dt * (bx - S.k2 * ax));
                    }
                    const double4 f = hf.template reduce<R>(a);
                    *wpart(zd_zphi, oc, part) = hf.template fwd<R>(rz, r);
                    *wpart(rom_zom, oc, part) = hf.template fwd<R>(ro, romv);
                    if (part == 0) facA[oc] = make_double2(f.x, f.y);
                    else facB[oc] = make_double2(f.z, hf.template fwd<R>(rb, (!IN && i == 0) ? 1.0 : 0.0));   // virtual row 0 = wall y=+1
                }
                ol -= (long long)nm;
            }
        };
        // (the interior-chunk variant cost this sweep 20 registers and a CTA per SM: measured slower, not dispatched)
        static_for<YR>([&](auto ic) { row(ic, std::false_type{}); });
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
    __shared__ __align__(16) double sA2[YR * 8], sB2[YR * 8], sWm[YR], sWp[YR], sA6[YR], sB6[YR];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    const double c = 1.0 / (P.beta * P.nu * P.dt), lam = S.k2 + c;
    double wp_[7], wab[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wp_[k] = wab[k] = 0.0;
    Rec3 bo, bp, bab, rp, rab, gm, gp;
    bo.init(); bp.init(); bab.init(); rp.init(); rab.init(); gm.init(); gp.init();   // gm, gp: adjoint solution U^T g = w
    Hepta3 hf; hf.init();
    double spm = 0, spp = 0, sabm = 0, sabp = 0;                      // w- . v_p, w+ . v_p, w- . v_ab, w+ . v_ab
    const int nit = ny + 3;
    size_t ol = S.inplane ? (size_t)S.m : 0;                          // offset of (row jj, mode m)
    const size_t nm = (size_t)P.nm;
    // inputs of row jj+1 are loaded while row jj is processed (the factor rows written at row jj-3 trail behind)
    double2 nfa = make_double2(1.0, 0.0), nfb = make_double2(0.0, 0.0); double nzo = 0.0, nzp = 0.0;
    if (S.act) { nfa = facA[ol]; nfb = facB[ol]; nzo = *cpart(zom_zvab, ol, part); nzp = *cpart(zphi_phip, ol, part); }
    for (int it0 = 0; it0 < nit; it0 += YR) {
        __syncthreads();
        stage8n(sA2, P.t[0].A2, ny, it0, -3, 1, YR); stage8n(sB2, P.t[0].B2, ny, it0, -3, 1, YR);
        stage1n(sWm, P.wm, ny, it0, -3, 1, YR, 0, 1); stage1n(sWp, P.wp, ny, it0, -3, 1, YR, 0, 1);
        stage1n(sA6, P.t[1].A2, ny, it0, ny - 1, -1, YR, 6, 8); stage1n(sB6, P.t[1].B2, ny, it0, ny - 1, -1, YR, 6, 8);   // virtual row ny-1-jj
        __syncthreads();
        auto row = [&](auto ic, auto interior) {      // IN: a chunk of interior rows, the range checks fold (see k_se)
            constexpr int R = decltype(ic)::value;
            constexpr bool IN = decltype(interior)::value;
            const int jj = it0 + R;
            if (IN || jj < nit) {
                double pp = 0.0, pab = 0.0;
                if (S.act && (IN || jj < ny)) {
                    if (IN || jj + CHAN_PF < ny) { const size_t op = ol + (size_t)CHAN_PF * nm; pf2(facA + op); pf2(facB + op); pf2(zom_zvab + op); pf2(zphi_phip + op); }
                    const double2 fa = nfa, fb = nfb;
                    const double zo = nzo, zp = nzp;
                    if (IN || jj + 1 < ny) { const size_t o1 = ol + nm; nfa = facA[o1]; nfb = facB[o1]; nzo = *cpart(zom_zvab, o1, part); nzp = *cpart(zphi_phip, o1, part); }
                    const int iv = ny - 1 - jj;
                    const double u3 = (!IN && (iv == 0 || iv == ny - 1)) ? 0.0 : sB6[R] - lam * sA6[R];
                    const double4 f = make_double4(fa.x, fa.y, fb.x, u3);
                    *wpart(omy, ol, part) = bwd3<R>(bo, f, zo);
                    pp = bwd3<R>(bp, f, zp);
                    // problem a: phi(-1) = 1, its forward-eliminated right-hand side is the unit vector at the last
                    // virtual row (physical row 0); problem b: phi(+1) = 1, z_b from SB
                    pab = bwd3<R>(bab, f, part ? fb.y : ((!IN && jj == 0) ? 1.0 : 0.0));
                    *wpart(zphi_phip, ol, part) = pp;
                    *wpart(phiab, ol, part) = pab;
                }
                wp_[R % 7] = pp; wab[R % 7] = pab;
                const int j = jj - 3;
                if (S.act && (IN || j >= 0)) {
                    const size_t oc = ol - 3 * nm;
                    const double* a2 = sA2 + R * 8;
                    double a[7];
                    helm_row_t<IN>(ny, j, S.k2, a2, sB2 + R * 8, a);
                    const bool wall = !IN && (j == 0 || j == ny - 1);
                    const double r = wall ? 0.0 : band7r<R>(a2, wp_), rr = wall ? 0.0 : band7r<R>(a2, wab);
                    // adjoint recurrence with the rows j-1, j-2, j-3 of U still in hf
                    const double tm = sWm[R] - hf.u1[(R + 2) % 3] * gm.x[(R + 2) % 3] - hf.u2[(R + 1) % 3] * gm.x[(R + 1) % 3] - hf.u3[R % 3] * gm.x[R % 3];
                    const double tp = sWp[R] - hf.u1[(R + 2) % 3] * gp.x[(R + 2) % 3] - hf.u2[(R + 1) % 3] * gp.x[(R + 1) % 3] - hf.u3[R % 3] * gp.x[R % 3];
                    const double4 f = hf.template reduce<R>(a);
                    const double gmn = tm * f.x, gpn = tp * f.x;
                    gm.x[R % 3] = gmn; gp.x[R % 3] = gpn;
                    const double zp = hf.template fwd<R>(rp, r), zab = hf.template fwd<R>(rab, rr);
                    spm += gmn * zp; spp += gpn * zp; sabm += gmn * zab; sabp += gpn * zab;
                    *wpart(zvp, oc, part) = zp;
                    *wpart(zom_zvab, oc, part) = zab;
                    if (part == 0) facA[oc] = make_double2(f.x, f.y); else facB[oc] = make_double2(f.z, f.w);
                }
                // both lanes of a mode read facA/facB at row jj+1 while only one of them writes each at row jj-3:
                // keep the pair (and so the four-row gap) in step without relying on implicit warp lockstep
                __syncwarp();
                ol += nm;
            }
        };
        // (the interior-chunk variant pushed this sweep past the 168 registers that let three CTAs share an SM, and was slower
        // under that cap as well: not dispatched)
        static_for<YR>([&](auto ic) { row(ic, std::false_type{}); });
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
    __shared__ __align__(16) double sB1[YR * 8], sLU[YR * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    double ca = 0.0, cb = 0.0;
    if (S.act) { const double* cf = reinterpret_cast<const double*>(coef + S.m); ca = cf[part]; cb = cf[2 + part]; }
    double wv[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wv[k] = 0.0;
    Rec3 bv, fw; bv.init(); fw.init();
    const int nit = ny + 3;
    const size_t nm = (size_t)P.nm;
    long long ol = (long long)(ny - 1) * P.nm + (S.inplane ? S.m : 0);
    double nmyz = 0.0, nmyp = 0.0, nzp = 0.0, npp = 0.0;                 // inputs of the next row, loaded one step ahead
    double2 nfa = make_double2(1.0, 0.0), nfb = make_double2(0.0, 0.0);
    if (S.act) {
        const size_t o0 = (size_t)ol;
        nmyz = *cpart(zvab, o0, part); nmyp = *cpart(phiab_v, o0, part); nfa = facA[o0]; nfb = facB[o0];
        nzp = *cpart(zvp, o0, part); npp = *cpart(phip_zv, o0, part);
    }
    for (int it0 = 0; it0 < nit; it0 += YR) {
        __syncthreads();
        stage8n(sB1, P.t[1].B1, ny, it0, -3, 1, YR); stage8n(sLU, P.t[1].lu1, ny, it0, -3, 1, YR);
        __syncthreads();
        auto row = [&](auto ic, auto interior) {      // IN: a chunk of interior rows, the range checks fold (see k_se)
            constexpr int R = decltype(ic)::value;
            constexpr bool IN = decltype(interior)::value;
            const int ii = it0 + R;
            if (IN || ii < nit) {
                const int j = ny - 1 - ii;
                double v = 0.0;
                // each lane reads only the slot of phi_ab / z_vab it owns (and later overwrites); the partner's
                // value comes by shuffle, so the in-place update of phi_ab by v is free of read/write hazards
                const bool on = S.act && (IN || j >= 0);
                const size_t o = on ? (size_t)ol : 0;
                double myz = 0.0, myp = 0.0, zp = 0.0, pp = 0.0;
                double2 fa = make_double2(1.0, 0.0), fb = make_double2(0.0, 0.0);
                if (on) {
                    if (IN || j - CHAN_PF >= 0) { const size_t op = o - (size_t)CHAN_PF * nm; pf2(facA + op); pf2(facB + op); pf2(zvp + op); pf2(zvab + op); pf2(phip_zv + op); pf2(phiab_v + op); }
                    myz = nmyz; myp = nmyp; fa = nfa; fb = nfb; zp = nzp; pp = npp;
                    if (IN || j > 0) {
                        const size_t o1 = o - nm;
                        nmyz = *cpart(zvab, o1, part); nmyp = *cpart(phiab_v, o1, part); nfa = facA[o1]; nfb = facB[o1];
                        nzp = *cpart(zvp, o1, part); npp = *cpart(phip_zv, o1, part);
                    }
                }
                const double otz = __shfl_xor_sync(0xffffffffu, myz, 1), otp = __shfl_xor_sync(0xffffffffu, myp, 1);
                if (on) {
                    const double za = part ? otz : myz, zb = part ? myz : otz, pa = part ? otp : myp, pb = part ? myp : otp;
                    v = bwd3<R>(bv, make_double4(fa.x, fa.y, fb.x, fb.y), zp + ca * za + cb * zb);
                    *wpart(phiab_v, o, part) = v;
                    *wpart(phi, o, part) = pp + ca * pa + cb * pb;
                }
                wv[R % 7] = v;
                if (S.act && (IN || ii >= 3))
                    *wpart(phip_zv, (size_t)(ol + 3 * (long long)nm), part) = d1fwd3<R>(fw, sLU + R * 8, band7r<R>(sB1 + R * 8, wv));
                ol -= (long long)nm;
            }
        };
        if (interior_chunk(it0, ny)) static_for<YR>([&](auto ic) { row(ic, std::true_type{}); });
        else static_for<YR>([&](auto ic) { row(ic, std::false_type{}); });
    }
}

// =====================================================================================================
// SD0 (descending): zv = forward D1(v) in orientation 1 alone -- the entry of the a1 chain when the state comes
// from chan_set_state instead of from SD.
// =====================================================================================================
__global__ void __launch_bounds__(YNT) k_sd0(YParams P, const double2* __restrict__ v, double2* __restrict__ zv) {
    __shared__ __align__(16) double sB1[YR * 8], sLU[YR * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    double wv[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wv[k] = 0.0;
    Rec3 fw; fw.init();
    const int nit = ny + 3;
    const size_t nm = (size_t)P.nm;
    long long ol = (long long)(ny - 1) * P.nm + (S.inplane ? S.m : 0);
    for (int it0 = 0; it0 < nit; it0 += YR) {
        __syncthreads();
        stage8n(sB1, P.t[1].B1, ny, it0, -3, 1, YR); stage8n(sLU, P.t[1].lu1, ny, it0, -3, 1, YR);
        __syncthreads();
        static_for<YR>([&](auto ic) {
            constexpr int R = decltype(ic)::value;
            const int ii = it0 + R;
            if (ii < nit) {
                wv[R % 7] = (S.act && ii < ny) ? *cpart(v, (size_t)ol, part) : 0.0;
                if (S.act && ii >= 3)
                    *wpart(zv, (size_t)(ol + 3 * (long long)nm), part) = d1fwd3<R>(fw, sLU + R * 8, band7r<R>(sB1 + R * 8, wv));
                ol -= (long long)nm;
            }
        });
    }
}

// =====================================================================================================
// SE (ascending, step a1).  reads zv, om_y (mean mode: U, W); writes u, w, zu = forward D1(u) (over zv),
// zw = forward D1(w), both in orientation 0.  u = i (kx dv - kz om_y)/k2, w = i (kz dv + kx om_y)/k2.
// The z-Nyquist slot is written as zeros (the buffers double as y-phase scratch).
// =====================================================================================================
__global__ void __launch_bounds__(YNT, 6) k_se(YParams P, double2* zv_zu, const double2* __restrict__ omy,
                                            const double* __restrict__ U, const double* __restrict__ W,
                                            double2* __restrict__ u, double2* __restrict__ w_, double2* __restrict__ zw) {
    __shared__ __align__(16) double sLUb[YR * 8], sB1[YR * 8], sLU[YR * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    const bool mean = S.inplane && S.m == 0;
    const bool wr = S.inplane;                  // every in-plane slot is written (zeros where there is no mode)
    const double rk2 = S.act ? 1.0 / S.k2 : 0.0;
    double wu[7], ww[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) wu[k] = ww[k] = 0.0;
    Rec3 bs, fu, fw; bs.init(); fu.init(); fw.init();
    const int nit = ny + 3;
    const size_t nm = (size_t)P.nm;
    size_t ol = S.inplane ? (size_t)S.m : 0;
    double nzv = 0.0, noy = 0.0;
    if (S.act) { nzv = *cpart(zv_zu, ol, part); noy = *cpart(omy, ol, part); }
    for (int it0 = 0; it0 < nit; it0 += YR) {
        __syncthreads();
        stage8n(sLUb, P.t[1].lu1, ny, it0, ny - 1, -1, YR);  // back substitution of the orientation-1 system: virtual row ny-1-jj
        stage8n(sB1, P.t[0].B1, ny, it0, -3, 1, YR); stage8n(sLU, P.t[0].lu1, ny, it0, -3, 1, YR);
        __syncthreads();
        // IN: every row of this chunk is an interior row (no wall, nothing beyond either end within the prefetch distance):
        // the per-row range checks fold away (the sweeps issue 40-60% of their slots, most of it index and predicate work)
        auto row = [&](auto ic, auto interior) {
            constexpr int R = decltype(ic)::value;
            constexpr bool IN = decltype(interior)::value;
            const int jj = it0 + R;
            if (IN || jj < nit) {
                double a = 0.0, b = 0.0;
                const bool ld = S.act && (IN || jj < ny);
                if (ld) {
                    if (IN || jj + CHAN_PF < ny) { const size_t op = ol + (size_t)CHAN_PF * nm; pf2(zv_zu + op); pf2(omy + op); }
                    const double zvv = nzv, oy = noy;
                    if (IN || jj + 1 < ny) { nzv = *cpart(zv_zu, ol + nm, part); noy = *cpart(omy, ol + nm, part); }   // next row, one step ahead
                    const double dv = d1bwd3<R>(bs, sLUb + R * 8, zvv);
                    a = S.kx * dv - S.kz * oy;
                    b = S.kz * dv + S.kx * oy;
                }
                // i * (a_re + i a_im) = -a_im + i a_re: each lane needs its partner's component
                const double oa = __shfl_xor_sync(0xffffffffu, a, 1), ob = __shfl_xor_sync(0xffffffffu, b, 1);
                double uj = 0.0, wj = 0.0;
                if (ld) { uj = (part ? oa : -oa) * rk2; wj = (part ? ob : -ob) * rk2; }
                if (mean && (IN || jj < ny) && part == 0) { uj = __ldg(U + jj); wj = __ldg(W + jj); }
                if (wr && (IN || jj < ny)) { *wpart(u, ol, part) = uj; *wpart(w_, ol, part) = wj; }
                wu[R % 7] = uj; ww[R % 7] = wj;
                if (wr && (IN || jj >= 3)) {
                    const size_t oc = ol - 3 * nm;
                    *wpart(zv_zu, oc, part) = d1fwd3<R>(fu, sLU + R * 8, band7r<R>(sB1 + R * 8, wu));
                    *wpart(zw, oc, part) = d1fwd3<R>(fw, sLU + R * 8, band7r<R>(sB1 + R * 8, ww));
                }
                ol += nm;
            }
        };
        if (interior_chunk(it0, ny)) static_for<YR>([&](auto ic) { row(ic, std::true_type{}); });
        else static_for<YR>([&](auto ic) { row(ic, std::false_type{}); });
    }
}

// =====================================================================================================
// SF (descending, step a1).  reads zu, zw, v; writes om_x = D1 w - i kz v, om_z = i kx v - D1 u (om_z over zw).
// =====================================================================================================
__global__ void __launch_bounds__(YNT) k_sf(YParams P, const double2* __restrict__ zu, double2* zw_oz, const double2* __restrict__ v,
                                            double2* __restrict__ ox) {
    __shared__ __align__(16) double sLU[YR * 8];
    const YS S = ys_setup(P);
    const int ny = P.ny, part = S.part;
    const bool wr = S.inplane;
    const bool hasv = S.act;                    // v of the mean mode and of the Nyquist slot counts as zero
    Rec3 bu, bw; bu.init(); bw.init();
    const size_t nm = (size_t)P.nm;
    long long ol = (long long)(ny - 1) * P.nm + (S.inplane ? S.m : 0);
    double nzu = 0.0, nzw = 0.0; c2 nv = mk(0, 0);
    if (wr) { nzu = *cpart(zu, (size_t)ol, part); nzw = *cpart(zw_oz, (size_t)ol, part); if (hasv) nv = ldc(v + ol); }
    for (int it0 = 0; it0 < ny; it0 += YR) {
        __syncthreads();
        stage8n(sLU, P.t[0].lu1, ny, it0, ny - 1, -1, YR);
        __syncthreads();
        static_for<YR>([&](auto ic) {
            constexpr int R = decltype(ic)::value;
            const int ii = it0 + R;
            if (ii < ny && wr) {
                const size_t o = (size_t)ol;
                if (ii + CHAN_PF < ny) { const size_t op = o - (size_t)CHAN_PF * nm; pf2(zu + op); pf2(zw_oz + op); pf2(v + op); }
                const double zuv = nzu, zwv = nzw;
                const c2 vj = nv;
                if (ii + 1 < ny) { nzu = *cpart(zu, o - nm, part); nzw = *cpart(zw_oz, o - nm, part); if (hasv) nv = ldc(v + o - nm); }
                const double du = d1bwd3<R>(bu, sLU + R * 8, zuv);
                const double dw = d1bwd3<R>(bw, sLU + R * 8, zwv);
                // -i kz v = (kz v.y, -kz v.x);  i kx v = (-kx v.y, kx v.x)
                *wpart(ox, o, part) = part ? dw - S.kz * vj.x : dw + S.kz * vj.y;
                *wpart(zw_oz, o, part) = part ? S.kx * vj.x - du : -S.kx * vj.y - du;
            }
            ol -= (long long)nm;
        });
    }
}

}  // namespace chn
