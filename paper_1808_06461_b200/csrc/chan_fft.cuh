// Wall-parallel (x,z) phase: batched plane FFTs with 3/2-rule zero padding, the pointwise products in
// physical space and the truncation.  Steps a3-a8 and the product part of a13 of DESIGN.md
// ("pseudo-spectral ... fully dealiased by zero padding"), L84 (batched plane FFTs), L124 (filter).
//
// Transform engine.  A length-n transform (n = 2^a 3^b) is a list of register-resident stages of radix
// 2,3,4,6,8,12 (and 16, 18 in the x pass; chan_plan.cpp chooses them), run IN PLACE in shared memory:
//   spectral -> physical: decimation in frequency, e^{+i}, natural order in, digit-reversed order out;
//   physical -> spectral: decimation in time, e^{-i}, the same stage list backwards.
// Physical space is only ever used pointwise, so the digit-reversed order is never undone.
// Stage s (radix R, sub-block m = product of the later radices, ncur = R m) owns a twiddle table
// tw[(k-1) m + p] = exp(-2 pi i p k / ncur), k = 1..R-1, p < m, so that consecutive butterflies read
// consecutive twiddles.  The first and last stage of a z transform read / write global memory directly
// (padding and truncation fused); the last inverse x stage, the products and the first forward x stage are
// one register pass.
//
// Every kernel body is written as `phase(ph, tid, nthreads, ...)` functions separated by barriers, all
// __host__ __device__, so that the index algebra can be exercised on the host without a GPU.
#pragma once
#include <cuda_runtime.h>

#include "chan_ykernels.cuh"

namespace chn {

#define CHAN_MAX_STAGES 8
#ifdef __CUDA_ARCH__
#define CHAN_ASSUME(x) __builtin_assume(x)
#else
#define CHAN_ASSUME(x) ((void)0)
#endif

struct FftStage {
    int R, m;              // radix, sub-block length (product of the later radices)
    const double2* tw;     // (R-1)*m twiddles, see above (unused when m == 1)
};
struct FftDev {
    int n, ns;
    FftStage st[CHAN_MAX_STAGES];
};

CHAN_HD c2 ldtw(const double2* p) {
#ifdef __CUDA_ARCH__
    const double2 v = __ldg(p);
#else
    const double2 v = *p;
#endif
    return mk(v.x, v.y);
}
// streaming global access: the plane data is touched once per kernel, keep it out of L1 so that the
// twiddle tables stay there
CHAN_HD c2 ldstream(const double2* p) {
#ifdef __CUDA_ARCH__
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return mk(v.x, v.y);
#else
    return mk(p->x, p->y);
#endif
}
CHAN_HD void ststream(double2* p, c2 v) {
#ifdef __CUDA_ARCH__
    asm volatile("st.global.L1::no_allocate.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
#else
    p->x = v.x; p->y = v.y;
#endif
}

// ---- small DFTs in registers: natural order in, natural order out; INV: e^{+i}, else e^{-i} ----------
template <bool INV> CHAN_HD c2 rot90(c2 a) { return INV ? mk(-a.y, a.x) : mk(a.y, -a.x); }   // a*(+i) : a*(-i)

template <bool INV> CHAN_HD void dft2(c2& a, c2& b) { const c2 t = a - b; a = a + b; b = t; }
template <bool INV> CHAN_HD void dft3(c2& a0, c2& a1, c2& a2) {
    const double s = 0.86602540378443864676;   // sin(pi/3)
    const c2 t = a1 + a2, d = a1 - a2;
    const c2 m = mk(a0.x - 0.5 * t.x, a0.y - 0.5 * t.y);
    const c2 jd = rot90<INV>(mk(s * d.x, s * d.y));
    a0 = a0 + t; a1 = m + jd; a2 = m - jd;
}
template <bool INV> CHAN_HD void dft4(c2& a0, c2& a1, c2& a2, c2& a3) {
    const c2 s0 = a0 + a2, d0 = a0 - a2, s1 = a1 + a3, d1 = a1 - a3;
    const c2 jd = rot90<INV>(d1);
    a0 = s0 + s1; a2 = s0 - s1; a1 = d0 + jd; a3 = d0 - jd;
}

// a * exp(-i t) (forward) or a * exp(+i t) (inverse), c = cos t, s = sin t
template <bool INV> CHAN_HD c2 mulcs(c2 a, double c, double s) {
    return INV ? mk(a.x * c - a.y * s, a.x * s + a.y * c) : mk(a.x * c + a.y * s, a.y * c - a.x * s);
}
// radix 16 = 4 x 4 (Cooley-Tukey, twiddles w16^(n2 k1))
template <bool INV> CHAN_HD void dft16(c2 (&a)[16]) {
    const double c1 = 0.92387953251128675613, s1 = 0.38268343236508977173, h = 0.70710678118654752440;   // pi/8, pi/4
    c2 y[4][4];
#pragma unroll
    for (int n2 = 0; n2 < 4; ++n2) { c2 p = a[n2], q = a[4 + n2], r = a[8 + n2], s = a[12 + n2]; dft4<INV>(p, q, r, s); y[0][n2] = p; y[1][n2] = q; y[2][n2] = r; y[3][n2] = s; }
    // w16^(n2 k1), angles n2 k1 pi/8
    y[1][1] = mulcs<INV>(y[1][1], c1, s1); y[1][2] = mulcs<INV>(y[1][2], h, h); y[1][3] = mulcs<INV>(y[1][3], s1, c1);
    y[2][1] = mulcs<INV>(y[2][1], h, h); y[2][2] = rot90<INV>(y[2][2]); y[2][3] = mulcs<INV>(y[2][3], -h, h);
    y[3][1] = mulcs<INV>(y[3][1], s1, c1); y[3][2] = mulcs<INV>(y[3][2], -h, h); y[3][3] = mulcs<INV>(y[3][3], -c1, -s1);
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) { c2 p = y[k1][0], q = y[k1][1], r = y[k1][2], s = y[k1][3]; dft4<INV>(p, q, r, s); a[k1] = p; a[k1 + 4] = q; a[k1 + 8] = r; a[k1 + 12] = s; }
}

// radix 9 = 3 x 3 (Cooley-Tukey, twiddles w9^(n2 k1)); in natural order, out natural order
template <bool INV> CHAN_HD void dft9(c2& x0, c2& x1, c2& x2, c2& x3, c2& x4, c2& x5, c2& x6, c2& x7, c2& x8) {
    const double c1 = 0.76604444311897803520, s1 = 0.64278760968653932632;    // 2 pi/9
    const double c2_ = 0.17364817766693034885, s2 = 0.98480775301220805937;   // 4 pi/9
    const double c4 = -0.93969262078590838405, s4 = 0.34202014332566873304;   // 8 pi/9
    // n = 3 n1 + n2: transforms over n1 for n2 = 0, 1, 2
    dft3<INV>(x0, x3, x6); dft3<INV>(x1, x4, x7); dft3<INV>(x2, x5, x8);
    // y[k1][n2] *= w9^(n2 k1):  (k1, n2) = (1,1): x4, (1,2): x5, (2,1): x7, (2,2): x8
    x4 = mulcs<INV>(x4, c1, s1); x5 = mulcs<INV>(x5, c2_, s2); x7 = mulcs<INV>(x7, c2_, s2); x8 = mulcs<INV>(x8, c4, s4);
    // X[k1 + 3 k2] = sum over n2 of y[k1][n2] w3^(n2 k2)
    dft3<INV>(x0, x1, x2); dft3<INV>(x3, x4, x5); dft3<INV>(x6, x7, x8);
    // now x0,x1,x2 = X[0],X[3],X[6]; x3,x4,x5 = X[1],X[4],X[7]; x6,x7,x8 = X[2],X[5],X[8]: back to natural order
    const c2 t1 = x1, t2 = x2, t3 = x3, t5 = x5, t6 = x6, t7 = x7;
    x1 = t3; x2 = t6; x3 = t1; x5 = t7; x6 = t2; x7 = t5;
}
// radix 18 = 2 x 9 by the prime-factor map n = (9 n1 + 2 n2) mod 18, k = (9 k1 + 10 k2) mod 18: no internal twiddles
template <bool INV> CHAN_HD void dft18(c2 (&a)[18]) {
    c2 e0 = a[0], e1 = a[2], e2 = a[4], e3 = a[6], e4 = a[8], e5 = a[10], e6 = a[12], e7 = a[14], e8 = a[16];      // n1 = 0
    c2 o0 = a[9], o1 = a[11], o2 = a[13], o3 = a[15], o4 = a[17], o5 = a[1], o6 = a[3], o7 = a[5], o8 = a[7];      // n1 = 1
    dft9<INV>(e0, e1, e2, e3, e4, e5, e6, e7, e8);
    dft9<INV>(o0, o1, o2, o3, o4, o5, o6, o7, o8);
    // k1 = 0 -> k = (10 k2) mod 18 = 0,10,2,12,4,14,6,16,8;  k1 = 1 -> k = (9 + 10 k2) mod 18 = 9,1,11,3,13,5,15,7,17
    a[0] = e0 + o0; a[9] = e0 - o0; a[10] = e1 + o1; a[1] = e1 - o1; a[2] = e2 + o2; a[11] = e2 - o2;
    a[12] = e3 + o3; a[3] = e3 - o3; a[4] = e4 + o4; a[13] = e4 - o4; a[14] = e5 + o5; a[5] = e5 - o5;
    a[6] = e6 + o6; a[15] = e6 - o6; a[16] = e7 + o7; a[7] = e7 - o7; a[8] = e8 + o8; a[17] = e8 - o8;
}

template <int R, bool INV> CHAN_HD void bfly(c2 (&a)[R]) {
    if constexpr (R == 18) {
        dft18<INV>(a);
    } else if constexpr (R == 16) {
        dft16<INV>(a);
    } else if constexpr (R == 2) {
        dft2<INV>(a[0], a[1]);
    } else if constexpr (R == 3) {
        dft3<INV>(a[0], a[1], a[2]);
    } else if constexpr (R == 4) {
        dft4<INV>(a[0], a[1], a[2], a[3]);
    } else if constexpr (R == 6) {
        // prime-factor map n = (3 n1 + 2 n2) mod 6, k = (3 k1 + 4 k2) mod 6: no internal twiddles
        c2 A0 = a[0], A1 = a[2], A2 = a[4], B0 = a[3], B1 = a[5], B2 = a[1];
        dft3<INV>(A0, A1, A2);
        dft3<INV>(B0, B1, B2);
        a[0] = A0 + B0; a[3] = A0 - B0; a[4] = A1 + B1; a[1] = A1 - B1; a[2] = A2 + B2; a[5] = A2 - B2;
    } else if constexpr (R == 8) {
        const double h = 0.70710678118654752440;
        c2 s0 = a[0] + a[4], d0 = a[0] - a[4], s1 = a[1] + a[5], d1 = a[1] - a[5];
        c2 s2 = a[2] + a[6], d2 = a[2] - a[6], s3 = a[3] + a[7], d3 = a[3] - a[7];
        // d_n *= w8^n (forward w8 = e^{-i pi/4}; inverse its conjugate)
        d1 = INV ? mk((d1.x - d1.y) * h, (d1.x + d1.y) * h) : mk((d1.x + d1.y) * h, (d1.y - d1.x) * h);
        d2 = rot90<INV>(d2);
        d3 = INV ? mk(-(d3.x + d3.y) * h, (d3.x - d3.y) * h) : mk((d3.y - d3.x) * h, -(d3.x + d3.y) * h);
        dft4<INV>(s0, s1, s2, s3);
        dft4<INV>(d0, d1, d2, d3);
        a[0] = s0; a[2] = s1; a[4] = s2; a[6] = s3; a[1] = d0; a[3] = d1; a[5] = d2; a[7] = d3;
    } else {
        static_assert(R == 12, "unsupported radix");
        // prime-factor map n = (4 n1 + 3 n2) mod 12, k = (4 k1 + 9 k2) mod 12: no internal twiddles
        c2 y00 = a[0], y10 = a[4], y20 = a[8];     // n2 = 0
        c2 y01 = a[3], y11 = a[7], y21 = a[11];    // n2 = 1
        c2 y02 = a[6], y12 = a[10], y22 = a[2];    // n2 = 2
        c2 y03 = a[9], y13 = a[1], y23 = a[5];     // n2 = 3
        dft3<INV>(y00, y10, y20); dft3<INV>(y01, y11, y21); dft3<INV>(y02, y12, y22); dft3<INV>(y03, y13, y23);
        dft4<INV>(y00, y01, y02, y03);             // k1 = 0 -> k = 0, 9, 6, 3
        dft4<INV>(y10, y11, y12, y13);             // k1 = 1 -> k = 4, 1, 10, 7
        dft4<INV>(y20, y21, y22, y23);             // k1 = 2 -> k = 8, 5, 2, 11
        a[0] = y00; a[9] = y01; a[6] = y02; a[3] = y03;
        a[4] = y10; a[1] = y11; a[10] = y12; a[7] = y13;
        a[8] = y20; a[5] = y21; a[2] = y22; a[11] = y23;
    }
}

// Twiddles of one butterfly, w^k for k = 1..R-1 with w = exp(-2 pi i p/ncur).  CHAN_TW_POWERS: only w is loaded
// (one 16-byte load) and the powers are formed by at most four successive products each (w2 = w w, w3 = w2 w,
// w4 = w2 w2, ...; error <= ~5 ulp); otherwise all R-1 come from the table.  With the shared-memory carve-out the
// transforms need, L1 keeps almost nothing and every table load is an L2 round trip: ncu showed them as the top
// long-scoreboard stall and ~40% of the memory instructions of the z passes.
#ifndef CHAN_TW_POWERS
#define CHAN_TW_POWERS 1
#endif
template <int R>
CHAN_HD void load_twiddles(const FftStage& S, int m, int p, c2 (&tw)[R - 1 > 0 ? R - 1 : 1]) {
    if constexpr (R > 12) {
        tw[0] = ldtw(S.tw + p);         // radix 16, 18: pass_item forms w^k on the fly (a register file of 15 or 17 powers would spill)
    } else if constexpr (R >= 2) {
#if CHAN_TW_POWERS
        tw[0] = ldtw(S.tw + p);
#pragma unroll
        for (int k = 2; k < R; ++k) tw[k - 1] = cmul(tw[k / 2 - 1], tw[k - k / 2 - 1]);     // w^k = w^(k/2) w^(k - k/2)
#else
#pragma unroll
        for (int k = 1; k < R; ++k) tw[k - 1] = ldtw(S.tw + (size_t)(k - 1) * m + p);
#endif
    }
}

// One butterfly of an in-place pass: elements base + k m, k < R, of sequence q.
//   DIF (inverse direction here): butterfly, then output k times conj(w^k);
//   DIT (forward direction here): input k times w^k, then butterfly.     w[k-1] = table twiddle (e^{-i}).
template <int R, bool INV, bool DIT, class Src, class Dst>
CHAN_HD void pass_item(const Src& src, const Dst& dst, int q, int base, int m, const c2 (&w)[R - 1 > 0 ? R - 1 : 1], bool twiddled) {
    c2 a[R];
#pragma unroll
    for (int k = 0; k < R; ++k) a[k] = src.load(base + k * m, q);
    if constexpr (R > 12) {
        // w^k as three interleaved running products (k mod 3), each stepping by w^3: a single chain of R-2 dependent
        // complex products was the largest fixed-latency stall of the x pass (ncu: "wait"), three chains a third as deep
        const c2 w1 = INV ? mk(w[0].x, -w[0].y) : w[0];
        auto twiddle_all = [&]() {
            const c2 w2 = cmul(w1, w1), w3 = cmul(w2, w1);
            c2 c0 = w3, c1 = w1, c2_ = w2;               // next powers with k = 0, 1, 2 (mod 3): w^3, w^1, w^2
#pragma unroll
            for (int k = 1; k < R; ++k) {
                if (k % 3 == 1) { a[k] = cmul(a[k], c1); if (k + 3 < R) c1 = cmul(c1, w3); }
                else if (k % 3 == 2) { a[k] = cmul(a[k], c2_); if (k + 3 < R) c2_ = cmul(c2_, w3); }
                else { a[k] = cmul(a[k], c0); if (k + 3 < R) c0 = cmul(c0, w3); }
            }
        };
        if (DIT && twiddled) twiddle_all();
        bfly<R, INV>(a);
        if (!DIT && twiddled) twiddle_all();
    } else {
        if (DIT && twiddled) {
#pragma unroll
            for (int k = 1; k < R; ++k) a[k] = cmul(a[k], INV ? mk(w[k - 1].x, -w[k - 1].y) : w[k - 1]);
        }
        bfly<R, INV>(a);
        if (!DIT && twiddled) {
#pragma unroll
            for (int k = 1; k < R; ++k) a[k] = cmul(a[k], INV ? mk(w[k - 1].x, -w[k - 1].y) : w[k - 1]);
        }
    }
#pragma unroll
    for (int k = 0; k < R; ++k) dst.store(base + k * m, q, a[k]);
}

struct PlaneParams {
    int ny, nz, nxh, nzh, mx, mz;
    long long nm;          // nz*nxh
    FftDev fx, fz;
};
struct FieldPtrs { const double2* f[8]; };
struct FieldPtrsW { double2* f[8]; };

// =====================================================================================================
// z transforms: tile of T k_x columns, shared layout [e][T] (column fastest).  Work item = (butterfly b,
// column t), t fastest over the lanes: every shared access of 8 lanes is one contiguous 128-byte row and
// the twiddle of a butterfly is a broadcast load.
// =====================================================================================================
// M > 0: the sub-block length as a compile-time constant (specialised kernels), M = 0: taken from the stage.
template <int R, bool INV, bool DIT, int M = 0, class Src, class Dst>
CHAN_HD void zpass(const Src& src, const Dst& dst, const FftStage& S, int n, int T, int tid, int nt, int half = -1) {
    // half >= 0: only that half of the butterflies (the cluster kernels split a stage between two CTAs)
    const int m = M > 0 ? M : S.m, ncur = R * m, nb = half < 0 ? n / R : n / R / 2, b0 = half > 0 ? nb : 0;
    const int total = nb * T;
    int lgT = 0;
    while ((1 << lgT) < T) ++lgT;               // T is a power of two
    for (int w = tid; w < total; w += nt) {
        const int b = b0 + (w >> lgT), t = w & (T - 1);
        const int blk = b / m, p = b - blk * m;
        if constexpr (M > 0) CHAN_ASSUME(p >= 0 && p < M && blk >= 0 && blk < n / (R * M));   // ranges: the truncating store folds per output
        c2 tw[R - 1 > 0 ? R - 1 : 1];
        if (m > 1) load_twiddles<R>(S, m, p, tw);
        pass_item<R, INV, DIT>(src, dst, t, blk * ncur + p, m, tw, m > 1);
    }
}
// L2 prefetch of the global inputs of every round but the first of the stage that reads global memory: a thread owns
// ceil(nb T / nt) butterflies of that stage and only the first one's loads are in flight when it starts; the later rounds
// then find their rows in L2 (about a third of the DRAM latency) without holding registers for them.
#ifndef CHAN_ZPREFETCH
#define CHAN_ZPREFETCH 1
#endif
template <int R, int M, class Src>
CHAN_HD void zprefetch(const Src& src, int n, int T, int tid, int nt) {
#if CHAN_ZPREFETCH
    const int m = M, ncur = R * m, nb = n / R, total = nb * T;
    int lgT = 0;
    while ((1 << lgT) < T) ++lgT;
    for (int w = tid + nt; w < total; w += nt) {
        const int b = w >> lgT, t = w & (T - 1);
        const int blk = b / m, p = b - blk * m;
#pragma unroll
        for (int k = 0; k < R; ++k) src.prefetch(blk * ncur + p + k * m, t);
    }
#endif
}
template <bool INV, bool DIT, class Src, class Dst>
CHAN_HD void zpass_any(const Src& src, const Dst& dst, const FftStage& S, int n, int T, int tid, int nt) {
    switch (S.R) {
        case 2: zpass<2, INV, DIT>(src, dst, S, n, T, tid, nt); break;
        case 3: zpass<3, INV, DIT>(src, dst, S, n, T, tid, nt); break;
        case 4: zpass<4, INV, DIT>(src, dst, S, n, T, tid, nt); break;
        case 6: zpass<6, INV, DIT>(src, dst, S, n, T, tid, nt); break;
        case 8: zpass<8, INV, DIT>(src, dst, S, n, T, tid, nt); break;
        case 16: zpass<16, INV, DIT>(src, dst, S, n, T, tid, nt); break;
        default: zpass<12, INV, DIT>(src, dst, S, n, T, tid, nt); break;
    }
}

// ---- K2 (a3): zero-pad in k_z, inverse c2c along z -------------------------------------------------
// in: plane-layout field (rows s = k_z slot, nz of them); out: zpad[f][jc][r][p], r = position in the
// digit-reversed physical z order.
struct ZInvIO {
    c2* sm; int T;
    bool gin, gout;                 // this stage reads / writes global memory
    const double2* src;             // plane of the field: [nz][nxh]
    double2* dst;                   // plane of zpad: [mz][nxh]
    int nxh, nzh, nz, mz, p0, tcount;
    bool zband = false;             // shared-memory reads of the zero band of the 3/2 padding (never filled) return zero
    CHAN_HD c2 load(int e, int t) const {
        if (!gin) return (zband && e >= nzh && e <= mz - nzh) ? mk(0, 0) : sm[e * T + t];
        int s = -1;
        if (e < nzh) s = e; else if (e > mz - nzh) s = e - (mz - nz);
        return (s >= 0 && t < tcount) ? ldstream(src + (size_t)s * nxh + p0 + t) : mk(0, 0);
    }
    CHAN_HD void store(int e, int t, c2 v) const {
        if (!gout) { sm[e * T + t] = v; return; }
        if (t < tcount) ststream(dst + (size_t)e * nxh + p0 + t, v);
    }
    CHAN_HD void prefetch(int e, int t) const {      // the global element load(e, t) will read, into L2
#ifdef __CUDA_ARCH__
        int s = -1;
        if (e < nzh) s = e; else if (e > mz - nzh) s = e - (mz - nz);
        if (s >= 0 && t < tcount) asm volatile("prefetch.global.L2 [%0];" ::"l"(src + (size_t)s * nxh + p0 + t));
#endif
    }
};
CHAN_HD void zinv_phase(int ph, int tid, int nt, const PlaneParams& P, int T, c2* sm, const double2* src, double2* dst, int p0) {
    ZInvIO io;
    io.sm = sm; io.T = T; io.gin = (ph == 0); io.gout = (ph == P.fz.ns - 1);
    io.src = src; io.dst = dst; io.nxh = P.nxh; io.nzh = P.nzh; io.nz = P.nz; io.mz = P.mz; io.p0 = p0;
    io.tcount = (P.nxh - p0 < T) ? P.nxh - p0 : T;
    zpass_any<true, false>(io, io, P.fz.st[ph], P.mz, T, tid, nt);
}

// ---- K4 (a7-a8): forward c2c along z, truncate, scale ----------------------------------------------
//   filt 0: retained modes into plane-layout fields (Nyquist slot zeroed), all p < pin = nxh;
//   filt 1: |q| <= kzc, p <= kxc into out[j][2kzc+1][kxc+1] (complex128);  filt 2: the same as complex64.
// in: xh[f][jc][r][pin].
struct ZFwdIO {
    c2* sm; int T;
    bool gin, gout;
    const double2* src;             // plane of xh: [mz][pin]
    double2* dst;                   // filt 0: plane [nz][nxh]; filt 1: plane [2kzc+1][kxc+1]
    int pin, nxh, nzh, nz, mz, p0, tcount, filt, kxc, kzc;
    double scale;
    CHAN_HD c2 load(int e, int t) const {
        if (!gin) return sm[e * T + t];
        return (t < tcount) ? ldstream(src + (size_t)e * pin + p0 + t) : mk(0, 0);
    }
    CHAN_HD void prefetch(int e, int t) const {
#ifdef __CUDA_ARCH__
        if (t < tcount) asm volatile("prefetch.global.L2 [%0];" ::"l"(src + (size_t)e * pin + p0 + t));
#endif
    }
    CHAN_HD void store(int e, int t, c2 v) const {
        if (!gout) { sm[e * T + t] = v; return; }
        if (t >= tcount) return;
        if (!filt) {
            int s;
            if (e < nzh) s = e; else if (e > mz - nzh) s = e - (mz - nz); else if (e == nzh) { s = nzh; v = mk(0, 0); } else return;
            ststream(dst + (size_t)s * nxh + p0 + t, mk(v.x * scale, v.y * scale));
        } else {
            const int nr = 2 * kzc + 1, npk = kxc + 1;
            int rr;
            if (e <= kzc) rr = e; else if (e >= mz - kzc) rr = e - mz + nr; else return;
            if (p0 + t >= npk) return;
            if (filt == 1) ststream(dst + (size_t)rr * npk + p0 + t, mk(v.x * scale, v.y * scale));
            else           // filt 2: the database in binary32, rounded once (to nearest even) from the fp64 result
                reinterpret_cast<float2*>(dst)[(size_t)rr * npk + p0 + t] = make_float2((float)(v.x * scale), (float)(v.y * scale));
        }
    }
};
CHAN_HD void zfwd_phase(int ph, int tid, int nt, const PlaneParams& P, int T, c2* sm, const double2* src, double2* dst, int pin,
                        int p0, double scale, int filt, int kxc, int kzc) {
    ZFwdIO io;
    io.sm = sm; io.T = T; io.gin = (ph == 0); io.gout = (ph == P.fz.ns - 1);
    io.src = src; io.dst = dst; io.pin = pin; io.nxh = P.nxh; io.nzh = P.nzh; io.nz = P.nz; io.mz = P.mz; io.p0 = p0;
    io.tcount = (pin - p0 < T) ? pin - p0 : T;
    io.filt = filt; io.kxc = kxc; io.kzc = kzc; io.scale = scale;
    zpass_any<false, true>(io, io, P.fz.st[P.fz.ns - 1 - ph], P.mz, T, tid, nt);
}

// Kernels.  k_z*_g: any stage list (run-time radix switch; correct for every 2^a 3^b length but the
// compiler keeps the registers of all radices alive).  k_z*_s<R0..R3>: the same phases with the stage
// radices as template parameters (R = 1: absent) -- the plans chan_api.cu dispatches to.
// plane j of an output field of the forward z pass: full field (filt 0), filtered complex128 (1) or complex64 (2)
CHAN_HD double2* zfwd_plane(const PlaneParams& P, double2* f, int j, int filt, int kxc, int kzc) {
    const size_t per = (size_t)(2 * kzc + 1) * (kxc + 1);
    if (filt == 0) return f + (size_t)j * P.nm;
    if (filt == 1) return f + (size_t)j * per;
    return reinterpret_cast<double2*>(reinterpret_cast<float2*>(f) + (size_t)j * per);
}
CHAN_HD ZInvIO make_zinv_io(const PlaneParams& P, int T, c2* sm, const double2* src, double2* dst, int p0) {
    ZInvIO io;
    io.sm = sm; io.T = T; io.gin = false; io.gout = false;
    io.src = src; io.dst = dst; io.nxh = P.nxh; io.nzh = P.nzh; io.nz = P.nz; io.mz = P.mz; io.p0 = p0;
    io.tcount = (P.nxh - p0 < T) ? P.nxh - p0 : T;
    return io;
}
CHAN_HD ZFwdIO make_zfwd_io(const PlaneParams& P, int T, c2* sm, const double2* src, double2* dst, int pin, int p0, double scale,
                            int filt, int kxc, int kzc) {
    ZFwdIO io;
    io.sm = sm; io.T = T; io.gin = false; io.gout = false;
    io.src = src; io.dst = dst; io.pin = pin; io.nxh = P.nxh; io.nzh = P.nzh; io.nz = P.nz; io.mz = P.mz; io.p0 = p0;
    io.tcount = (pin - p0 < T) ? pin - p0 : T;
    io.filt = filt; io.kxc = kxc; io.kzc = kzc; io.scale = scale;
    return io;
}

#ifdef __CUDACC__
#define CHAN_ZARGS_INV PlaneParams P, FieldPtrs in, int j0, int npl, double2* __restrict__ zpad, int T
#define CHAN_ZARGS_FWD PlaneParams P, const double2* __restrict__ xh, int pin, int j0, int npl, FieldPtrsW out, double scale, int filt, int kxc, int kzc, int T

__global__ void __launch_bounds__(256, 2) k_zfft_inv_g(CHAN_ZARGS_INV) {
    extern __shared__ double2 smem_raw[];
    c2* sm = reinterpret_cast<c2*>(smem_raw);
    const int p0 = blockIdx.x * T, jc = blockIdx.y, fi = blockIdx.z;
    const double2* src = in.f[fi] + (size_t)(j0 + jc) * P.nm;
    double2* dst = zpad + ((size_t)fi * npl + jc) * (size_t)P.mz * P.nxh;
#pragma unroll 1
    for (int ph = 0; ph < P.fz.ns; ++ph) {
        if (ph) __syncthreads();
        zinv_phase(ph, threadIdx.x, blockDim.x, P, T, sm, src, dst, p0);
    }
}
__global__ void __launch_bounds__(256, 2) k_zfft_fwd_g(CHAN_ZARGS_FWD) {
    extern __shared__ double2 smem_raw[];
    c2* sm = reinterpret_cast<c2*>(smem_raw);
    const int p0 = blockIdx.x * T, jc = blockIdx.y, fi = blockIdx.z;
    const int j = j0 + jc;
    const double2* src = xh + ((size_t)fi * npl + jc) * (size_t)P.mz * pin;
    double2* dst = zfwd_plane(P, out.f[fi], j, filt, kxc, kzc);
#pragma unroll 1
    for (int ph = 0; ph < P.fz.ns; ++ph) {
        if (ph) __syncthreads();
        zfwd_phase(ph, threadIdx.x, blockDim.x, P, T, sm, src, dst, pin, p0, scale, filt, kxc, kzc);
    }
}

// Asynchronous tile fill (cp.async, 16 bytes per copy, L1 bypassed): the stage that used to read global memory into
// registers, one butterfly at a time, exposed one memory latency per butterfly round and was half of the z passes'
// time (ncu source view: 44-58% of its samples on the first use of a loaded value).  Every thread now queues the copies of
// the WHOLE tile into its final shared-memory rows up front -- no registers held, 70-110 KB in flight per CTA -- and the
// first stage runs out of shared memory like the others.
#ifndef CHAN_ZASYNC
#define CHAN_ZASYNC 1
#endif
__device__ __forceinline__ void cp_async16(void* smem, const void* g) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(g) : "memory");
}
// CHAN_ZASYNC == 2 (measured, not the default): the same fill with one bulk copy per ROW PIECE (cp.async.bulk, T x 16
// contiguous bytes, completion counted in bytes on an mbarrier).  UBLKCP is a warp-uniform instruction: the compiler
// serialises the 32 lanes of a warp (ELECT / R2UR loop), and 64-byte pieces are too small to pay for that: K2 53 -> 62 ms,
// K4 30 -> 44 ms on config 5.  A strided tile wants a tensor map (one instruction per 256-row box), not 1-D bulk copies.
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n\tfence.mbarrier_init.release.cluster;" ::"r"(a), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(a), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem, const void* g, unsigned bytes, unsigned long long* bar) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem), a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(d), "l"(g), "r"(bytes), "r"(a) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    unsigned ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory"); }

// Bodies with explicit block coordinates (bx = column tile, jc = plane of the chunk, fi = field), shared by the
// stand-alone kernels below and by the merged plane kernel k_planes_s.
// default columns per z tile for a transform length (the rule of choose_tiling in chan_api.cu): the specialised kernels
// take that T as a literal (TC), so that tile addresses become one base plus immediates; any other T runs with TC = 0
__host__ __device__ constexpr int ztile_default(int mz) { int T = 16; while (T > 1 && (long)mz * T * 16 > 112 * 1024) T >>= 1; return T; }
template <int R0, int R1, int R2, int R3, int TC = 0, int NTC = 0>
__device__ __forceinline__ void zinv_body(const PlaneParams& P, const FieldPtrs& in, int j0, int npl, double2* __restrict__ zpad, int Trt,
                                          double2* smem_raw, int bx, int jc, int fi) {
    const int T = TC > 0 ? TC : Trt;
    constexpr int NS = (R0 > 1) + (R1 > 1) + (R2 > 1) + (R3 > 1);
    const int p0 = bx * T;
    ZInvIO io = make_zinv_io(P, T, reinterpret_cast<c2*>(smem_raw), in.f[fi] + (size_t)(j0 + jc) * P.nm,
                             zpad + ((size_t)fi * npl + jc) * (size_t)P.mz * P.nxh, p0);
    constexpr int M2 = R3, M1 = R2 * R3, M0 = R1 * R2 * R3, mz = R0 * M0;
    io.mz = mz; io.nzh = mz / 3; io.nz = 2 * (mz / 3);      // literals (= P.mz, P.nzh, P.nz of the plan this kernel is dispatched for)
    const int tid = threadIdx.x, nt = NTC > 0 ? NTC : blockDim.x;
    if constexpr (CHAN_ZASYNC && NS > 1) {
        // retained rows s != nzh of the field -> rows e(s) of the tile; columns beyond a ragged tile are zero-filled
        c2* sm = io.sm;
        if constexpr (CHAN_ZASYNC == 2) {
            __shared__ unsigned long long mbar;
            const unsigned rowbytes = (unsigned)io.tcount * 16u;
            if (tid == 0) mbar_init(&mbar, 1);
            __syncthreads();
            if (tid == 0) mbar_arrive_expect_tx(&mbar, (unsigned)(P.nz - 1) * rowbytes);
            for (int sl = tid; sl < P.nz; sl += nt) {
                if (sl == P.nzh) continue;
                const int e = sl < P.nzh ? sl : sl + (mz - P.nz);
                bulk_g2s(sm + e * T, io.src + (size_t)sl * P.nxh + p0, rowbytes, &mbar);
                for (int t = io.tcount; t < T; ++t) sm[e * T + t] = mk(0, 0);
            }
            mbar_wait(&mbar, 0);
        } else {
            // thread = (column t, row r0 + i rs): pointer increments only inside the loops; low band, then high band
            int lgT = 0;
            while ((1 << lgT) < T) ++lgT;
            const int t = tid & (T - 1), r0 = tid >> lgT, rs = nt >> lgT;        // nt is a multiple of 32 >= T
            constexpr int nzh_c = mz / 3, nz_c = 2 * (mz / 3);                     // literals, as above
            const bool live = t < io.tcount;
            const double2* g = io.src + (size_t)r0 * P.nxh + p0 + t;
            c2* d = sm + r0 * T + t;
            const size_t gs = (size_t)rs * P.nxh;
            const int ds = rs * T;
#pragma unroll 4
            for (int sl = r0; sl < nzh_c; sl += rs, g += gs, d += ds) { if (live) cp_async16(d, g); else *d = mk(0, 0); }
            g = io.src + (size_t)(nzh_c + 1 + r0) * P.nxh + p0 + t;
            d = sm + (nzh_c + 1 + r0 + (mz - nz_c)) * T + t;
#pragma unroll 4
            for (int sl = nzh_c + 1 + r0; sl < nz_c; sl += rs, g += gs, d += ds) { if (live) cp_async16(d, g); else *d = mk(0, 0); }
            cp_async_wait_all();
        }
        __syncthreads();
        io.gin = false; io.gout = false; io.zband = true;
        zpass<R0, true, false, M0>(io, io, P.fz.st[0], mz, T, tid, nt);
        io.zband = false;
    } else {
        io.gin = true; io.gout = (NS == 1);
        zprefetch<R0, M0>(io, mz, T, tid, nt);
        zpass<R0, true, false, M0>(io, io, P.fz.st[0], mz, T, tid, nt);
    }
    if constexpr (NS > 1) {
        __syncthreads();
        io.gin = false; io.gout = (NS == 2);
        zpass<R1, true, false, M1>(io, io, P.fz.st[1], mz, T, tid, nt);
    }
    if constexpr (NS > 2) {
        __syncthreads();
        io.gout = (NS == 3);
        zpass<R2, true, false, M2>(io, io, P.fz.st[2], mz, T, tid, nt);
    }
    if constexpr (NS > 3) {
        __syncthreads();
        io.gout = true;
        zpass<R3, true, false, 1>(io, io, P.fz.st[3], mz, T, tid, nt);
    }
}
template <int R0, int R1, int R2, int R3, int TC = 0, int NTC = 0>
__device__ __forceinline__ void zfwd_body(const PlaneParams& P, const double2* __restrict__ xh, int pin, int j0, int npl, const FieldPtrsW& out,
                                          double scale, int filt, int kxc, int kzc, int Trt, double2* smem_raw, int bx, int jc, int fi) {
    const int T = TC > 0 ? TC : Trt;
    constexpr int NS = (R0 > 1) + (R1 > 1) + (R2 > 1) + (R3 > 1);
    const int p0 = bx * T;
    const int j = j0 + jc;
    ZFwdIO io = make_zfwd_io(P, T, reinterpret_cast<c2*>(smem_raw), xh + ((size_t)fi * npl + jc) * (size_t)P.mz * pin,
                             zfwd_plane(P, out.f[fi], j, filt, kxc, kzc), pin, p0, scale, filt, kxc, kzc);
    constexpr int M2 = R3, M1 = R2 * R3, M0 = R1 * R2 * R3, mz = R0 * M0;
    io.mz = mz; io.nzh = mz / 3; io.nz = 2 * (mz / 3);      // = P.mz, P.nzh, P.nz of the plan this kernel is dispatched for, as literals
    const int tid = threadIdx.x, nt = NTC > 0 ? NTC : blockDim.x;
    io.gin = true;
    if constexpr (CHAN_ZASYNC && NS > 1) {
        c2* sm = io.sm;
        if constexpr (CHAN_ZASYNC == 2) {
            __shared__ unsigned long long mbar;
            const unsigned rowbytes = (unsigned)io.tcount * 16u;
            if (tid == 0) mbar_init(&mbar, 1);
            __syncthreads();
            if (tid == 0) mbar_arrive_expect_tx(&mbar, (unsigned)mz * rowbytes);
            for (int e = tid; e < mz; e += nt) {
                bulk_g2s(sm + e * T, io.src + (size_t)e * pin + p0, rowbytes, &mbar);
                for (int t = io.tcount; t < T; ++t) sm[e * T + t] = mk(0, 0);
            }
            mbar_wait(&mbar, 0);
        } else {
            int lgT = 0;
            while ((1 << lgT) < T) ++lgT;
            const int t = tid & (T - 1), r0 = tid >> lgT, rs = nt >> lgT;
            const bool live = t < io.tcount;
            const double2* g = io.src + (size_t)r0 * pin + p0 + t;
            c2* d = sm + r0 * T + t;
            const size_t gs = (size_t)rs * pin;
            const int ds = rs * T;
#pragma unroll 4
            for (int e = r0; e < mz; e += rs, g += gs, d += ds) { if (live) cp_async16(d, g); else *d = mk(0, 0); }
            cp_async_wait_all();
        }
        __syncthreads();
        io.gin = false;
    } else if constexpr (NS > 3) zprefetch<R3, 1>(io, mz, T, tid, nt);
    else if constexpr (NS > 2) zprefetch<R2, M2>(io, mz, T, tid, nt);
    else if constexpr (NS > 1) zprefetch<R1, M1>(io, mz, T, tid, nt);
    else zprefetch<R0, M0>(io, mz, T, tid, nt);
    if constexpr (NS > 3) {
        zpass<R3, false, true, 1>(io, io, P.fz.st[3], mz, T, tid, nt);
        __syncthreads();
        io.gin = false;
    }
    if constexpr (NS > 2) {
        zpass<R2, false, true, M2>(io, io, P.fz.st[2], mz, T, tid, nt);
        __syncthreads();
        io.gin = false;
    }
    if constexpr (NS > 1) {
        zpass<R1, false, true, M1>(io, io, P.fz.st[1], mz, T, tid, nt);
        __syncthreads();
        io.gin = false;
    }
    io.gout = true;
    zpass<R0, false, true, M0>(io, io, P.fz.st[0], mz, T, tid, nt);
}
template <int R0, int R1, int R2, int R3>
__global__ void __launch_bounds__(256, 2) k_zfft_inv_s(CHAN_ZARGS_INV) {
    extern __shared__ double2 smem_raw[];
    constexpr int TD = ztile_default(R0 * R1 * R2 * R3);
    if (T == TD && blockDim.x == 192) zinv_body<R0, R1, R2, R3, TD, 192>(P, in, j0, npl, zpad, T, smem_raw, blockIdx.x, blockIdx.y, blockIdx.z);
    else if (T == TD) zinv_body<R0, R1, R2, R3, TD>(P, in, j0, npl, zpad, T, smem_raw, blockIdx.x, blockIdx.y, blockIdx.z);
    else zinv_body<R0, R1, R2, R3>(P, in, j0, npl, zpad, T, smem_raw, blockIdx.x, blockIdx.y, blockIdx.z);
}
template <int R0, int R1, int R2, int R3>
__global__ void __launch_bounds__(256, 2) k_zfft_fwd_s(CHAN_ZARGS_FWD) {
    extern __shared__ double2 smem_raw[];
    // filt as a literal on the hot path (a3-a8 of every substep): the filter branches of the truncating store fold away
    constexpr int TD = ztile_default(R0 * R1 * R2 * R3);
    if (filt == 0 && T == TD && blockDim.x == 192) zfwd_body<R0, R1, R2, R3, TD, 192>(P, xh, pin, j0, npl, out, scale, 0, 0, 0, T, smem_raw, blockIdx.x, blockIdx.y, blockIdx.z);
    else if (filt == 0 && T == TD) zfwd_body<R0, R1, R2, R3, TD>(P, xh, pin, j0, npl, out, scale, 0, 0, 0, T, smem_raw, blockIdx.x, blockIdx.y, blockIdx.z);
    else if (filt == 0) zfwd_body<R0, R1, R2, R3>(P, xh, pin, j0, npl, out, scale, 0, 0, 0, T, smem_raw, blockIdx.x, blockIdx.y, blockIdx.z);
    else zfwd_body<R0, R1, R2, R3>(P, xh, pin, j0, npl, out, scale, filt, kxc, kzc, T, smem_raw, blockIdx.x, blockIdx.y, blockIdx.z);
}
#endif

// ---- 2-CTA cluster variants of the z passes ------------------------------------------------------------------------
// Where a tile of 8 columns (128-byte row pieces) does not fit the shared memory that lets two CTAs share an SM
// (config 5: 1728 rows x 8 columns x 16 B = 221 KB), the tile is split BY ROWS between the two CTAs of a thread-block
// cluster: rank r keeps rows [r n/2, (r+1) n/2).  Only the stage with the longest stride (R0, sub-block M0 = n/R0) couples
// the halves: its butterfly p + k M0, k < R0, has R0/2 elements in each half (R0 even), so that stage is split by
// butterflies and half of its shared-memory traffic goes through distributed shared memory; every other stage works on
// blocks of M0 rows that lie inside one half.  Inverse (DIF): the coupling stage is the first one (reads global memory,
// writes both halves), then a cluster barrier.  Forward (DIT): it is the last one (reads both halves, writes global
// memory), between two cluster barriers (the partner's shared memory must outlive the reads).
struct ZInvIOc {
    ZInvIO b; c2* smr; int eoff, nh;            // partner's half, first row of this half, rows per half
    CHAN_HD c2 load(int e, int t) const { return b.gin ? b.load(e, t) : b.sm[(e - eoff) * b.T + t]; }
    CHAN_HD void store(int e, int t, c2 v) const {
        if (b.gout) { b.store(e, t, v); return; }
        const int el = e - eoff;
        if ((unsigned)el < (unsigned)nh) b.sm[el * b.T + t] = v; else smr[(el < 0 ? el + nh : el - nh) * b.T + t] = v;
    }
};
struct ZFwdIOc {
    ZFwdIO b; const c2* smr; int eoff, nh;
    CHAN_HD c2 load(int e, int t) const {
        if (b.gin) return b.load(e, t);
        const int el = e - eoff;
        return ((unsigned)el < (unsigned)nh) ? b.sm[el * b.T + t] : smr[(el < 0 ? el + nh : el - nh) * b.T + t];
    }
    CHAN_HD void store(int e, int t, c2 v) const { if (b.gout) b.store(e, t, v); else b.sm[(e - eoff) * b.T + t] = v; }
};

#ifdef __CUDACC__
}  // namespace chn
#include <cooperative_groups.h>
namespace chn {
template <int R0, int R1, int R2, int R3>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(256, 2) k_zfft_inv_c(CHAN_ZARGS_INV) {
    extern __shared__ double2 smem_raw[];
    namespace cg = cooperative_groups;
    constexpr int NS = (R0 > 1) + (R1 > 1) + (R2 > 1) + (R3 > 1);
    static_assert(NS >= 2 && R0 % 2 == 0 && (R1 * R2 * R3) % 2 == 0, "the cluster split needs an even first radix, an even sub-block and a second stage");
    cg::cluster_group cl = cg::this_cluster();
    const int rank = (int)cl.block_rank();
    const int p0 = (int)(blockIdx.x >> 1) * T, jc = blockIdx.y, fi = blockIdx.z;
    constexpr int M2 = R3, M1 = R2 * R3, M0 = R1 * R2 * R3, mz = R0 * M0;
    ZInvIOc io;
    io.b = make_zinv_io(P, T, reinterpret_cast<c2*>(smem_raw), in.f[fi] + (size_t)(j0 + jc) * P.nm,
                        zpad + ((size_t)fi * npl + jc) * (size_t)P.mz * P.nxh, p0);
    io.smr = reinterpret_cast<c2*>(cl.map_shared_rank(smem_raw, rank ^ 1));
    io.nh = mz / 2; io.eoff = rank * io.nh;
    const int tid = threadIdx.x, nt = blockDim.x;
    io.b.gin = true; io.b.gout = false;
    zpass<R0, true, false, M0>(io, io, P.fz.st[0], mz, T, tid, nt, rank);
    cl.sync();
    io.b.gin = false; io.b.gout = (NS == 2);
    zpass<R1, true, false, M1>(io, io, P.fz.st[1], mz, T, tid, nt, rank);
    if constexpr (NS > 2) {
        __syncthreads();
        io.b.gout = (NS == 3);
        zpass<R2, true, false, M2>(io, io, P.fz.st[2], mz, T, tid, nt, rank);
    }
    if constexpr (NS > 3) {
        __syncthreads();
        io.b.gout = true;
        zpass<R3, true, false, 1>(io, io, P.fz.st[3], mz, T, tid, nt, rank);
    }
}
template <int R0, int R1, int R2, int R3>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(256, 2) k_zfft_fwd_c(CHAN_ZARGS_FWD) {
    extern __shared__ double2 smem_raw[];
    namespace cg = cooperative_groups;
    constexpr int NS = (R0 > 1) + (R1 > 1) + (R2 > 1) + (R3 > 1);
    static_assert(NS >= 2 && R0 % 2 == 0 && (R1 * R2 * R3) % 2 == 0, "the cluster split needs an even first radix, an even sub-block and a second stage");
    cg::cluster_group cl = cg::this_cluster();
    const int rank = (int)cl.block_rank();
    const int p0 = (int)(blockIdx.x >> 1) * T, jc = blockIdx.y, fi = blockIdx.z;
    const int j = j0 + jc;
    constexpr int M2 = R3, M1 = R2 * R3, M0 = R1 * R2 * R3, mz = R0 * M0;
    ZFwdIOc io;
    io.b = make_zfwd_io(P, T, reinterpret_cast<c2*>(smem_raw), xh + ((size_t)fi * npl + jc) * (size_t)P.mz * pin,
                        zfwd_plane(P, out.f[fi], j, filt, kxc, kzc), pin, p0, scale, filt, kxc, kzc);
    io.smr = reinterpret_cast<const c2*>(cl.map_shared_rank(smem_raw, rank ^ 1));
    io.nh = mz / 2; io.eoff = rank * io.nh;
    const int tid = threadIdx.x, nt = blockDim.x;
    io.b.gin = true; io.b.gout = false;
    if constexpr (NS > 3) {
        zpass<R3, false, true, 1>(io, io, P.fz.st[3], mz, T, tid, nt, rank);
        __syncthreads();
        io.b.gin = false;
    }
    if constexpr (NS > 2) {
        zpass<R2, false, true, M2>(io, io, P.fz.st[2], mz, T, tid, nt, rank);
        __syncthreads();
        io.b.gin = false;
    }
    zpass<R1, false, true, M1>(io, io, P.fz.st[1], mz, T, tid, nt, rank);
    io.b.gin = false;
    cl.sync();
    io.b.gout = true;
    zpass<R0, false, true, M0>(io, io, P.fz.st[0], mz, T, tid, nt, rank);
    cl.sync();
}
#endif

// =====================================================================================================
// x transforms (K3, a4-a6): one (plane, z) row per CTA.  Six spectral rows are packed into three complex
// sequences (A + iB with A, B Hermitian), inverse transformed, multiplied pointwise, and the products go
// back as packed forward transforms.  Shared layout [sequence][swz(e)] with
// swz(e) = e ^ ((e >> 3) & 7): contiguous runs of 8, stride-4 and stride-8 butterflies are all free of
// bank conflicts for 16-byte elements.  One thread owns butterfly b of EVERY sequence, so the twiddles
// are loaded once per butterfly and reused.
//   NPROD = 3: H = u x omega (reading R1).   NPROD = 7: uu,uv,uw,vv,vw,ww, om.om (filter, R12).
// zpad fields in order u,v,w,om_x,om_y,om_z.
// =====================================================================================================
CHAN_HD int swz(int e) { return e ^ ((e >> 3) & 7); }
struct XIO {
    c2* sm; int stride;
    // zero band of the 3/2 padding, entries blo..bhi: never written by the pack (zin: read as zero by the first
    // inverse stage) and never needed by the unpack (zout: not written by the last forward stage)
    int blo = 0, bhi = -1; bool zin = false, zout = false;
    CHAN_HD c2 load(int e, int q) const { return (zin && e >= blo && e <= bhi) ? mk(0, 0) : sm[q * stride + swz(e)]; }
    CHAN_HD void store(int e, int q, c2 v) const { if (!(zout && e >= blo && e <= bhi)) sm[q * stride + swz(e)] = v; }
};
template <int R, bool INV, bool DIT, int M = 0>
CHAN_HD void xpass(const XIO& io, const FftStage& S, int n, int nseq, int tid, int nt) {
    const int m = M > 0 ? M : S.m, ncur = R * m, nb = n / R;
    if constexpr (R > 12) {
        // radix 16, 18: a row has fewer butterflies than the CTA has threads, and 2R doubles of butterfly data leave no
        // room to interleave sequences: work item = (sequence, butterfly), one sequence at a time per thread
        const int total = nb * nseq;
#pragma unroll 1
        for (int w = tid; w < total; w += nt) {
            const int q = w / nb, b = w - q * nb;
            const int blk = b / m, p = b - blk * m;
            CHAN_ASSUME(p >= 0 && p < m && blk >= 0);      // known bits: the swizzle of base + k m then folds per k
            c2 tw[R - 1];
            if (m > 1) load_twiddles<R>(S, m, p, tw);
            pass_item<R, INV, DIT>(io, io, q, blk * ncur + p, m, tw, m > 1);
        }
    } else {
        for (int b = tid; b < nb; b += nt) {
            const int blk = b / m, p = b - blk * m;
            c2 tw[R - 1 > 0 ? R - 1 : 1];
            if (m > 1) load_twiddles<R>(S, m, p, tw);
            for (int q = 0; q < nseq; ++q) pass_item<R, INV, DIT>(io, io, q, blk * ncur + p, m, tw, m > 1);
        }
    }
}
template <bool INV, bool DIT>
CHAN_HD void xpass_any(const XIO& io, const FftStage& S, int n, int nseq, int tid, int nt) {
    switch (S.R) {
        case 2: xpass<2, INV, DIT>(io, S, n, nseq, tid, nt); break;
        case 3: xpass<3, INV, DIT>(io, S, n, nseq, tid, nt); break;
        case 4: xpass<4, INV, DIT>(io, S, n, nseq, tid, nt); break;
        case 6: xpass<6, INV, DIT>(io, S, n, nseq, tid, nt); break;
        case 8: xpass<8, INV, DIT>(io, S, n, nseq, tid, nt); break;
        case 16: xpass<16, INV, DIT>(io, S, n, nseq, tid, nt); break;
        case 18: xpass<18, INV, DIT>(io, S, n, nseq, tid, nt); break;
        default: xpass<12, INV, DIT>(io, S, n, nseq, tid, nt); break;
    }
}

// last inverse stage (radix F, m = 1, no twiddles) + products + first forward stage, in registers
template <int F, int NPROD>
CHAN_HD void xfused(const XIO& io, int n, int tid, int nt) {
    for (int b = tid; b < n / F; b += nt) {
        CHAN_ASSUME(b >= 0);
        c2 s0[F], s1[F], s2[F];
#pragma unroll
        for (int k = 0; k < F; ++k) { s0[k] = io.load(F * b + k, 0); s1[k] = io.load(F * b + k, 1); s2[k] = io.load(F * b + k, 2); }
        bfly<F, true>(s0); bfly<F, true>(s1); bfly<F, true>(s2);
        // s0 = u + i v, s1 = w + i om_x, s2 = om_y + i om_z at F physical points
        if constexpr (NPROD == 3) {
            c2 o[F];
#pragma unroll
            for (int k = 0; k < F; ++k) o[k] = mk(s0[k].y * s2[k].y - s1[k].x * s2[k].x, s1[k].x * s1[k].y - s0[k].x * s2[k].y);
            bfly<F, false>(o);
#pragma unroll
            for (int k = 0; k < F; ++k) io.store(F * b + k, 0, o[k]);
#pragma unroll
            for (int k = 0; k < F; ++k) o[k] = mk(s0[k].x * s2[k].x - s0[k].y * s1[k].y, 0.0);
            bfly<F, false>(o);
#pragma unroll
            for (int k = 0; k < F; ++k) io.store(F * b + k, 1, o[k]);
        } else {
            c2 o[F];
#pragma unroll
            for (int k = 0; k < F; ++k) o[k] = mk(s0[k].x * s0[k].x, s0[k].x * s0[k].y);
            bfly<F, false>(o);
#pragma unroll
            for (int k = 0; k < F; ++k) io.store(F * b + k, 0, o[k]);
#pragma unroll
            for (int k = 0; k < F; ++k) o[k] = mk(s0[k].x * s1[k].x, s0[k].y * s0[k].y);
            bfly<F, false>(o);
#pragma unroll
            for (int k = 0; k < F; ++k) io.store(F * b + k, 1, o[k]);
#pragma unroll
            for (int k = 0; k < F; ++k) o[k] = mk(s0[k].y * s1[k].x, s1[k].x * s1[k].x);
            bfly<F, false>(o);
#pragma unroll
            for (int k = 0; k < F; ++k) io.store(F * b + k, 2, o[k]);
#pragma unroll
            for (int k = 0; k < F; ++k) o[k] = mk(s1[k].y * s1[k].y + s2[k].x * s2[k].x + s2[k].y * s2[k].y, 0.0);
            bfly<F, false>(o);
#pragma unroll
            for (int k = 0; k < F; ++k) io.store(F * b + k, 3, o[k]);
        }
    }
}

CHAN_HD void xpack(const XIO& io, int mx, int nxh, const double2* zrow, size_t fstride, int tid, int nt, bool fill_zero) {
    // C[k] = A[k] + i B[k], C[mx-k] = conj(A[k]) + i conj(B[k]); Im of the k = 0 entries dropped (R14).
    // A thread owns columns k = tid + i nt of all three pairs: no index division, and the global loads of XK columns
    // (6 XK loads of 16 bytes) are issued before the first shared-memory store -- the pack was 29% of the x pass
    // (ncu source view), most of it waiting on two or three rounds of loads and on integer divisions.
    constexpr int XK = 3;
    for (int k0 = tid; k0 < nxh; k0 += nt * XK) {
        c2 A[XK][3], B[XK][3];
#pragma unroll
        for (int i = 0; i < XK; ++i) {
            const int k = k0 + i * nt;
            if (k < nxh) {
#pragma unroll
                for (int pr = 0; pr < 3; ++pr) {
                    A[i][pr] = ldstream(zrow + (size_t)(2 * pr) * fstride + k); B[i][pr] = ldstream(zrow + (size_t)(2 * pr + 1) * fstride + k);
                }
            }
        }
#pragma unroll
        for (int i = 0; i < XK; ++i) {
            const int k = k0 + i * nt;
            if (k < nxh) {
#pragma unroll
                for (int pr = 0; pr < 3; ++pr) {
                    const c2 a = A[i][pr], b = B[i][pr];
                    if (k == 0) io.store(0, pr, mk(a.x, b.x));
                    else { io.store(k, pr, mk(a.x - b.y, a.y + b.x)); io.store(mx - k, pr, mk(a.x + b.y, -a.y + b.x)); }
                }
            }
        }
    }
    const int nzero = fill_zero ? mx - 2 * nxh + 1 : 0;     // entries nxh .. mx-nxh (else the first stage reads them as zero)
    for (int w = tid; w < 3 * nzero; w += nt) {
        const int pr = w / nzero, k = w - pr * nzero;
        io.store(nxh + k, pr, mk(0, 0));
    }
}
template <int NPROD>
CHAN_HD void xunpack(const XIO& io, int mx, double2* xrow, size_t ostride, int pout, int tid, int nt) {
    constexpr int NC = (NPROD + 1) / 2;
    // A[k] = (D[k] + conj D[mx-k])/2, B[k] = (D[k] - conj D[mx-k])/(2i)
    for (int k = tid; k < pout; k += nt) {
#pragma unroll
        for (int pr = 0; pr < NC; ++pr) {
            const c2 d = io.load(k, pr), e = io.load(k == 0 ? 0 : mx - k, pr);
            ststream(xrow + (size_t)(2 * pr) * ostride + k, mk(0.5 * (d.x + e.x), 0.5 * (d.y - e.y)));
            if (2 * pr + 1 < NPROD) ststream(xrow + (size_t)(2 * pr + 1) * ostride + k, mk(0.5 * (d.y + e.y), -0.5 * (d.x - e.x)));
        }
    }
}

// Phases of one row: 0 pack | 1..ns-1 inverse stages 0..ns-2 | ns fused | ns+1..2ns-1 forward stages
// ns-2..0 | 2ns unpack.   zrow: row (jc, r) of the six zpad fields (field stride fstride);
// xrow: row of the NPROD xh fields (field stride ostride, row pitch pout).
template <int NPROD, int F>
CHAN_HD void xrow_phase(int ph, int tid, int nt, const PlaneParams& P, c2* sm, const double2* zrow, size_t fstride,
                        double2* xrow, size_t ostride, int pout) {
    constexpr int NC = (NPROD + 1) / 2;
    const int mx = P.mx, nxh = P.nxh, ns = P.fx.ns;
    XIO io; io.sm = sm; io.stride = mx;
    io.blo = nxh; io.bhi = mx - nxh;
    if (ph == 0) {
        xpack(io, mx, nxh, zrow, fstride, tid, nt, ns == 1);
    } else if (ph < ns) {
        io.zin = (ph == 1);
        xpass_any<true, false>(io, P.fx.st[ph - 1], mx, 3, tid, nt);
    } else if (ph == ns) {
        xfused<F, NPROD>(io, mx, tid, nt);
    } else if (ph < 2 * ns) {
        io.zout = (ph == 2 * ns - 1);
        xpass_any<false, true>(io, P.fx.st[2 * ns - 1 - ph], mx, NC, tid, nt);
    } else {
        xunpack<NPROD>(io, mx, xrow, ostride, pout, tid, nt);
    }
}

#ifdef __CUDACC__
#define CHAN_XARGS PlaneParams P, const double2* __restrict__ zpad, int npl, double2* __restrict__ xh, int pout

// any stage list (run-time radix switch)
template <int NPROD, int F>
__global__ void __launch_bounds__(256, 2) k_xfft_prod_g(CHAN_XARGS) {
    extern __shared__ double2 smem_raw[];
    c2* sm = reinterpret_cast<c2*>(smem_raw);    // [max(3, NC)][mx]
    const int r = blockIdx.x, jc = blockIdx.y;
    const size_t fstride = (size_t)npl * P.mz * P.nxh;
    const double2* zrow = zpad + ((size_t)jc * P.mz + r) * P.nxh;
    const size_t ostride = (size_t)npl * P.mz * pout;
    double2* xrow = xh + ((size_t)jc * P.mz + r) * pout;
    const int nph = 2 * P.fx.ns + 1;
#pragma unroll 1
    for (int ph = 0; ph < nph; ++ph) {
        if (ph) __syncthreads();
        xrow_phase<NPROD, F>(ph, threadIdx.x, blockDim.x, P, sm, zrow, fstride, xrow, ostride, pout);
    }
}

// stage radices as template parameters: R0, R1, R2 (1 = absent) then the fused radix F
// (the filter variant keeps four sequences in shared memory: where only one such CTA fits on an SM it runs 512 threads)
template <int NPROD, int F, int R0, int R1, int R2, int NTC = 0>
__device__ __forceinline__ void xprod_body(const PlaneParams& P, const double2* __restrict__ zpad, int npl, double2* __restrict__ xh, int pout,
                                           double2* smem_raw, int r, int jc) {
    constexpr int NC = (NPROD + 1) / 2;
    constexpr int M2 = F, M1 = R2 * F, M0 = R1 * R2 * F, mx = R0 * M0;
    const int tid = threadIdx.x, nt = NTC > 0 ? NTC : blockDim.x;      // NTC: the CTA size as a literal (trip counts of the item loops fold)
    XIO io; io.sm = reinterpret_cast<c2*>(smem_raw); io.stride = mx;
    io.blo = mx / 3; io.bhi = mx - mx / 3;
    // P.nxh of the plan this kernel is dispatched for, as a literal in the substep's kernel (the filter variant, at its 128-register
    // cap with a spill, got 5% slower with it and keeps the run-time value)
    const int nxh = NPROD == 3 ? mx / 3 : P.nxh;
    xpack(io, mx, nxh, zpad + ((size_t)jc * P.mz + r) * nxh, (size_t)npl * P.mz * nxh, tid, nt, R0 == 1);
    __syncthreads();
    if constexpr (R0 > 1) { io.zin = true; xpass<R0, true, false, M0>(io, P.fx.st[0], mx, 3, tid, nt); io.zin = false; __syncthreads(); }
    if constexpr (R1 > 1) { xpass<R1, true, false, M1>(io, P.fx.st[1], mx, 3, tid, nt); __syncthreads(); }
    if constexpr (R2 > 1) { xpass<R2, true, false, M2>(io, P.fx.st[2], mx, 3, tid, nt); __syncthreads(); }
    xfused<F, NPROD>(io, mx, tid, nt);
    __syncthreads();
    if constexpr (R2 > 1) { xpass<R2, false, true, M2>(io, P.fx.st[2], mx, NC, tid, nt); __syncthreads(); }
    if constexpr (R1 > 1) { xpass<R1, false, true, M1>(io, P.fx.st[1], mx, NC, tid, nt); __syncthreads(); }
    if constexpr (R0 > 1) { io.zout = true; xpass<R0, false, true, M0>(io, P.fx.st[0], mx, NC, tid, nt); io.zout = false; __syncthreads(); }
    if (NPROD == 3 && pout == nxh) xunpack<NPROD>(io, mx, xh + ((size_t)jc * P.mz + r) * nxh, (size_t)npl * P.mz * nxh, nxh, tid, nt);
    else xunpack<NPROD>(io, mx, xh + ((size_t)jc * P.mz + r) * pout, (size_t)npl * P.mz * pout, pout, tid, nt);
}
#ifndef CHAN_XNT
#define CHAN_XNT 256      // most threads of an x-pass CTA (two CTAs per SM)
#endif
template <int NPROD, int F, int R0, int R1, int R2>
__global__ void __launch_bounds__(NPROD == 7 ? 512 : CHAN_XNT, NPROD == 7 ? 1 : 2) k_xfft_prod_s(CHAN_XARGS) {
    extern __shared__ double2 smem_raw[];
    // (the same for 128-thread CTAs, as configs 3 and 4 run them, was measured 7% slower and is not dispatched)
    if (NPROD == 3 && blockDim.x == 256) xprod_body<NPROD, F, R0, R1, R2, 256>(P, zpad, npl, xh, pout, smem_raw, blockIdx.x, blockIdx.y);
    else xprod_body<NPROD, F, R0, R1, R2>(P, zpad, npl, xh, pout, smem_raw, blockIdx.x, blockIdx.y);
}

// =====================================================================================================
// Merged plane kernel: one launch carries the inverse z pass (K2) of plane chunk t, the x pass with the products
// (K3) of chunk t-1 and the forward z pass (K4) of chunk t-2, whose CTAs are INTERLEAVED in block-index order so
// that every SM hosts a mix of them: K3 is bound by the shared-memory pipe (DRAM ~20% busy), K2 and K4 by memory
// latency (shared-memory pipe half idle); running them side by side on an SM fills both units.  The three parts
// work on different chunk buffers (zpad and xh are double-buffered by the host loop), so a launch has no internal
// dependency; the order of launches on the stream carries the K2 -> K3 -> K4 dependency of each chunk.
// Block b of the merged grid: A-blocks (K3) sit at the positions where floor(b n3/n) steps, the others are
// B-blocks, first the n2 of K2, then the n4 of K4.
// =====================================================================================================
struct MergedArgs {
    // K2: chunk starting at plane j2, npl2 planes, writes zw
    FieldPtrs in; int j2, npl2; double2* zw;
    // K3: reads zr, writes xw, npl3 planes
    const double2* zr; int npl3; double2* xw;
    // K4: reads xr, chunk starting at plane j4, npl4 planes
    const double2* xr; int j4, npl4; FieldPtrsW out; double scale;
    int T;
    unsigned n2, n3, n4;      // blocks of each part (0: part absent from this launch)
    unsigned tiles;           // column tiles per plane of the z passes
};
template <int Z0, int Z1, int Z2, int Z3, int F, int X0, int X1, int X2>
__global__ void __launch_bounds__(256, 2) k_planes_s(PlaneParams P, MergedArgs A) {
    extern __shared__ double2 smem_raw[];
    const unsigned long long n = (unsigned long long)A.n2 + A.n3 + A.n4, b = blockIdx.x;
    const unsigned a0 = (unsigned)(b * A.n3 / n), a1 = (unsigned)((b + 1) * A.n3 / n);
    if (a1 > a0) {                                    // A-block number a0: row r of plane jc
        const int jc = (int)(a0 / (unsigned)P.mz), r = (int)(a0 - (unsigned)jc * P.mz);
        xprod_body<3, F, X0, X1, X2>(P, A.zr, A.npl3, A.xw, P.nxh, smem_raw, r, jc);
        return;
    }
    unsigned ib = (unsigned)(b - a0);                 // B-block number
    if (ib < A.n2) {
        const unsigned per = A.tiles * (unsigned)A.npl2;
        const int fi = (int)(ib / per); ib -= (unsigned)fi * per;
        const int jc = (int)(ib / A.tiles), bx = (int)(ib - (unsigned)jc * A.tiles);
        zinv_body<Z0, Z1, Z2, Z3>(P, A.in, A.j2, A.npl2, A.zw, A.T, smem_raw, bx, jc, fi);
    } else {
        ib -= A.n2;
        const unsigned per = A.tiles * (unsigned)A.npl4;
        const int fi = (int)(ib / per); ib -= (unsigned)fi * per;
        const int jc = (int)(ib / A.tiles), bx = (int)(ib - (unsigned)jc * A.tiles);
        zfwd_body<Z0, Z1, Z2, Z3>(P, A.xr, P.nxh, A.j4, A.npl4, A.out, A.scale, 0, 0, 0, A.T, smem_raw, bx, jc, fi);
    }
}
#endif

}  // namespace chn
