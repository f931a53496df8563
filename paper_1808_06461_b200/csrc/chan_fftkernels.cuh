// Wall-parallel (x,z) phase: batched plane FFTs with 3/2-rule zero padding, the pointwise products in
// physical space, truncation, and the filter / statistics reductions.  Steps a3-a8, a13, a14 of
// DESIGN.md; PAPER.md L80 ("pseudo-spectral ... fully dealiased by zero padding"), L84, L124.
//
// All transforms run in shared memory, in place, mixed radix {4,2,3}:
//   spectral -> physical:  decimation in frequency (natural order in, digit-reversed order out),
//   physical -> spectral:  decimation in time with the same radix plan backwards (digit-reversed in,
//                          natural out).
// Physical space is only ever used pointwise, so the digit-reversed order is never undone.
#pragma once
#include <cuda_runtime.h>

#include "chan_ykernels.cuh"

namespace chn {

#define CHAN_MAX_RADIX_PASSES 16

struct FftDev {
    int n;
    int npass;
    int radix[CHAN_MAX_RADIX_PASSES];
    const double2* tw;     // n twiddles exp(-2 pi i k/n)
};

template <int R, bool INV> __device__ __forceinline__ void bfly(c2 (&a)[R]);
template <> __device__ __forceinline__ void bfly<2, false>(c2 (&a)[2]) { c2 t = a[0] - a[1]; a[0] = a[0] + a[1]; a[1] = t; }
template <> __device__ __forceinline__ void bfly<2, true>(c2 (&a)[2]) { c2 t = a[0] - a[1]; a[0] = a[0] + a[1]; a[1] = t; }
template <bool INV> __device__ __forceinline__ void bfly4(c2 (&a)[4]) {
    c2 s0 = a[0] + a[2], d0 = a[0] - a[2], s1 = a[1] + a[3], d1 = a[1] - a[3];
    // forward: -i*d1 ; inverse: +i*d1
    c2 jd = INV ? mk(-d1.y, d1.x) : mk(d1.y, -d1.x);
    a[0] = s0 + s1; a[2] = s0 - s1; a[1] = d0 + jd; a[3] = d0 - jd;
}
template <> __device__ __forceinline__ void bfly<4, false>(c2 (&a)[4]) { bfly4<false>(a); }
template <> __device__ __forceinline__ void bfly<4, true>(c2 (&a)[4]) { bfly4<true>(a); }
template <bool INV> __device__ __forceinline__ void bfly3(c2 (&a)[3]) {
    const double s = 0.86602540378443864676;  // sin(pi/3)
    c2 t = a[1] + a[2], d = a[1] - a[2];
    c2 m = mk(a[0].x - 0.5 * t.x, a[0].y - 0.5 * t.y);
    // forward: w = exp(-2 pi i/3): b1 = m - i s d ; inverse: b1 = m + i s d
    c2 jd = INV ? mk(-s * d.y, s * d.x) : mk(s * d.y, -s * d.x);
    a[0] = a[0] + t; a[1] = m + jd; a[2] = m - jd;
}
template <> __device__ __forceinline__ void bfly<3, false>(c2 (&a)[3]) { bfly3<false>(a); }
template <> __device__ __forceinline__ void bfly<3, true>(c2 (&a)[3]) { bfly3<true>(a); }

__device__ __forceinline__ c2 twiddle(const double2* tw, int idx, bool inv) {
    double2 w = __ldg(tw + idx);
    return mk(w.x, inv ? -w.y : w.y);
}

// One in-place pass over `nseq` sequences of length n stored as data[e*es + q*ss] (e element, q sequence).
// DIF: butterfly then twiddle on the outputs; DIT: twiddle on the inputs then butterfly.
// ncur = size of the sub-blocks being split (DIF) / assembled (DIT); m = ncur/R.
template <int R, bool INV, bool DIT, bool SEQ_FAST>
__device__ __forceinline__ void fft_pass(c2* data, int n, int nseq, int es, int ss, int ncur, const double2* tw) {
    const int m = ncur / R;
    const int nb = n / R;                 // butterflies per sequence
    const int tws = n / ncur;             // twiddle stride
    const int total = nb * nseq;
    for (int w = threadIdx.x; w < total; w += blockDim.x) {
        int q, b;
        if (SEQ_FAST) { q = w % nseq; b = w / nseq; } else { q = w / nb; b = w - q * nb; }
        const int blk = b / m, p = b - blk * m;
        c2* base = data + (size_t)q * ss + (size_t)(blk * ncur + p) * es;
        c2 a[R];
#pragma unroll
        for (int k = 0; k < R; ++k) a[k] = base[(size_t)k * m * es];
        if (DIT) {
#pragma unroll
            for (int k = 1; k < R; ++k) a[k] = cmul(a[k], twiddle(tw, p * k * tws, INV));
        }
        bfly<R, INV>(a);
        if (!DIT) {
#pragma unroll
            for (int k = 1; k < R; ++k) a[k] = cmul(a[k], twiddle(tw, p * k * tws, INV));
        }
#pragma unroll
        for (int k = 0; k < R; ++k) base[(size_t)k * m * es] = a[k];
    }
}

// Full transform. INV=true,DIT=false : spectral->physical (unnormalised, e^{+i}); INV=false,DIT=true: physical->spectral.
template <bool INV, bool DIT, bool SEQ_FAST>
__device__ __forceinline__ void fft_inplace(c2* data, const FftDev& F, int nseq, int es, int ss) {
    if (!DIT) {
        int ncur = F.n;
        for (int ps = 0; ps < F.npass; ++ps) {
            const int R = F.radix[ps];
            if (R == 4) fft_pass<4, INV, false, SEQ_FAST>(data, F.n, nseq, es, ss, ncur, F.tw);
            else if (R == 2) fft_pass<2, INV, false, SEQ_FAST>(data, F.n, nseq, es, ss, ncur, F.tw);
            else fft_pass<3, INV, false, SEQ_FAST>(data, F.n, nseq, es, ss, ncur, F.tw);
            ncur /= R;
            __syncthreads();
        }
    } else {
        int ncur = 1;
        for (int ps = F.npass - 1; ps >= 0; --ps) {
            const int R = F.radix[ps];
            ncur *= R;
            if (R == 4) fft_pass<4, INV, true, SEQ_FAST>(data, F.n, nseq, es, ss, ncur, F.tw);
            else if (R == 2) fft_pass<2, INV, true, SEQ_FAST>(data, F.n, nseq, es, ss, ncur, F.tw);
            else fft_pass<3, INV, true, SEQ_FAST>(data, F.n, nseq, es, ss, ncur, F.tw);
            __syncthreads();
        }
    }
}

struct PlaneParams {
    int ny, nz, nxh, nzh, mx, mz;
    long long nm;          // nz*nxh
    FftDev fx, fz;
};

// =====================================================================================================
// K2 (a3): zero-pad in k_z and inverse c2c FFT along z for a tile of T k_x columns.
// grid = (nxh/T tiles, planes in chunk, fields); in: plane-layout field, out: zpad[f][jc][r][p].
// =====================================================================================================
struct FieldPtrs { const double2* f[8]; };

template <int T>
__global__ void __launch_bounds__(256) k_zfft_inv(PlaneParams P, FieldPtrs in, int j0, int npl, double2* __restrict__ zpad) {
    extern __shared__ double2 smem_raw[];
    c2* data = reinterpret_cast<c2*>(smem_raw);       // [mz][T]
    const int p0 = blockIdx.x * T, jc = blockIdx.y, fi = blockIdx.z;
    const int j = j0 + jc;
    const double2* src = in.f[fi] + (size_t)j * P.nm;
    const int nzh = P.nzh, mz = P.mz, nz = P.nz;
    const int tcount = min(T, P.nxh - p0);
    for (int w = threadIdx.x; w < mz * T; w += blockDim.x) {
        const int r = w / T, t = w - r * T;
        c2 v = mk(0, 0);
        int s = -1;
        if (r < nzh) s = r; else if (r > mz - nzh) s = r - (mz - nz);
        if (s >= 0 && t < tcount) v = ldc(src + (size_t)s * P.nxh + p0 + t);
        data[w] = v;
    }
    __syncthreads();
    fft_inplace<true, false, true>(data, P.fz, T, T, 1);
    double2* dst = zpad + ((size_t)fi * npl + jc) * (size_t)mz * P.nxh;
    for (int w = threadIdx.x; w < mz * T; w += blockDim.x) {
        const int r = w / T, t = w - r * T;
        if (t < tcount) stc(dst + (size_t)r * P.nxh + p0 + t, data[w]);
    }
}

// =====================================================================================================
// K4 (a7-a8): forward c2c FFT along z, truncate to the kept z modes, scale, store.
//   mode 0: store retained modes into plane-layout fields out.f[fi] (Nyquist slot zeroed), all p < nxh.
//   mode 1: filter: store |q| <= kzc, p <= kxc into out.f[fi][j][2kzc+1][kxc+1].
// in: xh[fi][jc][r][pin], pin = row pitch of xh (nxh, or kxc+1 for the filter).
// =====================================================================================================
struct FieldPtrsW { double2* f[8]; };

template <int T>
__global__ void __launch_bounds__(256) k_zfft_fwd(PlaneParams P, const double2* __restrict__ xh, int pin, int j0, int npl,
                                                  FieldPtrsW out, double scale, int filt, int kxc, int kzc) {
    extern __shared__ double2 smem_raw[];
    c2* data = reinterpret_cast<c2*>(smem_raw);
    const int p0 = blockIdx.x * T, jc = blockIdx.y, fi = blockIdx.z;
    const int j = j0 + jc;
    const int nzh = P.nzh, mz = P.mz, nz = P.nz;
    const int tcount = min(T, pin - p0);
    const double2* src = xh + ((size_t)fi * npl + jc) * (size_t)mz * pin;
    for (int w = threadIdx.x; w < mz * T; w += blockDim.x) {
        const int r = w / T, t = w - r * T;
        data[w] = (t < tcount) ? ldc(src + (size_t)r * pin + p0 + t) : mk(0, 0);
    }
    __syncthreads();
    fft_inplace<false, true, true>(data, P.fz, T, T, 1);
    if (!filt) {
        double2* dst = out.f[fi] + (size_t)j * P.nm;
        for (int w = threadIdx.x; w < nz * T; w += blockDim.x) {
            const int s = w / T, t = w - s * T;
            if (t >= tcount) continue;
            c2 v = mk(0, 0);
            if (s != nzh) { const int r = (s < nzh) ? s : s + (mz - nz); v = data[r * T + t]; v = mk(v.x * scale, v.y * scale); }
            stc(dst + (size_t)s * P.nxh + p0 + t, v);
        }
    } else {
        const int nr = 2 * kzc + 1, npk = kxc + 1;
        double2* dst = out.f[fi] + (size_t)j * nr * npk;
        for (int w = threadIdx.x; w < nr * T; w += blockDim.x) {
            const int rr = w / T, t = w - rr * T;
            if (t >= tcount || p0 + t >= npk) continue;
            const int r = (rr <= kzc) ? rr : mz - (nr - rr);   // rr = kzc+1.. -> q = -kzc..-1
            c2 v = data[r * T + t];
            stc(dst + (size_t)rr * npk + p0 + t, mk(v.x * scale, v.y * scale));
        }
    }
}

// =====================================================================================================
// K3 (a4-a6): one (plane, z) row per CTA.  Six spectral rows -> three packed complex sequences
// (A + iB with A, B Hermitian) -> inverse FFT of length mx -> six real rows in physical space ->
// products -> packed forward FFTs -> unpack -> truncate to p < pout.
//   NPROD = 3: H = u x omega (reading R1).   NPROD = 7: uu,uv,uw,vv,vw,ww, om.om (filter, R12).
// zpad fields in order u,v,w,om_x,om_y,om_z.
// =====================================================================================================
template <int NPROD>
__global__ void __launch_bounds__(256) k_xfft_prod(PlaneParams P, const double2* __restrict__ zpad, int npl,
                                                   double2* __restrict__ xh, int pout) {
    extern __shared__ double2 smem_raw[];
    constexpr int NC = (NPROD + 1) / 2;            // packed complex sequences after the products
    constexpr int NS = (NC > 3) ? NC : 3;
    c2* data = reinterpret_cast<c2*>(smem_raw);    // [NS][mx]
    const int mx = P.mx, nxh = P.nxh, mz = P.mz;
    const int r = blockIdx.x, jc = blockIdx.y;
    const size_t rowoff = ((size_t)jc * mz + r) * nxh;
    const size_t fstride = (size_t)npl * mz * nxh;
    // pack: C[k] = A[k] + i B[k], C[mx-k] = conj(A[k]) + i conj(B[k]); imaginary part of the k=0 entries dropped (R14)
    for (int w = threadIdx.x; w < 3 * (mx / 2 + 1); w += blockDim.x) {
        const int pr = w / (mx / 2 + 1), k = w - pr * (mx / 2 + 1);
        c2 A = mk(0, 0), B = mk(0, 0);
        if (k < nxh) {
            A = ldc(zpad + (size_t)(2 * pr) * fstride + rowoff + k);
            B = ldc(zpad + (size_t)(2 * pr + 1) * fstride + rowoff + k);
        }
        c2* C = data + (size_t)pr * mx;
        if (k == 0) C[0] = mk(A.x, B.x);
        else {
            C[k] = mk(A.x - B.y, A.y + B.x);
            if (k < mx - k) C[mx - k] = mk(A.x + B.y, -A.y + B.x);
        }
    }
    __syncthreads();
    fft_inplace<true, false, false>(data, P.fx, 3, 1, mx);
    // products (any order of the physical points)
    for (int n = threadIdx.x; n < mx; n += blockDim.x) {
        const c2 a = data[n], b = data[mx + n], c = data[2 * mx + n];
        const double u = a.x, v = a.y, w = b.x, ox = b.y, oy = c.x, oz = c.y;
        if (NPROD == 3) {
            data[n] = mk(v * oz - w * oy, w * ox - u * oz);
            data[mx + n] = mk(u * oy - v * ox, 0.0);
        } else {
            data[n] = mk(u * u, u * v);
            data[mx + n] = mk(u * w, v * v);
            data[2 * mx + n] = mk(v * w, w * w);
            data[3 * mx + n] = mk(ox * ox + oy * oy + oz * oz, 0.0);
        }
    }
    __syncthreads();
    fft_inplace<false, true, false>(data, P.fx, NC, 1, mx);
    // unpack: A[k] = (D[k] + conj D[mx-k])/2, B[k] = (D[k] - conj D[mx-k])/(2i)
    const size_t ofs = (size_t)npl * mz * pout;
    const size_t orow = ((size_t)jc * mz + r) * pout;
    for (int w = threadIdx.x; w < NC * pout; w += blockDim.x) {
        const int pr = w / pout, k = w - pr * pout;
        const c2* D = data + (size_t)pr * mx;
        const c2 d = D[k], e = D[k == 0 ? 0 : mx - k];
        const c2 A = mk(0.5 * (d.x + e.x), 0.5 * (d.y - e.y));
        const c2 B = mk(0.5 * (d.y + e.y), -0.5 * (d.x - e.x));
        stc(xh + (size_t)(2 * pr) * ofs + orow + k, A);
        if (2 * pr + 1 < NPROD) stc(xh + (size_t)(2 * pr + 1) * ofs + orow + k, B);
    }
}

// =====================================================================================================
// a13 first part: copy the retained modes of u,v,w (plane layout) into the filter output.
// =====================================================================================================
__global__ void k_filter_copy(PlaneParams P, FieldPtrs in, double2* __restrict__ out, int kxc, int kzc) {
    const int nr = 2 * kzc + 1, npk = kxc + 1;
    const size_t per = (size_t)P.ny * nr * npk;
    const size_t total = 3 * per;
    for (size_t w = (size_t)blockIdx.x * blockDim.x + threadIdx.x; w < total; w += (size_t)gridDim.x * blockDim.x) {
        const int fi = (int)(w / per);
        size_t rem = w - (size_t)fi * per;
        const int j = (int)(rem / ((size_t)nr * npk));
        rem -= (size_t)j * nr * npk;
        const int rr = (int)(rem / npk), p = (int)(rem - (size_t)rr * npk);
        const int s = (rr <= kzc) ? rr : P.nz - (nr - rr);
        out[w] = in.f[fi][(size_t)j * P.nm + (size_t)s * P.nxh + p];
    }
}

// =====================================================================================================
// a14: plane statistics, one CTA per y plane: sums over modes of w_p Re(a conj b).
// acc[10][ny] running sums (+=).
// =====================================================================================================
__global__ void __launch_bounds__(256) k_stats(PlaneParams P, FieldPtrs in /* u,v,w,ox,oy,oz */, double* __restrict__ acc) {
    const int j = blockIdx.x;
    double s[7] = {0, 0, 0, 0, 0, 0, 0};
    const size_t off = (size_t)j * P.nm;
    for (long long m = threadIdx.x; m < P.nm; m += blockDim.x) {
        const int p = (int)(m % P.nxh);
        const double wgt = (p == 0) ? 1.0 : 2.0;
        const c2 u = ldc(in.f[0] + off + m), v = ldc(in.f[1] + off + m), w = ldc(in.f[2] + off + m);
        const c2 ox = ldc(in.f[3] + off + m), oy = ldc(in.f[4] + off + m), oz = ldc(in.f[5] + off + m);
        s[0] += wgt * (u.x * u.x + u.y * u.y);
        s[1] += wgt * (u.x * v.x + u.y * v.y);
        s[2] += wgt * (u.x * w.x + u.y * w.y);
        s[3] += wgt * (v.x * v.x + v.y * v.y);
        s[4] += wgt * (v.x * w.x + v.y * w.y);
        s[5] += wgt * (w.x * w.x + w.y * w.y);
        s[6] += wgt * (ox.x * ox.x + ox.y * ox.y + oy.x * oy.x + oy.y * oy.y + oz.x * oz.x + oz.y * oz.y);
    }
    __shared__ double red[7][8];
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        double v = s[k];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) red[k][threadIdx.x >> 5] = v;
    }
    __syncthreads();
    if (threadIdx.x < 7) {
        double v = 0;
        for (int wv = 0; wv < (int)(blockDim.x >> 5); ++wv) v += red[threadIdx.x][wv];
        acc[(size_t)(3 + threadIdx.x) * P.ny + j] += v;
    }
    if (threadIdx.x == 32) {
        acc[0 * (size_t)P.ny + j] += in.f[0][off].x;
        acc[1 * (size_t)P.ny + j] += in.f[1][off].x;
        acc[2 * (size_t)P.ny + j] += in.f[2][off].x;
    }
}

// =====================================================================================================
// a2 / a8: plain transposes between LINE layout [nm][ny] and PLANE layout [ny][nm] (16-byte elements),
// 32x32 tiles through shared memory.  dir 0: line -> plane, 1: plane -> line.
// =====================================================================================================
__global__ void __launch_bounds__(256) k_transpose(const double2* __restrict__ in, double2* __restrict__ out, long long nm, int ny, int dir) {
    __shared__ double2 tile[32][33];
    // in is [R][C] -> out [C][R]
    const long long R = dir == 0 ? nm : ny, C = dir == 0 ? ny : nm;
    const long long c0 = (long long)blockIdx.x * 32, r0 = (long long)blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8
    for (int k = ty; k < 32; k += 8) {
        const long long r = r0 + k, c = c0 + tx;
        if (r < R && c < C) tile[k][tx] = in[r * C + c];
    }
    __syncthreads();
    for (int k = ty; k < 32; k += 8) {
        const long long c = c0 + k, r = r0 + tx;
        if (r < R && c < C) out[c * R + r] = tile[tx][k];
    }
}

}  // namespace chn
