// Plane-layout helper kernels around the transforms of chan_fft.cuh: the velocity part of the filter
// (a13), the plane statistics (a14) and the plain line <-> plane transposes (a2 / a8 at the ABI).
// PAPER.md L84, L124, L47.
#pragma once
#include <cuda_runtime.h>

#include "chan_fft.cuh"

namespace chn {

// =====================================================================================================
// a13 first part: copy the retained modes of u,v,w (plane layout) into the filter output.
// =====================================================================================================
__global__ void k_filter_copy(PlaneParams P, FieldPtrs in, double2* __restrict__ out, int kxc, int kzc, int f32) {
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
        const double2 val = in.f[fi][(size_t)j * P.nm + (size_t)s * P.nxh + p];
        if (!f32) out[w] = val;
        else reinterpret_cast<float2*>(out)[w] = make_float2((float)val.x, (float)val.y);   // binary32 database: round to nearest even
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
// a14 from a database just written (fp64): the (0,0) mode of the ten stored variables IS the plane statistics of
// the full field (second-order consistency) -- no pass over the fields.  acc[10][ny] += Re db[n][j][0][0].
// =====================================================================================================
__global__ void k_stats_from_db(int ny, size_t plane, const double2* __restrict__ db, double* __restrict__ acc) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= 10 * ny) return;
    acc[e] += db[(size_t)e * plane].x;
}

// =====================================================================================================
// One-dimensional co-spectra of uu,uv,uw,vv,vw,ww, om_i om_i at every y (NEXT-4 "more statistics"; PAPER.md L118,
// L163): ex[7][ny][nxh] = w_p sum over z slots of Re(a conj b), ez[7][ny][nz] = sum over p of w_p Re(a conj b).
// k_spectra_x: one thread per (y, p), marching over the z slots (consecutive lanes = consecutive p: coalesced);
// k_spectra_z: one warp per (y, z slot) row, lanes over p, shuffle reduction.  Outputs are overwritten.
// =====================================================================================================
__device__ __forceinline__ void cospectra7(const FieldPtrs& in, size_t o, double wgt, double (&s)[7]) {
    const c2 u = ldc(in.f[0] + o), v = ldc(in.f[1] + o), w = ldc(in.f[2] + o);
    const c2 ox = ldc(in.f[3] + o), oy = ldc(in.f[4] + o), oz = ldc(in.f[5] + o);
    s[0] += wgt * (u.x * u.x + u.y * u.y);
    s[1] += wgt * (u.x * v.x + u.y * v.y);
    s[2] += wgt * (u.x * w.x + u.y * w.y);
    s[3] += wgt * (v.x * v.x + v.y * v.y);
    s[4] += wgt * (v.x * w.x + v.y * w.y);
    s[5] += wgt * (w.x * w.x + w.y * w.y);
    s[6] += wgt * (ox.x * ox.x + ox.y * ox.y + oy.x * oy.x + oy.y * oy.y + oz.x * oz.x + oz.y * oz.y);
}
__global__ void __launch_bounds__(128) k_spectra_x(PlaneParams P, FieldPtrs in, double* __restrict__ ex) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (p >= P.nxh) return;
    double s[7] = {0, 0, 0, 0, 0, 0, 0};
    const size_t off = (size_t)j * P.nm + p;
    for (int z = 0; z < P.nz; ++z) cospectra7(in, off + (size_t)z * P.nxh, 1.0, s);
    const double wgt = (p == 0) ? 1.0 : 2.0;
#pragma unroll
    for (int k = 0; k < 7; ++k) ex[((size_t)k * P.ny + j) * P.nxh + p] = wgt * s[k];
}
__global__ void __launch_bounds__(256) k_spectra_z(PlaneParams P, FieldPtrs in, double* __restrict__ ez) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int z = blockIdx.x * (blockDim.x >> 5) + warp, j = blockIdx.y;
    if (z >= P.nz) return;
    double s[7] = {0, 0, 0, 0, 0, 0, 0};
    const size_t off = (size_t)j * P.nm + (size_t)z * P.nxh;
    for (int p = lane; p < P.nxh; p += 32) cospectra7(in, off + p, (p == 0) ? 1.0 : 2.0, s);
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        double v = s[k];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) ez[((size_t)k * P.ny + j) * P.nz + z] = v;
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
    // the mode dimension is tiled by blockIdx.x in both directions (gridDim.y is limited to 65535 tiles)
    const long long c0 = (long long)(dir == 0 ? blockIdx.y : blockIdx.x) * 32, r0 = (long long)(dir == 0 ? blockIdx.x : blockIdx.y) * 32;
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

// =====================================================================================================
// fp64 FMA micro-benchmark (bench.py's "alu" roof): 8 independent register-only DFMA chains per
// thread, `iters` rounds; nothing touches memory until the final store that keeps the chains alive.
// flops = 2 * 8 * iters * threads.
// =====================================================================================================
__global__ void __launch_bounds__(256) k_fma_peak(double* __restrict__ sink, int iters, double a, double b) {
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
#pragma unroll 4
    for (int i = 0; i < iters; ++i) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 12345.678) sink[0] = s;      // practically never: the store only pins the arithmetic
}

}  // namespace chn
