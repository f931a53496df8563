// Wall-normal (y) phase, common part: complex helpers, the parameter block of the marching sweeps
// (chan_ysweeps.cuh) and the mean-mode kernels (step a12 of DESIGN.md; PAPER.md L61 constant mass flux).
//
// Banded systems are solved by unpivoted elimination in ascending row order of an ORIENTATION:
// orientation 0 is the natural order j = 0..ny-1, orientation 1 the flipped order i = ny-1-j (the
// same system with rows and columns reversed).  A sweep that walks physical rows downwards can
// therefore back-substitute an orientation-0 system and forward-eliminate an orientation-1 system in
// the same pass, and vice versa, which is what chains the sweeps without extra passes.
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
#define CHAN_PF 4
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
