// Host-side plan of the channel substep: mesh operators, factorisations, wavenumbers, FFT plans.
// Everything here is computed in long double on the host, independently of the oracle
// (include/chan.h; readings R2-R5).
#pragma once
#include <cstddef>
#include <vector>

namespace chn {

// Stage list of one transform length (chan_fft.cuh): stage s has radix[s] and sub-block length
// m[s] = product of the later radices; its twiddles exp(-2 pi i p k/(radix m)), k = 1..radix-1, p < m,
// start at complex offset twoff[s] of tw, laid out [(k-1) m + p].
struct FftPlan {
    int n = 0;
    std::vector<int> radix;     // DIF order (largest sub-transform first); DIT runs it backwards
    std::vector<int> m;
    std::vector<size_t> twoff;
    std::vector<double> tw;     // interleaved re,im
};

// Row-constant tables for one orientation (0 = natural y order, 1 = flipped, i -> ny-1-i).
// Every table has ny rows; *8 tables are padded to 8 doubles per row for aligned vector loads.
struct OrientTables {
    std::vector<double> B1;   // [ny][8]  first-derivative right-hand band, offsets -3..3 in [0..6]
    std::vector<double> A2;   // [ny][8]
    std::vector<double> B2;   // [ny][8]
    std::vector<double> lu1;  // [ny][8]  unpivoted LU of A1: l1,l2,l3 (multipliers of z_{i-1..i-3}), 1/u_ii, u1,u2,u3, 0
};

struct Plan {
    int nx, ny, nz, nxh, nzh, mx, mz;
    double lx, lz, nu, dt;
    int half_lhs, half_rhs, forcing;
    std::vector<double> y;
    std::vector<double> A1, B1, A2, B2;  // [ny][7] natural orientation (debug / parity with the oracle)
    OrientTables ot[2];
    std::vector<double> wm, wp;          // [ny] weights of (D1 f)(-1) and (D1 f)(+1) as functionals of f
    std::vector<double> wq;              // [ny] trapezoid weights of the mass flux
    std::vector<double> kx, kz;          // [nxh], [nz] (kz of the Nyquist slot is 0)
    FftPlan fx, fz;                      // lengths mx and mz
    double rk_alpha[3], rk_beta[3], rk_gamma[3], rk_zeta[3];
};

// Stage lists of the x and z transforms (0 = the planner's own choice, see chan_plan.cpp); build_plan calls it with
// zeros, chan_debug_set_tuning() again with the caller's overrides.  Returns 0 or CHAN_EINVAL.
int plan_ffts(Plan& P, int xfuse, int maxradix_z, int maxradix_x);

// PAPER.md section 2.3 (L100-102), host only: wall-layer error of the discrete homogeneous Helmholtz solution at both walls
// (err2[0]: y = -1, err2[1]: y = +1), and the paper's remedy (the first `npoints` mesh points of each wall displaced to
// minimise it).  chan_plan.cpp.
int mesh_helmholtz_error(int ny, const double* y, double lam, int nfirst, double* err2);
int mesh_optimize(int ny, double* y, int npoints, double lam, double max_shift, int sweeps, double* err_before, double* err_after);

// Returns 0 or a CHAN_E* status.
int build_plan(Plan& P, int nx, int ny, int nz, double lx, double lz, const double* y, double re_tau, double dt,
               int half_lhs, int half_rhs, int forcing);

}  // namespace chn
