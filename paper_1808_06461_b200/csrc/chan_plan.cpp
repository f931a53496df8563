// Host plan: compact finite-difference rows on the caller's mesh, their factorisations, wavenumbers,
// FFT radix plans and twiddles.  long double throughout; rounded to double once.
//
// Compact rows ("seven-point compact finite differences", L100 "up to twelfth order of
// consistency"; reading R4): row j of the d-th derivative satisfies
//     sum_m a_m f^(d)(y_{j+m}) = sum_m b_m f(y_{j+m}),   a_0 = 1,
// exactly for all polynomials up to degree (#unknowns - 1).  The moment system is written in the
// Chebyshev basis T_k(t) on the stencil's own interval mapped to t in [-1,1] (reading R5), with the
// b_m scaled by the half-width^d, and solved by partially pivoted elimination plus one refinement step.
#include "chan_plan.h"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "../../include/chan.h"

namespace chn {
namespace {

typedef long double ld;

// Solve the dense n x n system M x = r (row-major M) by Gaussian elimination with partial pivoting.
bool dense_solve(int n, std::vector<ld> M, std::vector<ld> r, std::vector<ld>& x) {
    std::vector<int> perm(n);
    for (int i = 0; i < n; ++i) perm[i] = i;
    for (int c = 0; c < n; ++c) {
        int p = c;
        for (int i = c + 1; i < n; ++i)
            if (fabsl(M[i * n + c]) > fabsl(M[p * n + c])) p = i;
        if (M[p * n + c] == 0.0L) return false;
        if (p != c) {
            for (int k = 0; k < n; ++k) std::swap(M[c * n + k], M[p * n + k]);
            std::swap(r[c], r[p]);
        }
        for (int i = c + 1; i < n; ++i) {
            ld f = M[i * n + c] / M[c * n + c];
            if (f == 0.0L) continue;
            for (int k = c; k < n; ++k) M[i * n + k] -= f * M[c * n + k];
            r[i] -= f * r[c];
        }
    }
    x.assign(n, 0.0L);
    for (int i = n - 1; i >= 0; --i) {
        ld s = r[i];
        for (int k = i + 1; k < n; ++k) s -= M[i * n + k] * x[k];
        x[i] = s / M[i * n + i];
    }
    return true;
}

// T_k(t), T_k'(t), T_k''(t) for k = 0..n-1 by the three-term recurrences.
void cheb_all(ld t, int n, std::vector<ld>& T0, std::vector<ld>& T1, std::vector<ld>& T2) {
    T0.assign(n, 0); T1.assign(n, 0); T2.assign(n, 0);
    T0[0] = 1;
    if (n > 1) { T0[1] = t; T1[1] = 1; }
    for (int k = 2; k < n; ++k) {
        T0[k] = 2 * t * T0[k - 1] - T0[k - 2];
        T1[k] = 2 * T0[k - 1] + 2 * t * T1[k - 1] - T1[k - 2];
        T2[k] = 4 * T1[k - 1] + 2 * t * T2[k - 1] - T2[k - 2];
    }
}

// One compact row.  lhs/rhs: offset lists (lhs contains 0).  Writes a[3+m], b[3+m].
bool compact_row(const std::vector<double>& y, int j, const std::vector<int>& lhs, const std::vector<int>& rhs,
                 int deriv, double* a, double* b) {
    int lo = 0, hi = 0;
    for (int m : lhs) { lo = std::min(lo, m); hi = std::max(hi, m); }
    for (int m : rhs) { lo = std::min(lo, m); hi = std::max(hi, m); }
    const ld ylo = y[j + lo], yhi = y[j + hi];
    const ld ym = (ylo + yhi) / 2, hw = (yhi - ylo) / 2;
    std::vector<int> lf;
    for (int m : lhs) if (m != 0) lf.push_back(m);
    const int n = (int)lf.size() + (int)rhs.size();
    std::vector<ld> M((size_t)n * n), r(n), x, T0, T1, T2;
    // column data per stencil point
    auto fill = [&](int m, int col, bool is_lhs) {
        ld t = ((ld)y[j + m] - ym) / hw;
        cheb_all(t, n, T0, T1, T2);
        for (int k = 0; k < n; ++k) {
            ld v = is_lhs ? (deriv == 1 ? T1[k] : T2[k]) : -T0[k];
            if (col >= 0) M[(size_t)k * n + col] = v; else r[k] = -v;  // col < 0: the a_0 = 1 term
        }
    };
    int col = 0;
    for (int m : lf) fill(m, col++, true);
    for (int m : rhs) fill(m, col++, false);
    fill(0, -1, true);
    if (!dense_solve(n, M, r, x)) return false;
    // one step of iterative refinement in the same precision (residual is cheap and exact enough)
    std::vector<ld> res(n), dx;
    for (int k = 0; k < n; ++k) {
        ld s = r[k];
        for (int c = 0; c < n; ++c) s -= M[(size_t)k * n + c] * x[c];
        res[k] = s;
    }
    if (dense_solve(n, M, res, dx)) for (int k = 0; k < n; ++k) x[k] += dx[k];
    for (int k = 0; k < 7; ++k) { a[k] = 0; b[k] = 0; }
    a[3] = 1.0;
    col = 0;
    const ld sc = (deriv == 1) ? hw : hw * hw;  // unknown b' = b * hw^d  (LHS derivative columns carry 1/hw^d)
    for (int m : lf) a[3 + m] = (double)x[col++];
    for (int m : rhs) b[3 + m] = (double)(x[col++] / sc);
    return true;
}

// Unpivoted band LU of a [ny][7] table in long double; writes rows {l1,l2,l3,1/u_ii,u1,u2,u3,0}.
bool band_lu(int ny, const std::vector<ld>& T, std::vector<double>& out) {
    std::vector<ld> W(T);
    out.assign((size_t)ny * 8, 0.0);
    std::vector<ld> L((size_t)ny * 3, 0.0L);
    for (int j = 0; j < ny; ++j) {
        ld piv = W[(size_t)j * 7 + 3];
        if (piv == 0.0L) return false;
        for (int t = 1; t <= 3 && j + t < ny; ++t) {
            ld l = W[(size_t)(j + t) * 7 + 3 - t] / piv;
            L[(size_t)(j + t) * 3 + (t - 1)] = l;
            for (int cc = 1; cc <= 3; ++cc) W[(size_t)(j + t) * 7 + 3 - t + cc] -= l * W[(size_t)j * 7 + 3 + cc];
            W[(size_t)(j + t) * 7 + 3 - t] = 0;
        }
    }
    for (int j = 0; j < ny; ++j) {
        double* o = &out[(size_t)j * 8];
        o[0] = (double)L[(size_t)j * 3 + 0];
        o[1] = (double)L[(size_t)j * 3 + 1];
        o[2] = (double)L[(size_t)j * 3 + 2];
        o[3] = (double)(1.0L / W[(size_t)j * 7 + 3]);
        o[4] = (double)W[(size_t)j * 7 + 4];
        o[5] = (double)W[(size_t)j * 7 + 5];
        o[6] = (double)W[(size_t)j * 7 + 6];
    }
    return true;
}

// Solve T x = r for a [ny][7] band table without pivoting (long double).
bool band_solve(int ny, const std::vector<ld>& T, std::vector<ld>& x) {
    std::vector<ld> W(T);
    for (int j = 0; j < ny; ++j) {
        ld piv = W[(size_t)j * 7 + 3];
        if (piv == 0.0L) return false;
        for (int t = 1; t <= 3 && j + t < ny; ++t) {
            ld l = W[(size_t)(j + t) * 7 + 3 - t] / piv;
            for (int cc = 1; cc <= 3; ++cc) W[(size_t)(j + t) * 7 + 3 - t + cc] -= l * W[(size_t)j * 7 + 3 + cc];
            x[j + t] -= l * x[j];
        }
    }
    for (int j = ny - 1; j >= 0; --j) {
        ld s = x[j];
        for (int cc = 1; cc <= 3 && j + cc < ny; ++cc) s -= W[(size_t)j * 7 + 3 + cc] * x[j + cc];
        x[j] = s / W[(size_t)j * 7 + 3];
    }
    return true;
}

void flip_table(int ny, const std::vector<double>& T, std::vector<double>& F) {  // F[i][3+m] = T[ny-1-i][3-m]
    F.assign((size_t)ny * 7, 0.0);
    for (int i = 0; i < ny; ++i)
        for (int m = -3; m <= 3; ++m) F[(size_t)i * 7 + 3 + m] = T[(size_t)(ny - 1 - i) * 7 + 3 - m];
}

void pad8(int ny, const std::vector<double>& T, std::vector<double>& O) {
    O.assign((size_t)ny * 8, 0.0);
    for (int i = 0; i < ny; ++i) for (int k = 0; k < 7; ++k) O[(size_t)i * 8 + k] = T[(size_t)i * 7 + k];
}

// Stage list for length n = 2^a 3^b (chan_fft.cuh).  `fused_last` > 0 fixes the last radix (the x
// transform fuses that stage with the pointwise products); the rest is the shortest list of radices from
// {18,16,12,8,6,4,3,2} (fewest radix-12/16 stages among the shortest), radices with a factor 3 first so that the
// zero band of the 3/2 padding lines up with whole inputs of the first butterfly.
void best_radices(int rest, int maxr, std::vector<int>& cur, std::vector<int>& best) {
    static const int cand[8] = {18, 16, 12, 8, 6, 4, 3, 2};
    if (rest == 1) {
        auto key = [](const std::vector<int>& v) {
            int big = 0, c2 = 0, mx = 0;
            for (int r : v) { big += (r == 12) + 2 * (r > 12); c2 += (r <= 3); mx = r > mx ? r : mx; }
            return (long)v.size() * 100000 + big * 1000 + mx * 10 + c2;
        };
        if (best.empty() || key(cur) < key(best)) best = cur;
        return;
    }
    if (!best.empty() && cur.size() + 1 > best.size()) return;
    for (int r : cand) {
        if (r > maxr || rest % r) continue;
        if (!cur.empty() && r > cur.back()) continue;   // non-increasing: each multiset once
        cur.push_back(r);
        best_radices(rest / r, maxr, cur, best);
        cur.pop_back();
    }
}

bool make_fft_plan(int n, int fused_last, int maxr, FftPlan& F) {
    F.n = n;
    F.radix.clear(); F.m.clear(); F.twoff.clear(); F.tw.clear();
    int r = n;
    while (r % 3 == 0) r /= 3;
    while (r % 2 == 0) r /= 2;
    if (r != 1 || n < 2) return false;
    int rest = n;
    if (fused_last > 0) {
        if (n % fused_last) return false;
        rest = n / fused_last;
    }
    std::vector<int> cur, best;
    if (rest > 1) {
        best_radices(rest, maxr, cur, best);
        if (best.empty()) return false;
    }
    std::stable_sort(best.begin(), best.end(), [](int a, int b) {
        const int a3 = (a % 3 == 0), b3 = (b % 3 == 0);
        return a3 != b3 ? a3 > b3 : a > b;
    });
    F.radix = best;
    if (fused_last > 0) F.radix.push_back(fused_last);
    const ld two_pi = 6.283185307179586476925286766559005768L;
    int m = n;
    for (size_t s = 0; s < F.radix.size(); ++s) {
        const int R = F.radix[s];
        m /= R;
        F.m.push_back(m);
        F.twoff.push_back(F.tw.size() / 2);
        if (m == 1) continue;
        const long ncur = (long)R * m;
        for (int k = 1; k < R; ++k)
            for (int p = 0; p < m; ++p) {
                const long e = ((long)p * k) % ncur;
                const ld a = two_pi * (ld)e / (ld)ncur;
                F.tw.push_back((double)cosl(a));
                F.tw.push_back((double)(-sinl(a)));
            }
    }
    if (F.tw.empty()) { F.tw.push_back(1.0); F.tw.push_back(0.0); }
    return true;
}

}  // namespace

// ---- section 2.3 of the paper (L100-102): wall-layer error of the homogeneous Helmholtz solutions and the mesh remedy ----
namespace {

// D2 rows (A2, B2) of the mesh y for rows j in [lo, hi] into the [ny][7] tables (rows 0 and ny-1 are not used)
bool d2_rows(const std::vector<double>& y, int lo, int hi, std::vector<double>& A2, std::vector<double>& B2) {
    const int ny = (int)y.size();
    for (int j = std::max(lo, 1); j <= std::min(hi, ny - 2); ++j) {
        const int room = std::min(j, ny - 1 - j), s = std::min(3, room);
        std::vector<int> off;
        for (int m = -s; m <= s; ++m) off.push_back(m);
        if (!compact_row(y, j, off, off, 2, &A2[(size_t)j * 7], &B2[(size_t)j * 7])) return false;
    }
    return true;
}

// max over the first `nfirst` interior points next to the wall `side` (0: y = -1, 1: y = +1) of |phi_j - phi(y_j)|, phi the
// solution of phi'' = lam phi with phi = 1 at that wall and 0 at the other one
bool wall_error(const std::vector<double>& y, const std::vector<double>& A2, const std::vector<double>& B2, double lam, int nfirst,
                int side, double* err) {
    const int ny = (int)y.size();
    std::vector<ld> T((size_t)ny * 7, 0.0L), x(ny, 0.0L);
    for (int j = 1; j + 1 < ny; ++j)
        for (int k = 0; k < 7; ++k) T[(size_t)j * 7 + k] = (ld)B2[(size_t)j * 7 + k] - (ld)lam * (ld)A2[(size_t)j * 7 + k];
    T[3] = 1.0L; T[(size_t)(ny - 1) * 7 + 3] = 1.0L;
    x[side == 0 ? 0 : ny - 1] = 1.0L;
    if (!band_solve(ny, T, x)) return false;
    const ld k = sqrtl((ld)lam);
    ld e = 0;
    for (int n = 1; n <= nfirst && n + 1 < ny; ++n) {
        const int j = side == 0 ? n : ny - 1 - n;
        const ld d = side == 0 ? 1.0L + (ld)y[j] : 1.0L - (ld)y[j];      // distance from the wall that carries the 1
        const ld ex = expl(-k * d) * (1.0L - expl(-2.0L * k * (2.0L - d))) / (1.0L - expl(-4.0L * k));
        e = std::max(e, fabsl(x[j] - ex));
    }
    *err = (double)e;
    return true;
}

// Admissibility guard of the optimiser: every pivot of the unpivoted elimination of B2 - sigma A2 (Dirichlet rows) is
// negative, for sigma = 0, lam/100 and lam.  On admissible meshes (real negative D2-Dirichlet spectrum) all
// pivots are negative for every sigma >= 0; a displaced mesh whose spectrum has crossed to the right half plane shows
// positive pivots already at sigma = 0, and the marching kernels, which eliminate without pivoting, need the former.
bool pivots_negative(const std::vector<double>& A2, const std::vector<double>& B2, int ny, double lam) {
    const double sig[3] = {0.0, lam * 0.01, lam};
    for (double sg : sig) {
        std::vector<ld> W((size_t)ny * 7, 0.0L);
        for (int j = 1; j + 1 < ny; ++j)
            for (int k = 0; k < 7; ++k) W[(size_t)j * 7 + k] = (ld)B2[(size_t)j * 7 + k] - (ld)sg * (ld)A2[(size_t)j * 7 + k];
        W[3] = -1.0L; W[(size_t)(ny - 1) * 7 + 3] = -1.0L;
        for (int j = 0; j < ny; ++j) {
            const ld piv = W[(size_t)j * 7 + 3];
            if (!(piv < 0.0L)) return false;
            for (int t = 1; t <= 3 && j + t < ny; ++t) {
                const ld l = W[(size_t)(j + t) * 7 + 3 - t] / piv;
                for (int cc = 1; cc <= 3; ++cc) W[(size_t)(j + t) * 7 + 3 - t + cc] -= l * W[(size_t)j * 7 + 3 + cc];
            }
        }
    }
    return true;
}

}  // namespace

int mesh_helmholtz_error(int ny, const double* y, double lam, int nfirst, double* err2) {
    if (ny < 8 || !y || !(lam > 0) || nfirst < 1 || !err2) return CHAN_EINVAL;
    std::vector<double> yy(y, y + ny), A2((size_t)ny * 7, 0.0), B2((size_t)ny * 7, 0.0);
    for (int j = 1; j < ny; ++j) if (!(yy[j] > yy[j - 1])) return CHAN_EINVAL;
    if (!d2_rows(yy, 1, ny - 2, A2, B2)) return CHAN_EINVAL;
    for (int side = 0; side < 2; ++side) if (!wall_error(yy, A2, B2, lam, nfirst, side, &err2[side])) return CHAN_EINVAL;
    return CHAN_OK;
}

// Cyclic coordinate search with a halving step: point j (1 <= j <= npoints from each wall) may move by at most
// max_shift times the smaller of its two ORIGINAL neighbouring spacings, which keeps the mesh monotone for max_shift < 1/2
// and bounds the change of every spacing by 2 max_shift of the original one.  Objective: the wall error above at the
// wall the point belongs to.  Deterministic; the two walls are treated independently.
int mesh_optimize(int ny, double* y, int npoints, double lam, double max_shift, int sweeps, double* err_before, double* err_after) {
    if (ny < 16 || !y || npoints < 1 || 2 * (npoints + 4) > ny || !(lam > 0) || !(max_shift > 0) || max_shift >= 0.5 || sweeps < 1) return CHAN_EINVAL;
    std::vector<double> y0(y, y + ny), yy(y0), A2((size_t)ny * 7, 0.0), B2((size_t)ny * 7, 0.0);
    for (int j = 1; j < ny; ++j) if (!(yy[j] > yy[j - 1])) return CHAN_EINVAL;
    if (!d2_rows(yy, 1, ny - 2, A2, B2)) return CHAN_EINVAL;
    if (!pivots_negative(A2, B2, ny, lam)) return CHAN_EINVAL;      // the mesh handed in is not admissible itself
    const int nfirst = npoints + 3;
    // a mesh that is symmetric about y = 0 stays so: the mirror point moves with its twin and one wall is optimised
    bool sym = true;
    for (int j = 0; j < ny; ++j) if (y0[j] != -y0[ny - 1 - j]) sym = false;
    for (int side = 0; side < (sym ? 1 : 2); ++side) {
        double best;
        if (!wall_error(yy, A2, B2, lam, nfirst, side, &best)) return CHAN_EINVAL;
        if (err_before) { err_before[side] = best; if (sym) err_before[1] = best; }
        double step = max_shift;
        auto place = [&](int j, double v) {
            yy[j] = v;
            bool ok = d2_rows(yy, j - 3, j + 3, A2, B2);
            if (sym) { const int jm = ny - 1 - j; yy[jm] = -v; ok = ok && d2_rows(yy, jm - 3, jm + 3, A2, B2); }
            return ok;
        };
        for (int sw = 0; sw < sweeps; ++sw, step *= 0.5) {
            for (int n = 1; n <= npoints; ++n) {
                const int j = side == 0 ? n : ny - 1 - n;
                const double h = std::min(y0[j] - y0[j - 1], y0[j + 1] - y0[j]);
                const double keep = yy[j];
                double arg = keep;
                for (int sg = -1; sg <= 1; sg += 2) {
                    double cand = keep + sg * step * h;
                    cand = std::min(std::max(cand, y0[j] - max_shift * h), y0[j] + max_shift * h);
                    if (cand == keep) continue;
                    double e;
                    if (!place(j, cand) || !wall_error(yy, A2, B2, lam, nfirst, side, &e)) return CHAN_EINVAL;
                    if (e < best && pivots_negative(A2, B2, ny, lam)) { best = e; arg = cand; }
                }
                if (!place(j, arg)) return CHAN_EINVAL;
            }
        }
        if (err_after) { err_after[side] = best; if (sym) err_after[1] = best; }
    }
    for (int j = 0; j < ny; ++j) y[j] = yy[j];
    return CHAN_OK;
}

// Stage lists of the two transform lengths.  xfuse: 4 | 8 = radix of the x stage fused with the products (0: the one
// that gives the shorter stage list, then the one without radix-12 stages, then 4: lighter fused stage);
// maxr: largest radix of a z stage (0: 12); maxrx: largest radix of an x stage (0: 18 -- two shared-memory stages in
// front of the fused one at 1536 points [12,16|8] and at 2304 points [18,16|8]).
int plan_ffts(Plan& P, int xfuse, int maxr, int maxrx) {
    if (maxr < 2) maxr = 12;
    if (maxrx < 2) maxrx = 18;
    int fuse = 4;
    if (xfuse == 4 || xfuse == 8) fuse = xfuse;
    else {
        FftPlan f4, f8;
        auto key = [](const FftPlan& f) {
            int big = 0;
            for (int r : f.radix) big += (r == 12) + 3 * (r > 12);
            return (int)f.radix.size() * 100 + big;
        };
        if (make_fft_plan(P.mx, 4, maxrx, f4) && make_fft_plan(P.mx, 8, maxrx, f8) && key(f8) < key(f4)) fuse = 8;
    }
    if (!make_fft_plan(P.mx, fuse, maxrx, P.fx) || !make_fft_plan(P.mz, 0, maxr, P.fz)) return CHAN_EINVAL;
    return CHAN_OK;
}

int build_plan(Plan& P, int nx, int ny, int nz, double lx, double lz, const double* y, double re_tau, double dt,
               int half_lhs, int half_rhs, int forcing) {
    if (nx < 4 || nz < 4 || (nx & 1) || (nz & 1) || ny < 8 || !y) return CHAN_EINVAL;
    if (!(lx > 0) || !(lz > 0) || !(re_tau > 0) || !(dt > 0)) return CHAN_EINVAL;
    if (half_lhs < 1 || half_lhs > 3 || half_rhs < 1 || half_rhs > 3 || forcing < 0 || forcing > 1) return CHAN_EINVAL;
    for (int j = 1; j < ny; ++j) if (!(y[j] > y[j - 1])) return CHAN_EINVAL;
    if (y[0] != -1.0 || y[ny - 1] != 1.0) return CHAN_EINVAL;
    P.nx = nx; P.ny = ny; P.nz = nz; P.nxh = nx / 2; P.nzh = nz / 2; P.mx = 3 * nx / 2; P.mz = 3 * nz / 2;
    P.lx = lx; P.lz = lz; P.nu = 1.0 / re_tau; P.dt = dt;
    P.half_lhs = half_lhs; P.half_rhs = half_rhs; P.forcing = forcing;
    P.y.assign(y, y + ny);
    if (P.mx % 8) return CHAN_EINVAL;   // x: the last stage is fused with the products and needs the 8-aligned swizzle of chan_fft.cuh
    if (int rc = plan_ffts(P, 0, 0, 0)) return rc;

    // RK3 constants of [34] (reading R3)
    const double al[3] = {29.0 / 96.0, -3.0 / 40.0, 1.0 / 6.0}, be[3] = {37.0 / 160.0, 5.0 / 24.0, 1.0 / 6.0};
    const double ga[3] = {8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0}, ze[3] = {0.0, -17.0 / 60.0, -5.0 / 12.0};
    for (int i = 0; i < 3; ++i) { P.rk_alpha[i] = al[i]; P.rk_beta[i] = be[i]; P.rk_gamma[i] = ga[i]; P.rk_zeta[i] = ze[i]; }

    // compact rows
    P.A1.assign((size_t)ny * 7, 0.0); P.B1.assign((size_t)ny * 7, 0.0);
    P.A2.assign((size_t)ny * 7, 0.0); P.B2.assign((size_t)ny * 7, 0.0);
    for (int j = 0; j < ny; ++j) {
        const int room = std::min(j, ny - 1 - j);
        for (int d = 1; d <= 2; ++d) {
            std::vector<int> lo, ro;
            if (room == 0) {
                if (d == 2) continue;
                const int sg = (j == 0) ? 1 : -1;
                lo = {0, sg};
                ro = {0, sg, 2 * sg, 3 * sg};
            } else {
                const int sl = std::min(half_lhs, room), sr = std::min(half_rhs, room);
                for (int m = -sl; m <= sl; ++m) lo.push_back(m);
                for (int m = -sr; m <= sr; ++m) ro.push_back(m);
            }
            double* a = (d == 1 ? &P.A1[(size_t)j * 7] : &P.A2[(size_t)j * 7]);
            double* b = (d == 1 ? &P.B1[(size_t)j * 7] : &P.B2[(size_t)j * 7]);
            if (!compact_row(P.y, j, lo, ro, d, a, b)) return CHAN_EINVAL;
        }
    }

    // orientation tables and the LU of A1 in both orientations
    for (int o = 0; o < 2; ++o) {
        std::vector<double> a1, b1, a2, b2;
        if (o == 0) { a1 = P.A1; b1 = P.B1; a2 = P.A2; b2 = P.B2; }
        else { flip_table(ny, P.A1, a1); flip_table(ny, P.B1, b1); flip_table(ny, P.A2, a2); flip_table(ny, P.B2, b2); }
        pad8(ny, b1, P.ot[o].B1); pad8(ny, a2, P.ot[o].A2); pad8(ny, b2, P.ot[o].B2);
        std::vector<ld> T(a1.begin(), a1.end());
        if (!band_lu(ny, T, P.ot[o].lu1)) return CHAN_EINVAL;
    }

    // wall functionals: (D1 f)(wall) = e^T A1^{-1} B1 f = (A1^{-T} e)^T B1 f
    {
        std::vector<ld> At((size_t)ny * 7, 0.0L);
        for (int j = 0; j < ny; ++j)
            for (int m = -3; m <= 3; ++m)
                if (j + m >= 0 && j + m < ny) At[(size_t)j * 7 + 3 + m] = P.A1[(size_t)(j + m) * 7 + 3 - m];
        for (int side = 0; side < 2; ++side) {
            std::vector<ld> s(ny, 0.0L);
            s[side == 0 ? 0 : ny - 1] = 1.0L;
            if (!band_solve(ny, At, s)) return CHAN_EINVAL;
            std::vector<double>& w = (side == 0 ? P.wm : P.wp);
            w.assign(ny, 0.0);
            for (int c = 0; c < ny; ++c) {
                ld acc = 0;
                for (int m = -3; m <= 3; ++m) {  // w_c = sum_j s_j B1[j][c], j = c - m
                    int j = c - m;
                    if (j >= 0 && j < ny) acc += s[j] * (ld)P.B1[(size_t)j * 7 + 3 + m];
                }
                w[c] = (double)acc;
            }
        }
    }

    // trapezoid weights (reading R8)
    P.wq.assign(ny, 0.0);
    for (int j = 0; j + 1 < ny; ++j) {
        const double h = 0.5 * (P.y[j + 1] - P.y[j]);
        P.wq[j] += h; P.wq[j + 1] += h;
    }

    // wavenumbers (reading R2)
    const double two_pi = 6.283185307179586476925286766559;
    P.kx.resize(P.nxh); P.kz.resize(nz);
    for (int p = 0; p < P.nxh; ++p) P.kx[p] = two_pi * p / lx;
    for (int s = 0; s < nz; ++s) {
        int q = (s < P.nzh) ? s : (s == P.nzh ? 0 : s - nz);
        P.kz[s] = two_pi * q / lz;
    }
    return CHAN_OK;
}

}  // namespace chn
