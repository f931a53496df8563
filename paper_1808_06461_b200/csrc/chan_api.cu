// C ABI of libchan (include/chan.h): handle, workspace carving, launch sequences.
// No device memory is allocated here: everything is carved from the caller's workspace.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/chan.h"
#include "chan_fft.cuh"
#include "chan_planekernels.cuh"
#include "chan_plan.h"
#include "chan_post.cuh"
#include "chan_ykernels.cuh"
#include "chan_ysweeps.cuh"

using namespace chn;

namespace {
constexpr int kThreadsY = 128;
constexpr size_t kAlign = 256;
inline size_t up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }
}  // namespace

struct chan {
    Plan P;
    bool bound = false, have_state = false;
    int isub = 0;
    cudaStream_t stream = nullptr;
    char* ws = nullptr;
    size_t ws_bytes = 0;
    long long launches = 0;
    long long nsamples = 0;
    int cuda_err = 0;
    // sizes
    size_t F = 0;          // bytes of one complex field
    size_t s1_bytes = 0;   // bytes of the scratch field s1 (>= F; also the host staging of the filter output)
    long long nm = 0;
    int pc = 1;            // planes per FFT chunk
    int Tz = 1;            // k_x columns per z-FFT tile
    int xthreads = 128;    // threads per row CTA of the x pass
    int zthreads = 256;    // threads per tile CTA of the z passes
    void (*kzinv)(PlaneParams, FieldPtrs, int, int, double2*, int) = nullptr;
    void (*kzfwd)(PlaneParams, const double2*, int, int, int, FieldPtrsW, double, int, int, int, int) = nullptr;
    void (*kx3)(PlaneParams, const double2*, int, double2*, int) = nullptr;
    void (*kx7)(PlaneParams, const double2*, int, double2*, int) = nullptr;
    // 2-CTA cluster variants of the z passes (tile split by rows, twice the columns per tile), if compiled for this plan
    void (*kzinv_c)(PlaneParams, FieldPtrs, int, int, double2*, int) = nullptr;
    void (*kzfwd_c)(PlaneParams, const double2*, int, int, int, FieldPtrsW, double, int, int, int, int) = nullptr;
    bool zcluster = false;     // the z passes run through them, with Tzc columns per tile
    int Tzc = 0;
    void (*kmerged)(PlaneParams, MergedArgs) = nullptr;   // K2 | K3 | K4 of neighbouring chunks in one launch, if compiled for this plan
    bool merged = false;   // the substep's plane phase runs through kmerged
    bool zspecial = false, xspecial = false;
    int out_f32 = 0;           // filtered database as complex64 (chan_set_filter_precision)
    chan_tuning_t tune = {};   // caller overrides (chan_debug_set_tuning), 0 = the plan's own choice
    // device pointers (carved)
    double2 *v, *phi, *omy, *hv, *hg, *u, *w, *ox, *oz;   // plane layout fields
    double2 *H1, *H2, *H3;                                 // alias u, w, ox
    // y-phase scratch: only s1 is storage of its own, the rest alias field buffers that are dead while the
    // y-phase runs: facA = oz, facB = v, z2 = u, r1|r2 = ox, r3|r4 = w
    double2 *s1, *facA, *facB, *z1, *z2; double *r1, *r2, *r3, *r4; double4* coef;
    double2 *zpad, *xh;
    double *U, *W, *H1p, *H3p, *meanwork, *scal, *stats;
    // tables
    double* tab[2][4];     // B1, A2, B2, lu1 per orientation
    double *kx, *kz, *wm, *wp, *wq;
    double2 *twx, *twz;
    size_t need = 0;
    // per-kernel-class CUDA-event profiling (chan_debug_profile)
    bool prof_on = false;
    int cur_kc = 0;
    std::vector<cudaEvent_t> prof_ev;   // pairs
    std::vector<int> prof_cls;
};

namespace {

struct Carver {
    char* base; size_t off = 0;
    template <typename T> T* take(size_t bytes) { T* p = base ? reinterpret_cast<T*>(base + off) : nullptr; off += up(bytes); return p; }
};

void choose_tiling(chan_t* h) {
    const Plan& P = h->P;
    const chan_tuning_t& U = h->tune;
    int T = 16;
    while (T > 1 && (size_t)P.mz * T * 16 > 112 * 1024) T >>= 1;
    while (T > 1 && T > P.nxh) T >>= 1;
    h->Tz = U.tz ? U.tz : T;
    if (U.zthreads) h->zthreads = U.zthreads;
    else {
        // threads per z tile: the count that leaves the fewest idle (butterfly, column) slots over the stages -- a stage of
        // radix R has (mz / R) Tz items, each costing ~R; 1728 = 12^3 with Tz = 4 gives 576 items per stage: three full
        // rounds at 192 threads against two and a quarter at 256 (measured: K2 -2.7%, K4 -1.5%).  Ties go to more threads.
        long best = -1; int arg = 256;
        for (int nt = 256; nt >= 128; nt -= 32) {
            long slots = 0;
            for (int R : P.fz.radix) { const long items = (long)(P.mz / R) * h->Tz; slots += ((items + nt - 1) / nt) * nt * R; }
            if (best < 0 || slots < best) { best = slots; arg = nt; }
        }
        h->zthreads = arg;
    }
    // row pieces narrower than 128 B (fewer than 8 columns per tile) cost ~14% per halving (config 3); the cluster variant
    // splits the tile by rows over two CTAs and doubles the columns
    h->Tzc = 2 * h->Tz;
    const bool can = h->kzinv_c && h->Tzc <= 16 && h->Tzc <= P.nxh && !h->merged && (size_t)P.mz * h->Tzc * 8 <= 112 * 1024;
    h->zcluster = can && U.z_cluster == 2;    // measured slower than one CTA per narrower tile: opt-in
    h->xthreads = U.xthreads ? U.xthreads : (((size_t)3 * P.mx * 16 > 72 * 1024) ? 256 : 128);   // <= 3 CTAs per SM: use wider CTAs
    const size_t per_plane = (size_t)(h->merged ? 19 : 13) * P.mz * P.nxh * 16;
    // zpad + xh: about 11 planes of config 5 per chunk (longer grids, smaller tails)
    const unsigned long long budget = (unsigned long long)(U.chunk_mb ? U.chunk_mb : 3072) << 20;
    long long pc = (long long)(budget / per_plane);
    if (pc < 1) pc = 1;
    if (pc > P.ny) pc = P.ny;
    h->pc = (int)pc;
}

// Lays out the workspace; with base == nullptr only measures.
size_t carve(chan_t* h, char* base) {
    const Plan& P = h->P;
    Carver c{base};
    const size_t F = h->F;
    h->v = c.take<double2>(F); h->phi = c.take<double2>(F); h->omy = c.take<double2>(F);
    h->hv = c.take<double2>(F); h->hg = c.take<double2>(F);
    h->u = c.take<double2>(F); h->w = c.take<double2>(F); h->ox = c.take<double2>(F); h->oz = c.take<double2>(F);
    h->H1 = h->u; h->H2 = h->w; h->H3 = h->ox;
    h->s1_bytes = F > ((size_t)64 << 20) ? F : (10 * F < ((size_t)64 << 20) ? 10 * F : ((size_t)64 << 20));
    h->s1 = c.take<double2>(h->s1_bytes);
    h->z1 = h->s1; h->z2 = h->u; h->facA = h->oz; h->facB = h->v;
    const size_t half = (size_t)h->nm * P.ny;     // doubles in half a field
    h->r1 = (double*)h->ox; h->r2 = h->r1 ? h->r1 + half : nullptr;
    h->r3 = (double*)h->w; h->r4 = h->r3 ? h->r3 + half : nullptr;
    h->coef = c.take<double4>((size_t)h->nm * 32);
    // merged plane launches double-buffer the chunks: two zpad sets; the two 3-field xh sets fit in the 7-field xh
    h->zpad = c.take<double2>((size_t)(h->merged ? 12 : 6) * h->pc * P.mz * P.nxh * 16);
    h->xh = c.take<double2>((size_t)7 * h->pc * P.mz * P.nxh * 16);
    const size_t ny8 = (size_t)P.ny * 8;
    h->U = c.take<double>(ny8); h->W = c.take<double>(ny8); h->H1p = c.take<double>(ny8); h->H3p = c.take<double>(ny8);
    h->meanwork = c.take<double>(ny8 * 8);
    h->scal = c.take<double>(64);
    h->stats = c.take<double>((size_t)10 * P.ny * 8);
    for (int o = 0; o < 2; ++o) for (int k = 0; k < 4; ++k) h->tab[o][k] = c.take<double>(ny8 * 8);
    h->kx = c.take<double>((size_t)P.nxh * 8); h->kz = c.take<double>((size_t)P.nz * 8);
    h->wm = c.take<double>(ny8); h->wp = c.take<double>(ny8); h->wq = c.take<double>(ny8);
    h->twx = c.take<double2>(P.fx.tw.size() * 8); h->twz = c.take<double2>(P.fz.tw.size() * 8);
    return c.off;
}

bool ck(chan_t* h, cudaError_t e) {
    if (e != cudaSuccess) { h->cuda_err = (int)e; return false; }
    return true;
}
#define CK(x) do { if (!ck(h, (x))) return CHAN_ECUDA; } while (0)
void prof_mark(chan_t* h, int kc, bool begin) {
    if (!h->prof_on) return;
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return;
    cudaEventRecord(e, h->stream);
    h->prof_ev.push_back(e);
    if (begin) h->prof_cls.push_back(kc);
}
#define PB(kc) prof_mark(h, (kc), true)
#define LAUNCHED() do { ++h->launches; prof_mark(h, 0, false); if (!ck(h, cudaGetLastError())) return CHAN_ECUDA; } while (0)

YParams yparams(const chan_t* h) {
    const Plan& P = h->P;
    YParams Y;
    Y.ny = P.ny; Y.nz = P.nz; Y.nxh = P.nxh; Y.nzh = P.nzh; Y.nm = h->nm;
    for (int o = 0; o < 2; ++o) { Y.t[o].B1 = h->tab[o][0]; Y.t[o].A2 = h->tab[o][1]; Y.t[o].B2 = h->tab[o][2]; Y.t[o].lu1 = h->tab[o][3]; }
    Y.kx = h->kx; Y.kz = h->kz; Y.wm = h->wm; Y.wp = h->wp;
    Y.nu = P.nu; Y.dt = P.dt;
    Y.alpha = P.rk_alpha[h->isub]; Y.beta = P.rk_beta[h->isub]; Y.gamma = P.rk_gamma[h->isub]; Y.zeta = P.rk_zeta[h->isub];
    return Y;
}

PlaneParams pparams(const chan_t* h) {
    const Plan& P = h->P;
    PlaneParams Q;
    Q.ny = P.ny; Q.nz = P.nz; Q.nxh = P.nxh; Q.nzh = P.nzh; Q.mx = P.mx; Q.mz = P.mz; Q.nm = h->nm;
    auto fill = [](FftDev& D, const FftPlan& F, const double2* tw) {
        D.n = F.n; D.ns = (int)F.radix.size();
        for (int s = 0; s < D.ns; ++s) { D.st[s].R = F.radix[s]; D.st[s].m = F.m[s]; D.st[s].tw = tw + F.twoff[s]; }
    };
    fill(Q.fx, P.fx, h->twx);
    fill(Q.fz, P.fz, h->twz);
    return Q;
}

inline unsigned ygrid(const chan_t* h) { return (unsigned)((h->nm + kThreadsY - 1) / kThreadsY); }

inline unsigned sgrid(const chan_t* h) { return (unsigned)((2 * h->nm + YNT - 1) / YNT); }

// a1-a2, second half: zv (in s1) -> u, w, om_x, om_z
int run_derive_tail(chan_t* h) {
    YParams Y = yparams(h);
    PB(CHAN_KC_DERIVE_DOWN); k_se<<<sgrid(h), YNT, 0, h->stream>>>(Y, h->s1, h->omy, h->U, h->W, h->u, h->w, h->oz); LAUNCHED();
    PB(CHAN_KC_DERIVE_UP); k_sf<<<sgrid(h), YNT, 0, h->stream>>>(Y, h->s1, h->oz, h->v, h->ox); LAUNCHED();
    return CHAN_OK;
}
// a1-a2 from the state alone
int run_derive(chan_t* h) {
    YParams Y = yparams(h);
    PB(CHAN_KC_D1FWD); k_sd0<<<sgrid(h), YNT, 0, h->stream>>>(Y, h->v, h->s1); LAUNCHED();
    return run_derive_tail(h);
}

// ---- plan -> kernel dispatch -------------------------------------------------------------------------
// Stage lists with kernels specialised at compile time (chan_fft.cuh k_*_s); any other list of a 2^a 3^b
// length runs the generic kernels (k_*_g).  z lists: up to four radices; x lists: up to three radices in
// front of the fused radix (4 or 8).
#define CHAN_ZPLANS(X) X(6, 1, 1, 1) X(12, 1, 1, 1) X(6, 4, 1, 1) X(6, 8, 1, 1) X(12, 6, 1, 1) X(12, 8, 1, 1) X(12, 12, 1, 1) \
    X(6, 8, 4, 1) X(6, 6, 8, 1) X(6, 8, 8, 1) X(12, 6, 8, 1) X(12, 8, 8, 1) X(12, 12, 6, 1) X(12, 12, 8, 1) X(12, 12, 12, 1) \
    X(6, 8, 8, 4) X(6, 6, 8, 8) X(6, 8, 8, 8)
#define CHAN_ZPLANS_C(X) X(12, 12, 12, 1) X(6, 8, 8, 4) X(12, 12, 6, 1) X(12, 6, 1, 1) X(6, 8, 1, 1)
#define CHAN_XPLANS(X) X(4, 6, 1, 1) X(4, 12, 1, 1) X(4, 6, 4, 1) X(4, 6, 6, 1) X(4, 6, 8, 1) X(4, 12, 8, 1) X(4, 6, 6, 4) X(4, 6, 6, 6) \
    X(4, 6, 8, 4) X(4, 6, 6, 8) X(4, 6, 8, 8) X(4, 12, 6, 6) X(4, 12, 6, 8) X(4, 12, 8, 8) X(8, 6, 1, 1) X(8, 12, 1, 1) X(8, 12, 6, 1) \
    X(8, 12, 12, 1) X(8, 6, 8, 1) X(8, 12, 16, 1) X(8, 18, 16, 1) X(8, 18, 1, 1) X(8, 16, 1, 1) X(8, 12, 8, 1) X(8, 6, 6, 1) X(8, 6, 6, 8) X(8, 6, 8, 4) X(8, 6, 8, 8) X(8, 12, 6, 8)

// (z list | fused x radix, x list) pairs of config 5, 4, 3, of the "mid" parity case and of config 1
#define CHAN_MERGED_PLANS(X) X(12, 12, 12, 1, 8, 6, 6, 8) X(12, 12, 12, 1, 8, 18, 16, 1) X(6, 8, 8, 4, 8, 12, 16, 1) X(12, 12, 6, 1, 8, 12, 12, 1) X(12, 6, 1, 1, 8, 18, 1, 1) \
    X(6, 8, 1, 1, 8, 6, 1, 1)

typedef void (*zinv_fn)(PlaneParams, FieldPtrs, int, int, double2*, int);
typedef void (*zfwd_fn)(PlaneParams, const double2*, int, int, int, FieldPtrsW, double, int, int, int, int);
typedef void (*xprod_fn)(PlaneParams, const double2*, int, double2*, int);

bool same_list(const std::vector<int>& v, int n, const int* r) {
    int cnt = 0;
    for (int k = 0; k < n; ++k) if (r[k] > 1) ++cnt;
    if ((int)v.size() != cnt) return false;
    for (int k = 0; k < cnt; ++k) if (v[k] != r[k]) return false;
    return true;
}
void pick_kernels(chan_t* h) {
    const Plan& P = h->P;
    h->kzinv = k_zfft_inv_g; h->kzfwd = k_zfft_fwd_g;
    h->zspecial = false;
#define X(a, b, c, d) { const int r[4] = {a, b, c, d}; if (same_list(P.fz.radix, 4, r)) { h->kzinv = k_zfft_inv_s<a, b, c, d>; h->kzfwd = k_zfft_fwd_s<a, b, c, d>; h->zspecial = true; } }
    CHAN_ZPLANS(X)
#undef X
    const int F = P.fx.radix.back();
    h->kx3 = (F == 8) ? k_xfft_prod_g<3, 8> : k_xfft_prod_g<3, 4>;
    h->kx7 = (F == 8) ? k_xfft_prod_g<7, 8> : k_xfft_prod_g<7, 4>;
    h->xspecial = false;
    {
        std::vector<int> head(P.fx.radix.begin(), P.fx.radix.end() - 1);
        if (head.empty() && F == 4) { h->kx3 = k_xfft_prod_s<3, 4, 1, 1, 1>; h->kx7 = k_xfft_prod_s<7, 4, 1, 1, 1>; h->xspecial = true; }
        if (head.empty() && F == 8) { h->kx3 = k_xfft_prod_s<3, 8, 1, 1, 1>; h->kx7 = k_xfft_prod_s<7, 8, 1, 1, 1>; h->xspecial = true; }
#define X(f, a, b, c) { const int r[3] = {a, b, c}; if (F == f && same_list(head, 3, r)) { h->kx3 = k_xfft_prod_s<3, f, a, b, c>; h->kx7 = k_xfft_prod_s<7, f, a, b, c>; h->xspecial = true; } }
        CHAN_XPLANS(X)
#undef X
    }
    // cluster z kernels: compiled for the z lists of the benchmark shapes and of the small parity cases
    h->kzinv_c = nullptr; h->kzfwd_c = nullptr;
#define X(a, b, c, d) { const int r[4] = {a, b, c, d}; if (same_list(P.fz.radix, 4, r)) { h->kzinv_c = k_zfft_inv_c<a, b, c, d>; h->kzfwd_c = k_zfft_fwd_c<a, b, c, d>; } }
    CHAN_ZPLANS_C(X)
#undef X
    // merged plane kernel: compiled for the (z list, x list) pairs of the benchmark shapes only (each pair is one more
    // instantiation of all three bodies); any other plan runs the three kernels one after the other
    h->kmerged = nullptr;
    {
        std::vector<int> head(P.fx.radix.begin(), P.fx.radix.end() - 1);
#define X(z0, z1, z2, z3, f, x0, x1, x2) { const int rz[4] = {z0, z1, z2, z3}; const int rx[3] = {x0, x1, x2}; \
        if (F == f && same_list(P.fz.radix, 4, rz) && same_list(head, 3, rx)) h->kmerged = k_planes_s<z0, z1, z2, z3, f, x0, x1, x2>; }
        CHAN_MERGED_PLANS(X)
#undef X
    }
}

size_t merged_smem(const chan_t* h) {
    const size_t a = (size_t)3 * h->P.mx * 16, b = (size_t)h->P.mz * h->Tz * 16;
    return a > b ? a : b;
}

int zinv(chan_t* h, const PlaneParams& Q, const FieldPtrs& in, int nf, int j0, int npl) {
    if (h->zcluster) {
        const int T = h->Tzc;
        dim3 g(2 * ((Q.nxh + T - 1) / T), npl, nf);
        PB(CHAN_KC_ZFFT_INV); h->kzinv_c<<<g, 256, (size_t)Q.mz * T * 8, h->stream>>>(Q, in, j0, npl, h->zpad, T); LAUNCHED();
        return CHAN_OK;
    }
    const int T = h->Tz;
    const size_t sm = (size_t)Q.mz * T * 16;
    dim3 g((Q.nxh + T - 1) / T, npl, nf);
    PB(CHAN_KC_ZFFT_INV); h->kzinv<<<g, h->zthreads, sm, h->stream>>>(Q, in, j0, npl, h->zpad, T); LAUNCHED();
    return CHAN_OK;
}
int zfwd(chan_t* h, const PlaneParams& Q, int pin, int nf, int j0, int npl, const FieldPtrsW& out, double scale, int filt, int kxc, int kzc) {
    if (h->zcluster) {
        const int T = h->Tzc;
        dim3 g(2 * ((pin + T - 1) / T), npl, nf);
        PB(filt ? CHAN_KC_ZFFT_FWD_FILTER : CHAN_KC_ZFFT_FWD);
        h->kzfwd_c<<<g, 256, (size_t)Q.mz * T * 8, h->stream>>>(Q, h->xh, pin, j0, npl, out, scale, filt, kxc, kzc, T); LAUNCHED();
        return CHAN_OK;
    }
    const int T = h->Tz;
    const size_t sm = (size_t)Q.mz * T * 16;
    dim3 g((pin + T - 1) / T, npl, nf);
    PB(filt ? CHAN_KC_ZFFT_FWD_FILTER : CHAN_KC_ZFFT_FWD);
    h->kzfwd<<<g, h->zthreads, sm, h->stream>>>(Q, h->xh, pin, j0, npl, out, scale, filt, kxc, kzc, T); LAUNCHED();
    return CHAN_OK;
}
int xprod(chan_t* h, const PlaneParams& Q, int nprod, int npl, int pout) {
    xprod_fn fn = (nprod == 3) ? h->kx3 : h->kx7;
    const size_t smx = (size_t)(nprod == 3 ? 3 : 4) * Q.mx * 16;
    dim3 g(Q.mz, npl);
    PB(nprod == 3 ? CHAN_KC_XFFT_PROD : CHAN_KC_XFFT_PROD_FILTER);
    int nt = h->xthreads;
    if (nprod == 7 && h->xspecial && 2 * (smx + 1024) > 227 * 1024) nt = 512;    // one CTA per SM: fill it
    fn<<<g, nt, smx, h->stream>>>(Q, h->zpad, npl, h->xh, pout);
    LAUNCHED();
    return CHAN_OK;
}

// a3-a8 (nprod = 3) or the product part of a13 (nprod = 7)
int run_planes(chan_t* h, int nprod, const FieldPtrsW& out, int kxc, int kzc) {
    const Plan& P = h->P;
    PlaneParams Q = pparams(h);
    FieldPtrs in;
    in.f[0] = h->u; in.f[1] = h->v; in.f[2] = h->w; in.f[3] = h->ox; in.f[4] = h->omy; in.f[5] = h->oz;
    const int pout = (nprod == 3) ? P.nxh : kxc + 1;
    const double scale = 1.0 / ((double)P.mx * (double)P.mz);
    for (int j0 = 0; j0 < P.ny; j0 += h->pc) {
        const int npl = (P.ny - j0 < h->pc) ? P.ny - j0 : h->pc;
        int rc = zinv(h, Q, in, 6, j0, npl);
        if (rc) return rc;
        if ((rc = xprod(h, Q, nprod, npl, pout))) return rc;
        rc = zfwd(h, Q, pout, nprod, j0, npl, out, scale, nprod == 7 ? 1 + h->out_f32 : 0, kxc, kzc);
        if (rc) return rc;
    }
    return CHAN_OK;
}

// a3-a8 and the product part of a13 from the SAME z-padded chunks: the filter of the state a substep starts from
// costs no inverse z sweep of its own
int run_planes_both(chan_t* h, const FieldPtrsW& outH, const FieldPtrsW& outF, int kxc, int kzc) {
    const Plan& P = h->P;
    PlaneParams Q = pparams(h);
    FieldPtrs in;
    in.f[0] = h->u; in.f[1] = h->v; in.f[2] = h->w; in.f[3] = h->ox; in.f[4] = h->omy; in.f[5] = h->oz;
    const double scale = 1.0 / ((double)P.mx * (double)P.mz);
    for (int j0 = 0; j0 < P.ny; j0 += h->pc) {
        const int npl = (P.ny - j0 < h->pc) ? P.ny - j0 : h->pc;
        int rc = zinv(h, Q, in, 6, j0, npl);
        if (rc) return rc;
        // the filter products first: its z pass reads the small xh, then the H pass overwrites xh and (later) u, w, om_x
        if ((rc = xprod(h, Q, 7, npl, kxc + 1))) return rc;
        if ((rc = zfwd(h, Q, kxc + 1, 7, j0, npl, outF, scale, 1 + h->out_f32, kxc, kzc))) return rc;
        if ((rc = xprod(h, Q, 3, npl, P.nxh))) return rc;
        if ((rc = zfwd(h, Q, P.nxh, 3, j0, npl, outH, scale, 0, 0, 0))) return rc;
    }
    return CHAN_OK;
}

// a3-a8 through the merged kernel: launch t carries K2 of chunk t, K3 of chunk t-1 and K4 of chunk t-2 (chan_fft.cuh);
// chunk c uses zpad set c&1 and xh set c&1
int run_planes_merged(chan_t* h, const FieldPtrsW& out) {
    const Plan& P = h->P;
    PlaneParams Q = pparams(h);
    const int pc = h->pc, nch = (P.ny + pc - 1) / pc, T = h->Tz;
    const size_t zset = (size_t)6 * pc * P.mz * P.nxh, xset = (size_t)3 * pc * P.mz * P.nxh;
    auto planes_of = [&](int c) { return (P.ny - c * pc < pc) ? P.ny - c * pc : pc; };
    const size_t sm = merged_smem(h);
    for (int t = 0; t < nch + 2; ++t) {
        MergedArgs A = {};
        A.T = T; A.tiles = (unsigned)((P.nxh + T - 1) / T); A.scale = 1.0 / ((double)P.mx * (double)P.mz);
        A.in.f[0] = h->u; A.in.f[1] = h->v; A.in.f[2] = h->w; A.in.f[3] = h->ox; A.in.f[4] = h->omy; A.in.f[5] = h->oz;
        A.out = out;
        if (t < nch) { A.j2 = t * pc; A.npl2 = planes_of(t); A.zw = h->zpad + (size_t)(t & 1) * zset; A.n2 = A.tiles * (unsigned)A.npl2 * 6u; }
        if (t >= 1 && t <= nch) {
            const int c = t - 1;
            A.npl3 = planes_of(c); A.zr = h->zpad + (size_t)(c & 1) * zset; A.xw = h->xh + (size_t)(c & 1) * xset; A.n3 = (unsigned)P.mz * (unsigned)A.npl3;
        }
        if (t >= 2) { const int c = t - 2; A.j4 = c * pc; A.npl4 = planes_of(c); A.xr = h->xh + (size_t)(c & 1) * xset; A.n4 = A.tiles * (unsigned)A.npl4 * 3u; }
        PB(CHAN_KC_PLANES_MERGED); h->kmerged<<<A.n2 + A.n3 + A.n4, 256, sm, h->stream>>>(Q, A); LAUNCHED();
    }
    return CHAN_OK;
}

int run_nonlinear(chan_t* h) {
    FieldPtrsW out;
    out.f[0] = h->H1; out.f[1] = h->H2; out.f[2] = h->H3;
    return h->merged ? run_planes_merged(h, out) : run_planes(h, 3, out, 0, 0);
}

// a9-a12
int run_ysolve(chan_t* h) {
    const Plan& P = h->P;
    YParams Y = yparams(h);
    MeanParams M;
    M.ny = P.ny; M.nm = h->nm; M.A2 = h->tab[0][1]; M.B2 = h->tab[0][2]; M.wq = h->wq; M.wm = h->wm; M.wp = h->wp;
    M.nu = P.nu; M.dt = P.dt; M.alpha = Y.alpha; M.beta = Y.beta; M.gamma = Y.gamma; M.zeta = Y.zeta; M.forcing = P.forcing;
    const size_t smm = (size_t)15 * P.ny * 8;
    PB(CHAN_KC_MEAN); k_mean<<<1, 256, smm, h->stream>>>(M, h->H1, h->H3, h->U, h->W, h->H1p, h->H3p, h->scal); LAUNCHED();
    // buffers that are dead during the y-phase carry its scratch:
    // s1: zd -> z_phi -> phi_p -> zv;  oz: R_om -> z_om -> z_vab;  u, ox: factor rows (H1, H3 are consumed by SA);
    // w: z_vp (H2 is consumed by SB);  v: phi_ab, then the new v in place
    const unsigned g = sgrid(h);
    PB(CHAN_KC_Y1); k_sa<<<g, YNT, 0, h->stream>>>(Y, h->H1, h->H3, h->omy, h->hg, h->s1, h->oz); LAUNCHED();
    PB(CHAN_KC_Y2); k_sb<<<g, YNT, 0, h->stream>>>(Y, h->H2, h->phi, h->hv, h->s1, h->oz, h->u, h->ox); LAUNCHED();
    PB(CHAN_KC_Y3); k_sc<<<g, YNT, 0, h->stream>>>(Y, h->u, h->ox, h->oz, h->s1, h->omy, h->v, h->w, h->coef); LAUNCHED();
    PB(CHAN_KC_Y4); k_sd<<<g, YNT, 0, h->stream>>>(Y, h->u, h->ox, h->w, h->oz, h->s1, h->v, h->coef, h->phi); LAUNCHED();
    return CHAN_OK;
}

int transpose(chan_t* h, int dir, const double2* in, double2* out) {
    const long long nm = h->nm;
    const int ny = h->P.ny;
    // the mode dimension (up to 2^31 / 32 tiles) always on gridDim.x, the y dimension on gridDim.y
    dim3 g((unsigned)((nm + 31) / 32), (unsigned)((ny + 31) / 32));
    PB(CHAN_KC_TRANSPOSE); k_transpose<<<g, 256, 0, h->stream>>>(in, out, nm, ny, dir); LAUNCHED();
    return CHAN_OK;
}

double2* field_ptr(const chan_t* h, int f) {
    switch (f) {
        case CHAN_F_V: return h->v; case CHAN_F_PHI: return h->phi; case CHAN_F_OMY: return h->omy;
        case CHAN_F_U: return h->u; case CHAN_F_W: return h->w; case CHAN_F_OMX: return h->ox; case CHAN_F_OMZ: return h->oz;
        case CHAN_F_H1: return h->H1; case CHAN_F_H2: return h->H2; case CHAN_F_H3: return h->H3;
        case CHAN_F_HV_PREV: return h->hv; case CHAN_F_HG_PREV: return h->hg;
        default: return nullptr;
    }
}

// tiling, kernel dispatch, size limits and workspace layout for the current plan and tuning overrides
int configure(chan_t* h) {
    if ((int)h->P.fx.radix.size() > CHAN_MAX_STAGES || (int)h->P.fz.radix.size() > CHAN_MAX_STAGES) return CHAN_EINVAL;
    pick_kernels(h);
    if (h->tune.plane_overlap == 2 && !h->kmerged) return CHAN_EINVAL;
    h->merged = h->kmerged && h->tune.plane_overlap == 2;   // measured on config 5: no gain over separate launches, so opt-in
    choose_tiling(h);
    if (h->tune.z_cluster == 2 && !h->zcluster) return CHAN_EINVAL;
    if ((size_t)4 * h->P.mx * 16 > 220 * 1024 || (size_t)h->P.mz * h->Tz * 16 > 220 * 1024) return CHAN_EINVAL;
    if ((size_t)15 * h->P.ny * 8 > 220 * 1024) return CHAN_EINVAL;   // mean-mode solve lives in shared memory
    h->need = carve(h, nullptr);
    return CHAN_OK;
}

// second half of chan_set_state: v, phi, om_y are in place (plane layout)
int finish_set_state(chan_t* h, const double* dU, const double* dW) {
    const Plan& P = h->P;
    // the (0,0) mode and the z-Nyquist slot are not part of the state (reading R2)
    for (double2* f : {h->v, h->phi, h->omy}) {
        CK(cudaMemset2DAsync(f, (size_t)h->nm * 16, 0, 16, P.ny, h->stream));
        CK(cudaMemset2DAsync(f + (size_t)P.nzh * P.nxh, (size_t)h->nm * 16, 0, (size_t)P.nxh * 16, P.ny, h->stream));
    }
    CK(cudaMemcpyAsync(h->U, dU, (size_t)P.ny * 8, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemcpyAsync(h->W, dW, (size_t)P.ny * 8, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemsetAsync(h->hv, 0, h->F, h->stream)); CK(cudaMemsetAsync(h->hg, 0, h->F, h->stream));
    CK(cudaMemsetAsync(h->H1p, 0, (size_t)P.ny * 8, h->stream)); CK(cudaMemsetAsync(h->H3p, 0, (size_t)P.ny * 8, h->stream));
    PB(CHAN_KC_MEAN); k_flux<<<1, 32, 0, h->stream>>>(P.ny, h->wq, h->U, h->scal); LAUNCHED();
    h->isub = 0; h->have_state = true;
    return run_derive(h);
}

}  // namespace

extern "C" {

int chan_create(chan_t** out, const chan_grid_t* grid, const chan_box_t* box, double re_tau, double dt, const chan_opts_t* opts) {
    if (!out || !grid || !box) return CHAN_EINVAL;
    *out = nullptr;
    chan_t* h = new (std::nothrow) chan();
    if (!h) return CHAN_ENOSPACE;
    const int hl = opts ? opts->lhs_halfwidth : 3, hr = opts ? opts->rhs_halfwidth : 3, fo = opts ? opts->forcing : 0;
    int rc = build_plan(h->P, grid->nx, grid->ny, grid->nz, box->lx, box->lz, box->y, re_tau, dt, hl ? hl : 3, hr ? hr : 3, fo);
    if (rc != CHAN_OK) { delete h; return rc; }
    h->nm = (long long)h->P.nz * h->P.nxh;
    h->F = (size_t)h->nm * h->P.ny * 16;
    if ((rc = configure(h)) != CHAN_OK) { delete h; return rc; }
    *out = h;
    return CHAN_OK;
}

int chan_debug_set_tuning(chan_t* h, const chan_tuning_t* t) {
    if (!h || !t) return CHAN_EINVAL;
    if (h->bound) return CHAN_ESTATE;
    for (int r : t->reserved) if (r) return CHAN_EINVAL;
    auto pow2 = [](int v) { return v == 1 || v == 2 || v == 4 || v == 8 || v == 16; };
    if ((t->xfuse && t->xfuse != 4 && t->xfuse != 8) || (t->maxradix_z && (t->maxradix_z < 2 || t->maxradix_z > 12)) ||
        (t->maxradix_x && (t->maxradix_x < 2 || t->maxradix_x > 18)) || (t->tz && !pow2(t->tz)) ||
        (t->zthreads && (t->zthreads < 32 || t->zthreads > 256 || t->zthreads % 32)) || (t->xthreads && (t->xthreads < 32 || t->xthreads > CHAN_XNT)) ||
        t->chunk_mb < 0 || t->plane_overlap < 0 || t->plane_overlap > 2 || t->z_cluster < 0 || t->z_cluster > 2)
        return CHAN_EINVAL;
    const chan_tuning_t old = h->tune;
    const FftPlan ofx = h->P.fx, ofz = h->P.fz;
    h->tune = *t;
    int rc = plan_ffts(h->P, t->xfuse, t->maxradix_z, t->maxradix_x);
    if (rc == CHAN_OK) rc = configure(h);
    if (rc != CHAN_OK) { h->tune = old; h->P.fx = ofx; h->P.fz = ofz; configure(h); }
    return rc;
}

int chan_debug_get_tuning(const chan_t* h, chan_tuning_t* out) {
    if (!h || !out) return CHAN_EINVAL;
    *out = chan_tuning_t{};
    out->xfuse = h->P.fx.radix.back();
    for (int r : h->P.fz.radix) out->maxradix_z = r > out->maxradix_z ? r : out->maxradix_z;
    for (size_t k = 0; k + 1 < h->P.fx.radix.size(); ++k) out->maxradix_x = h->P.fx.radix[k] > out->maxradix_x ? h->P.fx.radix[k] : out->maxradix_x;
    out->tz = h->Tz; out->zthreads = h->zthreads; out->xthreads = h->xthreads;
    out->chunk_mb = h->tune.chunk_mb ? h->tune.chunk_mb : 3072;
    out->planes_per_chunk = h->pc;
    out->plane_overlap = h->merged ? 2 : 1;
    out->z_cluster = h->zcluster ? 2 : 1;
    if (h->zcluster) out->tz = h->Tzc;
    return CHAN_OK;
}

int chan_destroy(chan_t* h) {
    if (h) for (cudaEvent_t e : h->prof_ev) cudaEventDestroy(e);
    delete h;
    return CHAN_OK;
}

size_t chan_workspace_bytes(const chan_t* h) { return h ? h->need : 0; }

int chan_bind(chan_t* h, void* dev_workspace, size_t bytes, void* cuda_stream) {
    if (!h || !dev_workspace) return CHAN_EINVAL;
    if (bytes < h->need) return CHAN_ENOSPACE;
    if ((uintptr_t)dev_workspace % kAlign) return CHAN_EINVAL;
    h->ws = (char*)dev_workspace; h->ws_bytes = bytes; h->stream = (cudaStream_t)cuda_stream;
    carve(h, h->ws);
    const Plan& P = h->P;
    CK(cudaMemsetAsync(h->ws, 0, h->need, h->stream));
    auto upl = [&](void* d, const void* s, size_t n) { return cudaMemcpyAsync(d, s, n, cudaMemcpyHostToDevice, h->stream); };
    for (int o = 0; o < 2; ++o) {
        CK(upl(h->tab[o][0], P.ot[o].B1.data(), P.ot[o].B1.size() * 8));
        CK(upl(h->tab[o][1], P.ot[o].A2.data(), P.ot[o].A2.size() * 8));
        CK(upl(h->tab[o][2], P.ot[o].B2.data(), P.ot[o].B2.size() * 8));
        CK(upl(h->tab[o][3], P.ot[o].lu1.data(), P.ot[o].lu1.size() * 8));
    }
    CK(upl(h->kx, P.kx.data(), P.kx.size() * 8)); CK(upl(h->kz, P.kz.data(), P.kz.size() * 8));
    CK(upl(h->wm, P.wm.data(), P.wm.size() * 8)); CK(upl(h->wp, P.wp.data(), P.wp.size() * 8));
    CK(upl(h->wq, P.wq.data(), P.wq.size() * 8));
    CK(upl(h->twx, P.fx.tw.data(), P.fx.tw.size() * 8)); CK(upl(h->twz, P.fz.tw.data(), P.fz.tw.size() * 8));
    CK(cudaStreamSynchronize(h->stream));   // the host vectors may not outlive the copies otherwise
    // dynamic shared memory of the kernels this handle dispatches to, once (not per launch)
    CK(cudaFuncSetAttribute((const void*)h->kzinv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)P.mz * h->Tz * 16)));
    CK(cudaFuncSetAttribute((const void*)h->kzfwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)P.mz * h->Tz * 16)));
    CK(cudaFuncSetAttribute((const void*)h->kx3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)3 * P.mx * 16)));
    CK(cudaFuncSetAttribute((const void*)h->kx7, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)4 * P.mx * 16)));
    CK(cudaFuncSetAttribute(k_mean, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)15 * P.ny * 8)));
    if (h->zcluster) {
        CK(cudaFuncSetAttribute((const void*)h->kzinv_c, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)P.mz * h->Tzc * 8)));
        CK(cudaFuncSetAttribute((const void*)h->kzfwd_c, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)P.mz * h->Tzc * 8)));
    }
    if (h->merged) CK(cudaFuncSetAttribute((const void*)h->kmerged, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)merged_smem(h)));
    h->bound = true; h->have_state = false; h->isub = 0; h->nsamples = 0;
    return CHAN_OK;
}

int chan_set_state(chan_t* h, const void* dv, const void* dphi, const void* domy, const double* dU, const double* dW) {
    if (!h || !dv || !dphi || !domy || !dU || !dW) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    int rc;
    if ((rc = transpose(h, 0, (const double2*)dv, h->v))) return rc;
    if ((rc = transpose(h, 0, (const double2*)dphi, h->phi))) return rc;
    if ((rc = transpose(h, 0, (const double2*)domy, h->omy))) return rc;
    return finish_set_state(h, dU, dW);
}

int chan_get_state(const chan_t* hc, void* dv, void* dphi, void* domy, double* dU, double* dW) {
    chan_t* h = const_cast<chan_t*>(hc);
    if (!h || !dv || !dphi || !domy || !dU || !dW) return CHAN_EINVAL;
    if (!h->bound || !h->have_state) return CHAN_ESTATE;
    int rc;
    if ((rc = transpose(h, 1, h->v, (double2*)dv))) return rc;
    if ((rc = transpose(h, 1, h->phi, (double2*)dphi))) return rc;
    if ((rc = transpose(h, 1, h->omy, (double2*)domy))) return rc;
    CK(cudaMemcpyAsync(dU, h->U, (size_t)h->P.ny * 8, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemcpyAsync(dW, h->W, (size_t)h->P.ny * 8, cudaMemcpyDeviceToDevice, h->stream));
    return CHAN_OK;
}

// Host state in: each field goes host -> s1 (scratch field, idle between substeps) -> transposed into place, one after the
// other on the bound stream; the tail of chan_set_state (Nyquist/mean slots, history, mass flux, a1) follows.
int chan_set_state_host(chan_t* h, const void* hv, const void* hphi, const void* homy, const double* hU, const double* hW) {
    if (!h || !hv || !hphi || !homy || !hU || !hW) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    double2* dst[3] = {h->v, h->phi, h->omy};
    const void* src[3] = {hv, hphi, homy};
    int rc;
    for (int k = 0; k < 3; ++k) {
        CK(cudaMemcpyAsync(h->s1, src[k], h->F, cudaMemcpyHostToDevice, h->stream));
        if ((rc = transpose(h, 0, h->s1, dst[k]))) return rc;
    }
    CK(cudaMemcpyAsync(h->meanwork, hU, (size_t)h->P.ny * 8, cudaMemcpyHostToDevice, h->stream));
    CK(cudaMemcpyAsync(h->meanwork + h->P.ny, hW, (size_t)h->P.ny * 8, cudaMemcpyHostToDevice, h->stream));
    if ((rc = finish_set_state(h, h->meanwork, h->meanwork + h->P.ny))) return rc;
    CK(cudaStreamSynchronize(h->stream));     // the host buffers are the caller's again when this returns (chan.h)
    return CHAN_OK;
}

int chan_get_state_host(chan_t* h, void* hv, void* hphi, void* homy, double* hU, double* hW) {
    if (!h || !hv || !hphi || !homy || !hU || !hW) return CHAN_EINVAL;
    if (!h->bound || !h->have_state) return CHAN_ESTATE;
    double2* src[3] = {h->v, h->phi, h->omy};
    void* dst[3] = {hv, hphi, homy};
    int rc;
    for (int k = 0; k < 3; ++k) {
        if ((rc = transpose(h, 1, src[k], h->s1))) return rc;
        CK(cudaMemcpyAsync(dst[k], h->s1, h->F, cudaMemcpyDeviceToHost, h->stream));
    }
    CK(cudaMemcpyAsync(hU, h->U, (size_t)h->P.ny * 8, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaMemcpyAsync(hW, h->W, (size_t)h->P.ny * 8, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return CHAN_OK;
}

int chan_substep(chan_t* h) {
    if (!h) return CHAN_EINVAL;
    if (!h->bound || !h->have_state) return CHAN_ESTATE;
    int rc;
    if ((rc = run_nonlinear(h))) return rc;
    if ((rc = run_ysolve(h))) return rc;
    h->isub = (h->isub + 1) % 3;
    return run_derive_tail(h);
}

int chan_step(chan_t* h) {
    if (!h) return CHAN_EINVAL;
    if (!h->bound || !h->have_state || h->isub != 0) return CHAN_ESTATE;
    for (int i = 0; i < 3; ++i) { int rc = chan_substep(h); if (rc) return rc; }
    return CHAN_OK;
}

}  // extern "C"

namespace {

// the ten output planes of the filter: three velocity copies, then the seven products through the plane kernels
int filter_args(chan_t* h, int kxc, int kzc, void* dev_out, size_t out_bytes, FieldPtrsW& oF) {
    const Plan& P = h->P;
    if (kxc < 0 || kzc < 0 || kxc > P.nxh - 1 || kzc > P.nzh - 1) return CHAN_EINVAL;
    const size_t per = (size_t)P.ny * (2 * kzc + 1) * (kxc + 1), esz = h->out_f32 ? 8 : 16;
    if (out_bytes < per * 10 * esz) return CHAN_ENOSPACE;
    for (int k = 0; k < 7; ++k) oF.f[k] = (double2*)((char*)dev_out + (size_t)(3 + k) * per * esz);
    PlaneParams Q = pparams(h);
    FieldPtrs in; in.f[0] = h->u; in.f[1] = h->v; in.f[2] = h->w;
    PB(CHAN_KC_FILTER_COPY); k_filter_copy<<<296, 256, 0, h->stream>>>(Q, in, (double2*)dev_out, kxc, kzc, h->out_f32); LAUNCHED();
    return CHAN_OK;
}

int step_filter_impl(chan_t* h, int kxc, int kzc, void* dev_out, size_t out_bytes) {
    FieldPtrsW oF, oH;
    int rc;
    if ((rc = filter_args(h, kxc, kzc, dev_out, out_bytes, oF))) return rc;
    oH.f[0] = h->H1; oH.f[1] = h->H2; oH.f[2] = h->H3;
    if ((rc = run_planes_both(h, oH, oF, kxc, kzc))) return rc;
    if ((rc = run_ysolve(h))) return rc;
    h->isub = 1;
    if ((rc = run_derive_tail(h))) return rc;
    for (int i = 1; i < 3; ++i) if ((rc = chan_substep(h))) return rc;
    return CHAN_OK;
}

}  // namespace

extern "C" {

int chan_filter_store(chan_t* h, int kxc, int kzc, void* dev_out, size_t out_bytes) {
    if (!h || !dev_out) return CHAN_EINVAL;
    if (!h->bound || !h->have_state) return CHAN_ESTATE;
    FieldPtrsW o;
    int rc = filter_args(h, kxc, kzc, dev_out, out_bytes, o);
    if (rc) return rc;
    return run_planes(h, 7, o, kxc, kzc);
}

int chan_step_filter(chan_t* h, int kxc, int kzc, void* dev_out, size_t out_bytes) {
    if (!h || !dev_out) return CHAN_EINVAL;
    if (!h->bound || !h->have_state || h->isub != 0) return CHAN_ESTATE;
    return step_filter_impl(h, kxc, kzc, dev_out, out_bytes);
}

int chan_filter_store_host(chan_t* h, int kxc, int kzc, void* host_out, size_t out_bytes) {
    if (!h || !host_out) return CHAN_EINVAL;
    if (!h->bound || !h->have_state) return CHAN_ESTATE;
    const Plan& P = h->P;
    if (kxc < 0 || kzc < 0 || kxc > P.nxh - 1 || kzc > P.nzh - 1) return CHAN_EINVAL;
    const size_t bytes = (size_t)P.ny * (2 * kzc + 1) * (kxc + 1) * 10 * (h->out_f32 ? 8 : 16);
    if (out_bytes < bytes) return CHAN_ENOSPACE;
    // staged in the y-phase scratch field s1 (idle between substeps): at most one field's worth of output
    if (bytes > h->s1_bytes) return CHAN_ENOSPACE;
    int rc = chan_filter_store(h, kxc, kzc, h->s1, bytes);
    if (rc) return rc;
    CK(cudaMemcpyAsync(host_out, h->s1, bytes, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return CHAN_OK;
}

int chan_set_filter_precision(chan_t* h, int bytes_per_real) {
    if (!h || (bytes_per_real != 4 && bytes_per_real != 8)) return CHAN_EINVAL;
    h->out_f32 = (bytes_per_real == 4);
    return CHAN_OK;
}

int chan_run(chan_t* h, const chan_run_t* r, long long* snapshots) {
    if (!h || !r) return CHAN_EINVAL;
    if (!h->bound || !h->have_state || h->isub != 0) return CHAN_ESTATE;
    if (r->nsteps < 0 || r->filter_every < 0 || r->stats_every < 0) return CHAN_EINVAL;
    if (r->filter_every > 0 && (!r->dev_ring || r->ring_slots < 1)) return CHAN_EINVAL;
    long long emitted = 0;
    for (int n = 0; n < r->nsteps; ++n) {
        int rc;
        const bool st = r->stats_every > 0 && n % r->stats_every == 0, fl = r->filter_every > 0 && n % r->filter_every == 0;
        // statistics of a step that also emits an fp64 database come out of that database's (0,0) modes
        const bool st_db = st && fl && !h->out_f32;
        if (st && !st_db && (rc = chan_stats(h, CHAN_STATS_ACCUMULATE, nullptr, nullptr))) return rc;
        if (fl) {
            char* slot = (char*)r->dev_ring + (size_t)(emitted % r->ring_slots) * r->slot_bytes;
            if ((rc = step_filter_impl(h, r->kx_cut, r->kz_cut, slot, r->slot_bytes))) return rc;
            if (st_db) {
                const size_t plane = (size_t)(2 * r->kz_cut + 1) * (r->kx_cut + 1);
                PB(CHAN_KC_STATS); k_stats_from_db<<<(10 * h->P.ny + 255) / 256, 256, 0, h->stream>>>(h->P.ny, plane, (const double2*)slot, h->stats); LAUNCHED();
                ++h->nsamples;
            }
            ++emitted;
        } else if ((rc = chan_step(h))) return rc;
    }
    if (snapshots) *snapshots = emitted;
    return CHAN_OK;
}

int chan_stats(chan_t* h, int flags, double* host_out, long long* nsamples) {
    if (!h) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    const Plan& P = h->P;
    if (flags & CHAN_STATS_RESET) {
        CK(cudaMemsetAsync(h->stats, 0, (size_t)10 * P.ny * 8, h->stream));
        h->nsamples = 0;
    }
    if (flags & CHAN_STATS_ACCUMULATE) {
        if (!h->have_state) return CHAN_ESTATE;
        PlaneParams Q = pparams(h);
        FieldPtrs in; in.f[0] = h->u; in.f[1] = h->v; in.f[2] = h->w; in.f[3] = h->ox; in.f[4] = h->omy; in.f[5] = h->oz;
        PB(CHAN_KC_STATS); k_stats<<<P.ny, 256, 0, h->stream>>>(Q, in, h->stats); LAUNCHED();
        ++h->nsamples;
    }
    if (flags & CHAN_STATS_READ) {
        if (!host_out) return CHAN_EINVAL;
        CK(cudaMemcpyAsync(host_out, h->stats, (size_t)10 * P.ny * 8, cudaMemcpyDeviceToHost, h->stream));
        CK(cudaStreamSynchronize(h->stream));
        if (nsamples) *nsamples = h->nsamples;
    }
    return CHAN_OK;
}

int chan_spectra(chan_t* h, double* dev_ex, size_t ex_bytes, double* dev_ez, size_t ez_bytes) {
    if (!h || (!dev_ex && !dev_ez)) return CHAN_EINVAL;
    if (!h->bound || !h->have_state) return CHAN_ESTATE;
    const Plan& P = h->P;
    if ((dev_ex && ex_bytes < (size_t)7 * P.ny * P.nxh * 8) || (dev_ez && ez_bytes < (size_t)7 * P.ny * P.nz * 8)) return CHAN_ENOSPACE;
    PlaneParams Q = pparams(h);
    FieldPtrs in; in.f[0] = h->u; in.f[1] = h->v; in.f[2] = h->w; in.f[3] = h->ox; in.f[4] = h->omy; in.f[5] = h->oz;
    if (dev_ex) { PB(CHAN_KC_STATS); k_spectra_x<<<dim3((P.nxh + 127) / 128, P.ny), 128, 0, h->stream>>>(Q, in, dev_ex); LAUNCHED(); }
    if (dev_ez) { PB(CHAN_KC_STATS); k_spectra_z<<<dim3((P.nz + 7) / 8, P.ny), 256, 0, h->stream>>>(Q, in, dev_ez); LAUNCHED(); }
    return CHAN_OK;
}

int chan_get_scalars(chan_t* h, double* out4) {
    if (!h || !out4) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    CK(cudaMemcpyAsync(out4, h->scal, 32, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return CHAN_OK;
}

int chan_set_pgrad(chan_t* h, double g) {
    if (!h) return CHAN_EINVAL;
    if (!h->bound || h->P.forcing != 1) return CHAN_ESTATE;
    CK(cudaMemcpyAsync(h->scal, &g, 8, cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return CHAN_OK;
}

const char* chan_strerror(int s) {
    switch (s) {
        case CHAN_OK: return "ok";
        case CHAN_EINVAL: return "invalid argument";
        case CHAN_ENOSPACE: return "workspace or output buffer too small";
        case CHAN_ESTATE: return "call out of order";
        case CHAN_ECUDA: return "CUDA error";
        case CHAN_ELIMIT: return "problem larger than the static scratch limit of this entry point";
        default: return "unknown status";
    }
}

int chan_debug_get_field(const chan_t* hc, int field, void* dev_out) {
    chan_t* h = const_cast<chan_t*>(hc);
    if (!h || !dev_out) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    double2* p = field_ptr(h, field);
    if (!p) return CHAN_EINVAL;
    return transpose(h, 1, p, (double2*)dev_out);
}

int chan_debug_set_field(chan_t* h, int field, const void* dev_in) {
    if (!h || !dev_in) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    double2* p = field_ptr(h, field);
    if (!p) return CHAN_EINVAL;
    return transpose(h, 0, (const double2*)dev_in, p);
}

int chan_debug_run_stage(chan_t* h, int stage) {
    if (!h) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    switch (stage) {
        case CHAN_STAGE_DERIVE: return run_derive(h);
        case CHAN_STAGE_NONLINEAR: return run_nonlinear(h);
        case CHAN_STAGE_YSOLVE: return run_ysolve(h);
        default: return CHAN_EINVAL;
    }
}

int chan_debug_set_substep_index(chan_t* h, int i) {
    if (!h || i < 0 || i > 2) return CHAN_EINVAL;
    h->isub = i;
    return CHAN_OK;
}

int chan_debug_get_band_tables(const chan_t* h, double* out) {
    if (!h || !out) return CHAN_EINVAL;
    const size_t n = (size_t)h->P.ny * 7;
    std::memcpy(out, h->P.A1.data(), n * 8); std::memcpy(out + n, h->P.B1.data(), n * 8);
    std::memcpy(out + 2 * n, h->P.A2.data(), n * 8); std::memcpy(out + 3 * n, h->P.B2.data(), n * 8);
    return CHAN_OK;
}

long long chan_debug_launch_count(const chan_t* h) { return h ? h->launches : 0; }

int chan_debug_describe(const chan_t* h, char* buf, size_t n) {
    if (!h || !buf || n == 0) return CHAN_EINVAL;
    std::string s = "x:";
    const auto& rx = h->P.fx.radix; const auto& rz = h->P.fz.radix;
    for (size_t k = 0; k + 1 < rx.size(); ++k) s += (k ? "," : " ") + std::to_string(rx[k]);
    s += " |" + std::to_string(rx.back()) + "  z:";
    for (size_t k = 0; k < rz.size(); ++k) s += (k ? "," : " ") + std::to_string(rz[k]);
    s += "  specialised x/z: " + std::to_string((int)h->xspecial) + "/" + std::to_string((int)h->zspecial);
    s += "  merged plane launches: " + std::to_string((int)h->merged);
    s += "  z cluster: " + std::to_string((int)h->zcluster);
    s += "  tz " + std::to_string(h->zcluster ? h->Tzc : h->Tz) + "  threads x/z " + std::to_string(h->xthreads) + "/" + std::to_string(h->zthreads);
    s += "  planes per chunk " + std::to_string(h->pc);
    std::strncpy(buf, s.c_str(), n - 1);
    buf[n - 1] = 0;
    return CHAN_OK;
}

int chan_debug_profile(chan_t* h, int enable) {
    if (!h) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    if (enable) {
        for (cudaEvent_t e : h->prof_ev) cudaEventDestroy(e);
        h->prof_ev.clear(); h->prof_cls.clear();
    }
    h->prof_on = enable != 0;
    return CHAN_OK;
}

int chan_debug_profile_read(chan_t* h, double* host_ms, long long* host_counts) {
    if (!h || !host_ms || !host_counts) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    CK(cudaStreamSynchronize(h->stream));
    for (int k = 0; k < CHAN_KC_COUNT; ++k) { host_ms[k] = 0.0; host_counts[k] = 0; }
    const size_t n = h->prof_cls.size();
    for (size_t i = 0; i < n && 2 * i + 1 < h->prof_ev.size(); ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, h->prof_ev[2 * i], h->prof_ev[2 * i + 1]) == cudaSuccess) {
            host_ms[h->prof_cls[i]] += ms; host_counts[h->prof_cls[i]] += 1;
        }
    }
    return CHAN_OK;
}

// ---- mesh tools of the paper's section 2.3 (NEXT-4), host only ------------------------------------------------------
int chan_mesh_helmholtz_error(int ny, const double* host_y, double lambda, int nfirst, double* host_err2) {
    return mesh_helmholtz_error(ny, host_y, lambda, nfirst, host_err2);
}
int chan_mesh_optimize(int ny, double* host_y, int npoints, double lambda, double max_shift, int sweeps, double* host_err_before2,
                       double* host_err_after2) {
    return mesh_optimize(ny, host_y, npoints, lambda, max_shift, sweeps, host_err_before2, host_err_after2);
}

// ---- post-processing of a stored database (NEXT-2) -----------------------------------------------------
size_t chan_post_scratch_bytes(const chan_t* h, int kxc, int kzc) {
    if (!h || kxc < 0 || kzc < 0 || kxc > h->P.nxh - 1 || kzc > h->P.nzh - 1) return 0;
    return (size_t)7 * h->P.ny * (2 * kzc + 1) * (kxc + 1) * 16;
}

static int post_check(chan_t* h, int kxc, int kzc, const void* db, const void* out, const void* scratch, size_t sbytes, PostParams& Q) {
    if (!h || !db || !out || !scratch) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    const Plan& P = h->P;
    if (kxc < 0 || kzc < 0 || kxc > P.nxh - 1 || kzc > P.nzh - 1) return CHAN_EINVAL;
    if (sbytes < chan_post_scratch_bytes(h, kxc, kzc)) return CHAN_ENOSPACE;
    Q.ny = P.ny; Q.nr = 2 * kzc + 1; Q.npk = kxc + 1; Q.kzc = kzc; Q.nz = P.nz;
    Q.B1 = h->tab[0][0]; Q.A2 = h->tab[0][1]; Q.B2 = h->tab[0][2]; Q.lu1 = h->tab[0][3];
    Q.kx = h->kx; Q.kz = h->kz; Q.wm = h->wm; Q.wp = h->wp; Q.nu = P.nu;
    return CHAN_OK;
}

int chan_post_pressure(chan_t* h, int kxc, int kzc, const void* dev_db, void* dev_p, void* dev_scratch, size_t scratch_bytes) {
    PostParams Q;
    int rc = post_check(h, kxc, kzc, dev_db, dev_p, dev_scratch, scratch_bytes, Q);
    if (rc) return rc;
    const size_t per = (size_t)Q.ny * Q.nr * Q.npk;
    double2* S = (double2*)dev_scratch;
    const unsigned g = (unsigned)((Q.nr * Q.npk + 127) / 128);
    PB(CHAN_KC_POST); k_post_divdiv<<<g, 128, 0, h->stream>>>(Q, (const double2*)dev_db, S + per, S, 0); LAUNCHED();
    PB(CHAN_KC_POST); k_post_pressure<<<g, 128, 0, h->stream>>>(Q, (const double2*)dev_db, S, S + per, S + 2 * per, S + 3 * per, S + 4 * per, (double2*)dev_p); LAUNCHED();
    return CHAN_OK;
}

int chan_post_strain_norm(chan_t* h, int kxc, int kzc, const void* dev_db, void* dev_out, void* dev_scratch, size_t scratch_bytes) {
    PostParams Q;
    int rc = post_check(h, kxc, kzc, dev_db, dev_out, dev_scratch, scratch_bytes, Q);
    if (rc) return rc;
    const unsigned g = (unsigned)((Q.nr * Q.npk + 127) / 128);
    PB(CHAN_KC_POST); k_post_divdiv<<<g, 128, 0, h->stream>>>(Q, (const double2*)dev_db, (double2*)dev_scratch, (double2*)dev_out, 1); LAUNCHED();
    return CHAN_OK;
}

// ---- the one entry point that needs no caller scratch and allocates nothing ---------------------------------------------
// chan_post_strain_norm with its scratch plane set in a file-scope device array (include/chan.h).  In host code the
// array's name is only a stand-in for the symbol: its device address comes from cudaGetSymbolAddress, asked once per
// device with that device current and kept in a small table.
static __device__ __align__(256) double2 g_chan_static_scratch[CHAN_STATIC_SCRATCH_BYTES / sizeof(double2)];

static int static_scratch_ptr(double2** out) {
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static double2* table[kMaxDev] = {};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDev) return CHAN_ECUDA;
    std::lock_guard<std::mutex> lock(mu);
    if (!table[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_chan_static_scratch) != cudaSuccess || !p) return CHAN_ECUDA;
        table[dev] = (double2*)p;
    }
    *out = table[dev];
    return CHAN_OK;
}

size_t chan_post_strain_norm_static_limit(void) { return (size_t)CHAN_STATIC_SCRATCH_BYTES; }

int chan_post_strain_norm_static(chan_t* h, int kxc, int kzc, const void* dev_db, void* dev_out) {
    if (!h || !dev_db || !dev_out) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    const Plan& P = h->P;
    if (kxc < 0 || kzc < 0 || kxc > P.nxh - 1 || kzc > P.nzh - 1) return CHAN_EINVAL;
    // one complex plane set [ny][2 kzc + 1][kxc + 1] of scratch: beyond the static array, refuse
    if ((size_t)P.ny * (2 * kzc + 1) * (kxc + 1) * sizeof(double2) > (size_t)CHAN_STATIC_SCRATCH_BYTES) return CHAN_ELIMIT;
    double2* scratch = nullptr;
    int rc = static_scratch_ptr(&scratch);
    if (rc) { h->cuda_err = (int)cudaGetLastError(); return rc; }
    PostParams Q;
    Q.ny = P.ny; Q.nr = 2 * kzc + 1; Q.npk = kxc + 1; Q.kzc = kzc; Q.nz = P.nz;
    Q.B1 = h->tab[0][0]; Q.A2 = h->tab[0][1]; Q.B2 = h->tab[0][2]; Q.lu1 = h->tab[0][3];
    Q.kx = h->kx; Q.kz = h->kz; Q.wm = h->wm; Q.wp = h->wp; Q.nu = P.nu;
    // nothing in the scratch has to start at zero: every mode's forward sweep writes its column before the backward
    // sweep reads it (post_d1), so the contents left by the previous call are never read
    const unsigned g = (unsigned)((Q.nr * Q.npk + 127) / 128);
    PB(CHAN_KC_POST); k_post_divdiv<<<g, 128, 0, h->stream>>>(Q, (const double2*)dev_db, scratch, (double2*)dev_out, 1); LAUNCHED();
    return CHAN_OK;
}

int chan_post_sgs(chan_t* h, int kxc, int kzc, const void* dev_db, void* dev_tau, void* dev_scratch, size_t scratch_bytes) {
    PostParams Q;
    int rc = post_check(h, kxc, kzc, dev_db, dev_tau, dev_scratch, scratch_bytes, Q);
    if (rc) return rc;
    if (h->isub != 0) return CHAN_ESTATE;
    const Plan& P = h->P;
    const size_t per = (size_t)Q.ny * Q.nr * Q.npk;
    // the stored velocities into the handle's own u, v, w (zeros beyond the cutoff; the vorticity slots are cleared: the
    // seventh product of the filter pass is not used), then the library's dealiased product path, pruned to the cutoff
    for (double2* f : {h->u, h->s1, h->w, h->ox, h->oz}) CK(cudaMemsetAsync(f, 0, h->F, h->stream));
    double2* keep_omy = h->omy;               // om_y is state: read a zero field instead of clobbering it
    PB(CHAN_KC_POST); k_post_scatter<<<296, 256, 0, h->stream>>>(Q, P.nxh, (const double2*)dev_db, h->u, h->s1, h->w); LAUNCHED();
    // v is state as well: the scattered v lives in the scratch field s1 for the duration of the pass
    double2* keep_v = h->v;
    h->v = h->s1; h->omy = h->ox;
    FieldPtrsW o;
    double2* T = (double2*)dev_scratch;
    for (int k = 0; k < 7; ++k) o.f[k] = T + (size_t)k * per;
    const int f32 = h->out_f32;
    h->out_f32 = 0;
    rc = run_planes(h, 7, o, kxc, kzc);
    h->out_f32 = f32; h->v = keep_v; h->omy = keep_omy;
    if (rc) return rc;
    PB(CHAN_KC_POST); k_post_sub<<<296, 256, 0, h->stream>>>(6 * per, (const double2*)dev_db + 3 * per, T, (double2*)dev_tau); LAUNCHED();
    // u, w, om_x, om_z were clobbered: rebuild them from the state if there is one
    if (h->have_state) return run_derive(h);
    return CHAN_OK;
}

int chan_debug_fma_peak(chan_t* h, double* host_tflops) {
    if (!h || !host_tflops) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = sms * 8, iters = 1 << 16;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {        // first round warms the clocks up
        CK(cudaEventRecord(e0, h->stream));
        k_fma_peak<<<blocks, 256, 0, h->stream>>>(h->scal + 7, iters, 0.999999, 1e-9);
        ++h->launches;
        CK(cudaEventRecord(e1, h->stream));
        CK(cudaEventSynchronize(e1));
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        const double tf = 2.0 * 8.0 * iters * (double)blocks * 256.0 / (ms * 1e-3) / 1e12;
        if (rep && tf > best) best = tf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (!ck(h, cudaGetLastError())) return CHAN_ECUDA;
    *host_tflops = best;
    return CHAN_OK;
}

int chan_debug_transpose(chan_t* h, int dir, const void* dev_in, void* dev_out) {
    if (!h || !dev_in || !dev_out || dir < 0 || dir > 1) return CHAN_EINVAL;
    if (!h->bound) return CHAN_ESTATE;
    return transpose(h, dir, (const double2*)dev_in, (double2*)dev_out);
}

}  // extern "C"
