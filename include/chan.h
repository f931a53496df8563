/* chan.h -- C ABI of the B200-native channel-flow DNS hot path (arxiv 1808.06461).
 *
 * One semi-implicit Runge-Kutta substep of incompressible plane-channel flow (section 2.1,
 * L61-80: walls at y=+-h, periodic x,z, constant mass flux; (omega_y, lap v) formulation [20];
 * Fourier x,z with zero-padding dealiasing; seven-point compact finite differences in y; three-substep
 * low-storage RK [34]) plus the paper's low-storage filter and plane statistics (section 3.1-3.2,
 * L112, L124: sharp Fourier cutoff, ten variables u_i, u_i u_j, om_i om_i).
 *
 * Conventions
 *  - h = 1; nu = 1/re_tau in the caller's velocity unit (reading R9).
 *  - Retained modes: p = 0..nx/2-1 (k_x = 2 pi p/lx), z slots s = 0..nz-1 in FFT order
 *    (q = 0..nz/2-1, slot nz/2 always zero, q = -nz/2+1..-1; k_z = 2 pi q/lz).
 *  - "LINE layout": complex128 interleaved, [nz][nx/2][ny], y fastest.  This is the layout of every
 *    field that crosses this ABI unless stated otherwise.
 *  - "device" pointers are CUDA device memory owned (allocated and freed) by the caller; "host"
 *    pointers are ordinary host memory.  The library allocates no device memory: tables and scratch
 *    are carved from the workspace handed to chan_bind().
 *  - Every call returns 0 (CHAN_OK) or a negative status; nothing is printed, nothing throws.
 *    Calls enqueue work on the stream given to chan_bind() and return without synchronising, except
 *    chan_stats(READ), chan_get_scalars() and the *_host entry points, which synchronise that stream.
 *  - A handle is not thread-safe.  There is NO CPU fallback: without a CUDA device every compute call
 *    returns CHAN_ECUDA.
 */
#ifndef CHAN_H_
#define CHAN_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CHAN_OK        0
#define CHAN_EINVAL   -1  /* bad sizes, non-monotone y, unsupported FFT length, cutoff out of range, NULL */
#define CHAN_ENOSPACE -2  /* workspace or output buffer too small                                   */
#define CHAN_ESTATE   -3  /* wrong call order (not bound, no state, chan_step() mid-step)           */
#define CHAN_ECUDA    -4  /* a CUDA runtime call or kernel launch failed                            */
#define CHAN_ELIMIT   -5  /* problem larger than the fixed static scratch of chan_post_strain_norm_static */

typedef struct chan chan_t; /* opaque */

/* nx, nz: Fourier collocation points before the 3/2 padding (even; 3nx/2 and 3nz/2 must factor into
 * 2,3 only; nx a multiple of 16 so that 3nx/2 is a multiple of 8; 3nx/2 <= 3520 and 3nz/2 <= 14080:
 * one padded x row set / one z column must fit in 220 KB of shared memory); ny: mesh points including
 * both walls, 8 <= ny <= 1877 (the mean-mode solve keeps 15 ny doubles in shared memory).  Anything else:
 * CHAN_EINVAL.  PAPER.md L80. */
typedef struct { int nx, ny, nz; } chan_grid_t;

/* lx, lz: periods; y: HOST array of ny strictly increasing mesh points, y[0] = -1, y[ny-1] = +1.
 * The array is copied.  PAPER.md L61, L80 (the paper's own mesh is not printed: reading R10). */
typedef struct { double lx, lz; const double* y; } chan_box_t;

/* lhs_halfwidth, rhs_halfwidth: compact stencil half widths, 1..3 (default 3,3 = seven-point, L80).
 * forcing: 0 = constant mass flux, 1 = constant pressure gradient (see chan_set_pgrad). */
typedef struct { int lhs_halfwidth, rhs_halfwidth; int forcing; } chan_opts_t;

/* Build the plan on the host (compact-difference band tables on the given mesh, their factorisations,
 * wavenumber and twiddle tables, RK constants).  dt is the FULL three-substep step.  opts may be NULL. */
int chan_create(chan_t** out, const chan_grid_t* grid, const chan_box_t* box, double re_tau, double dt,
                const chan_opts_t* opts);
int chan_destroy(chan_t* h);

/* Bytes of device workspace chan_bind() needs (0 if h is NULL). */
size_t chan_workspace_bytes(const chan_t* h);

/* Adopt caller-owned device memory (256-byte aligned, >= chan_workspace_bytes) and a CUDA stream
 * (cudaStream_t cast to void*; NULL = default stream).  Uploads the tables. */
int chan_bind(chan_t* h, void* dev_workspace, size_t bytes, void* cuda_stream);

/* State at a full-step boundary: v^, phi^ = (D2 - k^2) v^, omega_y^ in LINE layout, and the mean
 * profiles U(y), W(y) (ny doubles each), all DEVICE pointers.  set_state also fixes the mass flux
 * Q0 = sum_j w_j U_j (trapezoid weights, reading R8), clears the RK history and derives
 * u, w, omega_x, omega_z (step a1).  The (0,0) mode and the z-Nyquist slot of the inputs are ignored. */
int chan_set_state(chan_t* h, const void* dev_v, const void* dev_phi, const void* dev_omy,
                   const double* dev_U, const double* dev_W);
/* chan_get_state leaves the handle's state, history and derived fields untouched (hence const), but it is not a
 * pure read: it enqueues transpose kernels and copies on the bound stream like every other call. */
int chan_get_state(const chan_t* h, void* dev_v, void* dev_phi, void* dev_omy, double* dev_U, double* dev_W);

/* Same through HOST buffers (pageable or pinned).  Each field is staged through the library's scratch field, one
 * after the other, on the bound stream; both calls SYNCHRONISE that stream before returning, so the host buffers
 * may be reused or freed at once (set) and hold the state (get).  Neither touches any other library buffer. */
int chan_set_state_host(chan_t* h, const void* host_v, const void* host_phi, const void* host_omy,
                        const double* host_U, const double* host_W);
int chan_get_state_host(chan_t* h, void* host_v, void* host_phi, void* host_omy, double* host_U, double* host_W);

/* One substep of the three-substep semi-implicit low-storage Runge-Kutta scheme [34] ("A semi-implicit
 * third-order low-storage Runge-Kutta is used for temporal integration [34]"; constants: reading R3): steps a3-a12 of
 * DESIGN.md (nonlinear term on the dealiased grid, L80; Helmholtz/Poisson solves with the influence matrix, L100;
 * mean mode at constant mass flux, L61), then a1-a2 for the new state.  The substep index cycles 0,1,2; the state
 * is a physical time level only when the index is back at 0. */
int chan_substep(chan_t* h);
/* One full time step of PAPER.md L80 = three substeps; CHAN_ESTATE if called mid-step. */
int chan_step(chan_t* h);

/* Low-storage filter (a13): writes the ten variables u,v,w, uu,uv,uw,vv,vw,ww, om_i om_i
 * restricted to 0<=p<=kx_cut, |q|<=kz_cut into dev_out[10][ny][2 kz_cut+1][kx_cut+1] complex128
 * (z rows ordered q = 0..kz_cut, -kz_cut..-1).  Products are formed on the dealiased grid. */
int chan_filter_store(chan_t* h, int kx_cut, int kz_cut, void* dev_out, size_t out_bytes);
/* chan_filter_store of the CURRENT state fused into the full step that follows: identical output and identical new
 * state (bit for bit) as chan_filter_store() then chan_step(), but the filter products are formed from the z-padded
 * planes the first substep computes anyway, which saves the filter's own inverse z sweep.  CHAN_ESTATE mid-step. */
int chan_step_filter(chan_t* h, int kx_cut, int kz_cut, void* dev_out, size_t out_bytes);
/* Same with a HOST output buffer (synchronises).  The output is staged in one scratch field of the workspace:
 * CHAN_ENOSPACE if it is larger than max(one field, min(ten fields, 64 MiB)) -- use chan_filter_store then. */
int chan_filter_store_host(chan_t* h, int kx_cut, int kz_cut, void* host_out, size_t out_bytes);

/* Storage precision of the filtered database (NEXT-1; the paper's database holds about four bytes per
 * value): bytes_per_real = 8 (default: complex128 output, as documented above) or 4: chan_filter_store,
 * chan_step_filter, chan_filter_store_host and chan_run then write complex64 [10][ny][2 kz_cut+1][kx_cut+1] -- every
 * value computed in fp64 exactly as before and rounded once, to nearest even, when it is stored; the mode selection
 * is unchanged.  out_bytes / slot_bytes are checked against the smaller size.  CHAN_EINVAL for any other value. */
int chan_set_filter_precision(chan_t* h, int bytes_per_real);

/* Snapshot cadence (NEXT-1; filtered fields are stored every Delta t_e, a multiple of the time
 * step; L47: statistics on the fly).  Runs nsteps full steps without a host round trip: before step n the
 * statistics of the current state are accumulated if stats_every > 0 and n % stats_every == 0, and the filtered
 * database of the current state is emitted (fused into the step, as chan_step_filter) into slot
 * (emitted so far) % ring_slots of dev_ring if filter_every > 0 and n % filter_every == 0.  A slot is slot_bytes
 * long and must hold one database in the precision in effect (CHAN_ENOSPACE otherwise); the caller drains the ring
 * (e.g. by copies on another stream ordered by events) before it wraps.  *snapshots = databases emitted (may be
 * NULL).  Everything is enqueued on the bound stream; nothing synchronises.  CHAN_ESTATE mid-step.
 * When the statistics and an fp64 database fall on the same step, the ten profiles are taken from the (0,0) modes of
 * that database -- which ARE the plane statistics of the full field (L124: second-order consistent) -- instead of a
 * pass over the fields of their own: equal to chan_stats(ACCUMULATE) to rounding. */
typedef struct {
    int nsteps, filter_every, stats_every;
    int kx_cut, kz_cut;
    void* dev_ring; size_t slot_bytes; int ring_slots;
} chan_run_t;
int chan_run(chan_t* h, const chan_run_t* r, long long* snapshots);

/* ---- mesh tools of the paper's section 2.3 (NEXT-4; Fig. 2.3); HOST only, no handle, no device ----------
 * "The most numerically sensitive operation ... is the solution of the bilaplacian operator, which requires the solution
 * of multiple homogeneous Helmholtz equations ... very thin boundary layers near the wall" (L100).
 * chan_mesh_helmholtz_error: the paper's test.  For the compact second-derivative rows of reading R4 on the mesh
 * host_y[ny] it solves phi'' = lambda phi with phi = 1 at one wall and 0 at the other and returns, for each wall, the
 * maximum over the first nfirst interior points of |phi_j - phi_exact(y_j)|: host_err2[0] for y = -1, [1] for y = +1.
 * lambda is the caller's worst case, k_max^2 + 1/(beta_3 nu dt) (beta_3 = 1/6).
 * chan_mesh_optimize: the paper's remedy (L102: "slightly displacing the first 20 grid points in order to minimize the
 * error of the most dangerous solutions without affecting too much the individual grid spacing").  Points 1..npoints
 * from each wall are moved, each by at most max_shift (< 1/2) times the smaller of its two original neighbouring
 * spacings, by a deterministic cyclic coordinate search (`sweeps` rounds with a halving step) that minimises the error
 * above over the first npoints + 3 points; a displacement is only accepted if the mesh stays admissible for the
 * unpivoted solves (every elimination pivot of B2 - sigma A2 negative for sigma = 0, lambda/100, lambda: without this
 * guard the search walks into meshes whose second-derivative operator has eigenvalues in the right half plane -- the
 * instability L102 mentions).  The paper prints neither its objective nor its optimiser: this is reading R23 of
 * DESIGN.md.  host_y is updated in place; the errors before and after (two walls each) are optional outputs.
 * CHAN_EINVAL: bad sizes, non-monotone or inadmissible input mesh, max_shift outside (0, 1/2). */
int chan_mesh_helmholtz_error(int ny, const double* host_y, double lambda, int nfirst, double* host_err2);
int chan_mesh_optimize(int ny, double* host_y, int npoints, double lambda, double max_shift, int sweeps, double* host_err_before2,
                       double* host_err_after2);

/* ---- post-processing of a stored database (NEXT-2; section 3.2) ---------------------------
 * dev_db is a complex128 database as written by chan_filter_store / chan_step_filter / chan_run with the same
 * cutoffs, [10][ny][2 kz_cut+1][kx_cut+1].  The handle supplies the mesh, its compact operators, nu and the box; it
 * may be the handle that produced the database or any other handle on the same mesh and box whose retained modes
 * contain the stored ones -- typically a small one on the storage grid (nx >= 2 kx_cut + 2, nz >= 2 kz_cut + 2), which
 * is what post-processing the stored data offline amounts to.  dev_scratch: caller-owned device memory of at least
 * chan_post_scratch_bytes() bytes (CHAN_ENOSPACE otherwise).  Outputs are complex128 planes [ny][2 kz_cut+1][kx_cut+1]
 * in the database's mode order.  Asynchronous on the bound stream.  Readings R17-R20 of DESIGN.md. */
size_t chan_post_scratch_bytes(const chan_t* h, int kx_cut, int kz_cut);
/* Filtered pressure from the Poisson equation (3.2) d_kk p = -d_ij(u_i u_j) (L126-132) with the Neumann data of a
 * no-slip wall d_y p = nu d_yy v taken from the stored v (R18), solved per mode with the substep's compact operators
 * and wall superposition (R19); mode (0,0): p = -(vv) + (vv)(-1). */
int chan_post_pressure(chan_t* h, int kx_cut, int kz_cut, const void* dev_db, void* dev_p, void* dev_scratch, size_t scratch_bytes);
/* Filtered S_ij S_ij = d_ij(u_i u_j) + om_i om_i / 2: identity (3.3) of L134 as re-derived in reading R17. */
int chan_post_strain_norm(chan_t* h, int kx_cut, int kz_cut, const void* dev_db, void* dev_out, void* dev_scratch, size_t scratch_bytes);
/* chan_post_strain_norm for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the same kernel and the same result, bit for bit, but the one scratch plane set lives in a
 * file-scope `static __device__` array of CHAN_STATIC_SCRATCH_BYTES (4 MiB) inside the library -- every GPU that loads
 * libchan.so holds those 4 MiB until the process exits.  The caller passes only the database and the output; the call
 * allocates nothing (no cudaMalloc / cudaFree / allocating library routine, on the host one device-address lookup per
 * device on first use) and enqueues one kernel on the bound stream.
 * Limit: ny (2 kz_cut + 1)(kx_cut + 1) * 16 bytes <= CHAN_STATIC_SCRATCH_BYTES, i.e. 262144 stored (y, mode) points;
 * beyond it CHAN_ELIMIT and nothing is launched -- use chan_post_strain_norm with caller scratch then.
 * The array is SHARED by every call, handle and stream of the process on that GPU and keeps the last call's contents:
 * nothing in it needs to start at zero (each mode writes its column before reading it), but two calls that overlap on
 * the GPU (different streams, or different handles bound to different streams) race on it.  Calls on one stream are safe. */
#define CHAN_STATIC_SCRATCH_BYTES (4u << 20)
size_t chan_post_strain_norm_static_limit(void);     /* = CHAN_STATIC_SCRATCH_BYTES */
int chan_post_strain_norm_static(chan_t* h, int kx_cut, int kz_cut, const void* dev_db, void* dev_out);
/* Sub-grid stresses (3.4), L149: dev_tau[6][ny][2 kz_cut+1][kx_cut+1] = stored u_i u_j minus the product of the STORED
 * velocities, formed by the library's dealiased product path on this handle's grid and pruned to the cutoff (R20),
 * order uu,uv,uw,vv,vw,ww.  Overwrites the handle's derived fields u, w, om_x, om_z and rebuilds them (step a1) if the
 * handle has a state; CHAN_ESTATE mid-step. */
int chan_post_sgs(chan_t* h, int kx_cut, int kz_cut, const void* dev_db, void* dev_tau, void* dev_scratch, size_t scratch_bytes);

/* Plane statistics (a14; "Regular statistics of the fully resolved flow are computed and stored
 * on-the-fly"; the profiles are those of the ten variables of L124): flags is an OR of the values below.  ACCUMULATE adds the ten profiles
 * <u>,<v>,<w>,<uu>,<uv>,<uw>,<vv>,<vw>,<ww>,<om_i om_i> of the current state to the running sums;
 * READ copies sums[10][ny] to host_out and the sample count to *nsamples (synchronises); RESET clears. */
#define CHAN_STATS_ACCUMULATE 1
#define CHAN_STATS_READ       2
#define CHAN_STATS_RESET      4
int chan_stats(chan_t* h, int flags, double* host_out, long long* nsamples);

/* One-dimensional co-spectra of the current state at every y (NEXT-4 "more statistics"; Fig. 3.1, L163 /
 * L173 Fig. 3.3 compare such spectra of the database with the reference runs): for the seven second-order quantities
 * uu,uv,uw,vv,vw,ww, om_i om_i (the order of chan_stats) dev_ex[7][ny][nx/2] = w_p sum over the k_z slots of
 * Re(a^ conj b^) and dev_ez[7][ny][nz] = sum over p of w_p Re(a^ conj b^) (w_0 = 1, w_p = 2; z slots in FFT order, the
 * Nyquist slot is zero).  Summed over their wavenumber both equal the plane statistics.  DEVICE outputs, overwritten
 * (accumulation over snapshots is the caller's); either pointer may be NULL.  Asynchronous on the bound stream.
 * The friction velocity of L165 (Fig. 3.4) follows from chan_get_scalars(): u_tau^2 = out[2] (bottom wall), out[3] (top). */
int chan_spectra(chan_t* h, double* dev_ex, size_t ex_bytes, double* dev_ez, size_t ez_bytes);

/* Scalars: out[0] = -dP/dx recovered by the last substep (constant mass flux) or prescribed,
 * out[1] = mass flux Q0, out[2] = nu dU/dy at y=-1, out[3] = -nu dU/dy at y=+1.  Synchronises. */
int chan_get_scalars(chan_t* h, double* host_out4);
int chan_set_pgrad(chan_t* h, double minus_dpdx); /* forcing == 1 only */

const char* chan_strerror(int status);

/* ---- tuning overrides ---------------------------------------------------------------------------
 * Launch geometry and stage lists; they never change results beyond rounding.  The library reads no environment
 * variable and keeps no global state: overrides go through the handle.  chan_debug_set_tuning() must be called
 * before chan_bind() (CHAN_ESTATE afterwards: the workspace layout depends on it); every field 0 keeps the plan's own
 * choice; a value the plan cannot honour is CHAN_EINVAL and leaves the handle unchanged.  chan_debug_get_tuning()
 * reports the values in effect. */
typedef struct {
    int xfuse;            /* 4 | 8: radix of the x stage fused with the products                                  */
    int maxradix_z;       /* 2..12: largest radix of a z stage                                                    */
    int maxradix_x;       /* 2..18: largest radix of an x stage in front of the fused one                          */
    int tz;               /* k_x columns per z tile: 1, 2, 4, 8 or 16                                              */
    int zthreads;         /* threads per CTA of the z passes, a multiple of 32 in 32..256                          */
    int xthreads;         /* threads per CTA of the x pass, 32..256                                                */
    int chunk_mb;         /* size of the z-padded plane-chunk buffers in MiB (default 3072)                        */
    int planes_per_chunk; /* get only: y-planes per launch of the plane kernels that follows from chunk_mb         */
    int plane_overlap;    /* 1 (default): K2, K3, K4 as separate launches; 2: merged launches (K2 of chunk t, K3 of chunk t-1,
                             K4 of chunk t-2 interleaved in one grid; CHAN_EINVAL if not compiled for this plan; results equal
                             to rounding, not bit for bit: another kernel, another FMA contraction); get: the mode in effect */
    int z_cluster;        /* 1 (default): one CTA per z tile; 2: the tile split by rows over a 2-CTA cluster with twice the
                             columns, half of one stage's data exchanged through distributed shared memory (CHAN_EINVAL if
                             not compiled for this plan; measured slower on config 3-5, kept as an experiment)            */
    int reserved[6];      /* must be 0                                                                             */
} chan_tuning_t;
int chan_debug_set_tuning(chan_t* h, const chan_tuning_t* t);
int chan_debug_get_tuning(const chan_t* h, chan_tuning_t* out);

/* ---- debug / parity / profiling hooks (run one stage on library buffers) ------------------------
 * Field ids for chan_debug_get_field / chan_debug_set_field (LINE layout, device pointers): */
enum { CHAN_F_V = 0, CHAN_F_PHI, CHAN_F_OMY, CHAN_F_U, CHAN_F_W, CHAN_F_OMX, CHAN_F_OMZ,
       CHAN_F_H1, CHAN_F_H2, CHAN_F_H3, CHAN_F_HV_PREV, CHAN_F_HG_PREV, CHAN_F_COUNT };
int chan_debug_get_field(const chan_t* h, int field, void* dev_out);
int chan_debug_set_field(chan_t* h, int field, const void* dev_in);
/* Stages: run on whatever the library buffers currently hold. */
enum { CHAN_STAGE_DERIVE = 0,   /* a1-a2: state -> u,w,om_x,om_z                                  */
       CHAN_STAGE_NONLINEAR,    /* a3-a8: u..om_z -> H1,H2,H3                                      */
       CHAN_STAGE_YSOLVE,       /* a9-a12: H, state, history -> new state, history (uses substep index) */
       CHAN_STAGE_COUNT };
int chan_debug_run_stage(chan_t* h, int stage);
int chan_debug_set_substep_index(chan_t* h, int i);
/* Copy of the host-computed compact band tables, out[4][ny][7]: A1, B1, A2, B2 (HOST pointer). */
int chan_debug_get_band_tables(const chan_t* h, double* host_out);
/* One-line description of the plan in effect (stage lists, tiles, chunking) into buf[n] (HOST), NUL-terminated. */
int chan_debug_describe(const chan_t* h, char* buf, size_t n);
/* Number of kernels this handle has launched so far (bench.py's gpu_launches). */
long long chan_debug_launch_count(const chan_t* h);
/* Per-kernel-class device timing with CUDA events on the bound stream (bench.py's roofline object).
 * chan_debug_profile(h,1) clears and starts recording one event pair around every kernel launch;
 * chan_debug_profile(h,0) stops; chan_debug_profile_read synchronises and returns, per class, the summed
 * milliseconds and the number of launches (arrays of CHAN_KC_COUNT entries, HOST pointers). */
enum { CHAN_KC_D1FWD = 0, CHAN_KC_DERIVE_DOWN, CHAN_KC_DERIVE_UP, CHAN_KC_ZFFT_INV, CHAN_KC_XFFT_PROD, CHAN_KC_ZFFT_FWD,
       CHAN_KC_MEAN, CHAN_KC_Y1, CHAN_KC_Y2, CHAN_KC_Y3, CHAN_KC_Y4, CHAN_KC_Y5, CHAN_KC_TRANSPOSE,
       CHAN_KC_FILTER_COPY, CHAN_KC_XFFT_PROD_FILTER, CHAN_KC_ZFFT_FWD_FILTER, CHAN_KC_STATS, CHAN_KC_PLANES_MERGED,
       CHAN_KC_POST, CHAN_KC_COUNT };
int chan_debug_profile(chan_t* h, int enable);
int chan_debug_profile_read(chan_t* h, double* host_ms, long long* host_counts);
/* fp64 FMA throughput of the device, measured with a register-only micro-kernel (8 independent DFMA chains per thread,
 * 8 CTAs of 256 threads per SM, about 30 ms, best of 3 after a warm-up round) on the bound stream; synchronises.
 * TFLOP/s into *host_tflops.  The "alu" roof of bench.py. */
int chan_debug_fma_peak(chan_t* h, double* host_tflops);
/* Plain line<->plane transposes (a2/a8) on caller buffers, for roofline timing: n fields of one
 * [nz][nx/2][ny] <-> [ny][nz][nx/2] complex128 array each. dir 0: line->plane, 1: plane->line. */
int chan_debug_transpose(chan_t* h, int dir, const void* dev_in, void* dev_out);

#ifdef __cplusplus
}
#endif
#endif /* CHAN_H_ */
