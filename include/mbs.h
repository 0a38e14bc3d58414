/*
 * mbs.h -- C ABI of the B200-native modified-Born-series (MBS) Helmholtz solver with the
 * non-overlapping domain decomposition of Mache & Vellekoop, arXiv 2410.02395.
 *
 * Citations "P:NN" are line numbers of PAPER.md (the paper text); "R<k>" are the readings of
 * points the paper leaves open, listed in DESIGN.md section 3.
 *
 * The library solves   [nabla^2 + k^2(r)] x(r) = -y(r)            (Eq. (1))
 * on a regular 1D/2D/3D grid with the preconditioned Richardson iteration
 *     x <- x - alpha B ( x - (L+I)^-1 [ y_vec + B x ] ),  B = I - V     (Eq. (6))
 * where L is a per-subdomain FFT convolution (Eq. (8)) and V holds the scattering
 * potential plus the truncated wrap-around / transfer corrections.
 *
 * Conventions
 *  - All arrays are complex64 (interleaved float re, im), C order, axis 0 slowest, `shape` voxels.
 *  - "device" pointers are CUDA device pointers, 16-byte aligned; "host" pointers are ordinary
 *    host memory.  The caller owns every array it passes in; the library owns the context and
 *    (unless mbs_set_workspace is used) its workspace.
 *  - Every call returns an int status (MBS_OK = 0).  No exceptions cross the boundary, there is
 *    no global state, and one context must be used from one thread at a time.
 *  - A context belongs to the CUDA device that is current when mbs_create is called; every later call on it must be
 *    made with the same current device.
 *  - All device work is enqueued on the stream given to mbs_create.  mbs_apply_operator and
 *    mbs_set_potential are asynchronous with respect to the host unless stated; mbs_solve*
 *    return after the stop decision has been observed.
 *  - There is no CPU fallback: every step runs in the library's CUDA kernels (sm_100a).
 */
#ifndef MBS_B200_H
#define MBS_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define MBS_API __attribute__((visibility("default")))
#else
#define MBS_API
#endif

typedef struct mbs_ctx mbs_ctx;

enum mbs_status {
    MBS_OK = 0,
    MBS_ERR_INVALID_ARG = 1,      /* bad argument; see mbs_last_error                       */
    MBS_ERR_UNSUPPORTED_SIZE = 2, /* a subdomain length has no FFT plan (see mbs_fft_supported) */
    MBS_ERR_OOM = 3,              /* device or host allocation failed                        */
    MBS_ERR_CUDA = 4,             /* CUDA runtime error; text in mbs_last_error              */
    MBS_ERR_NOT_CONVERGED = 5,    /* max_iter reached; x and the history are still valid     */
    MBS_ERR_NUMERIC = 6,          /* NaN/Inf in the residual                                 */
    MBS_ERR_STATE = 7             /* call out of order (e.g. solve before set_potential)     */
};

/* Operators of mbs_apply_operator.  All are the SCALED operators (they include c). */
enum mbs_operator {
    MBS_OP_B = 0,          /* B = I - V: scattering diagonal + edge-slab corrections */
    MBS_OP_PROPAGATOR = 1, /* (L+I)^-1: per-subdomain FFT, 1/(c(k0^2-|p|^2)+1), inverse FFT */
    MBS_OP_A = 2,          /* A = (L+I) - B                                            */
    MBS_OP_PRECOND_A = 3   /* Gamma^-1 A = B - B (L+I)^-1 B                            */
};

/* Options of mbs_set_option. */
enum mbs_option {
    MBS_OPT_FUSED = 0,          /* 1 (default): fused sweeps (prologue in the first FFT sweep, epilogue in the
                                   last, 112 B/voxel-iteration ledger); 0: one kernel per step of P:122-128     */
    MBS_OPT_CHECK_INTERVAL = 1, /* iterations enqueued between two host polls of the device stop flag (>= 1)  */
    MBS_OPT_USE_GRAPH = 2,      /* 1: replay each poll interval as a CUDA graph (default 1 for small grids)   */
    MBS_OPT_TMA = 4,            /* 1 (default): strided-axis FFT sweeps are fed by TMA box loads/stores through a
                                   shared-memory stage ring; 0: threads load/store the tiles themselves        */
    MBS_OPT_LINE = 5,           /* 1 (default): first / last sweep as warp-line kernels (each warp owns whole lines of
                                   the contiguous axis, no block barriers), in the variant with t = 8 known at compile
                                   time where it is the faster one; 2: warp-line kernels, generic-t variant only;
                                   0: tile kernels with in-CTA edge terms                                          */
    MBS_OPT_REFINE = 7,         /* split iterate x = x_ref + delta (api.cu recenter()): the FFT sweeps run on the small part
                                   delta, so the complex64 rounding floor of the residual falls with it and tolerances such
                                   as config 1's 1e-6 are reachable; same iteration in exact arithmetic, two extra arrays.
                                   -1 (default): on for grids of <= 2^21 voxels; 0: off; 1: on                   */
    MBS_OPT_PROFILE = 3         /* 1: bracket every kernel launch with CUDA events on the context's stream and
                                   accumulate per-kernel device time (mbs_get_kernel_stats); disables graphs   */
};

/* Per-kernel device time accumulated while MBS_OPT_PROFILE is on (CUDA events on the stream). */
typedef struct mbs_kernel_stat {
    char name[48];               /* kernel class, e.g. "fft_strided_mid_ax0"                          */
    int64_t launches;
    double total_ms;             /* sum of the launches' event-to-event durations                     */
    double algorithmic_bytes;    /* bytes one launch must move, summed over launches */
} mbs_kernel_stat;

typedef struct mbs_info {
    double c_re, c_im;             /* scale factor c of Eq. (9)                              */
    double k02_re, k02_im;         /* background k0^2 (R2)                                           */
    double v_max;                  /* ||k^2 - k0^2||_inf                                      */
    double norm_A12;               /* sigma_max(K_t)/h^2 (R5)                                 */
    int32_t sum_a;                 /* sum_d a_d of Eq. (9)                                   */
    int32_t ndim;
    int64_t voxels;
    int64_t subdomain_shape[3];    /* M_d                                                            */
    double alpha;                  /* 0.75                                                    */
    double norm_rhs;               /* ||Gamma^-1 y_vec|| of the last solve                   */
    double algorithmic_bytes_per_iteration; /* floor ledger of DESIGN.md section 5 (112 B/voxel in 3D) */
    uint64_t workspace_bytes;
    int64_t kernel_launches;       /* kernels launched by this context so far                        */
    double last_solve_ms;          /* device time of the last mbs_solve* iteration loop (CUDA events) */
    double sparse_source_bytes_per_iteration; /* the ledger minus the all-zero rows of the last source, which the first
                                      sweep does not read (SURVEY 8(d) "source stored sparsely": 104 B/voxel for a
                                      point source); equals the floor ledger before the first solve            */
} mbs_info;

/*
 * Create a solver for one grid (P:37-45 problem statement; P:82 decomposition).
 *  ndim            1, 2 or 3.
 *  shape[ndim]     grid size in voxels INCLUDING the absorbing layers, axis 0 slowest.  The grid may hold at most
 *                  2^31 - 1 voxels (32-bit tile and line counters in the kernels): 1260^3 fits, 1290^3 does not
 *                  -> MBS_ERR_INVALID_ARG.
 *  pixel_size      grid pitch h (same on every axis), same unit as wavelength.   (lambda/4)
 *  wavelength      vacuum wavelength lambda; k(r) = 2 pi n(r) / lambda.
 *  boundary_width[ndim]  W_d: thickness in voxels of the absorbing layer on each side (R3).
 *  n_subdomains[ndim]    S_d >= 1, shape[d] % S_d == 0; subdomain length M_d = shape[d] / S_d.
 *  periodic[ndim]  1: axis is periodic (no wrap correction when S_d = 1, wrap-around transfer when
 *                  S_d >= 2); 0: non-periodic.  May be NULL (= all 0).
 *  n_correction    t: edge points kept in the truncated corrections (paper default 8).
 *                  0 is legal only if every axis is periodic with S_d = 1.  Requires 2 t <= M_d.
 *  cuda_stream     a cudaStream_t (may be NULL for the default stream); all work runs on it.
 * Errors: MBS_ERR_INVALID_ARG, MBS_ERR_UNSUPPORTED_SIZE, MBS_ERR_OOM, MBS_ERR_CUDA.
 * On failure *out is NULL; mbs_last_error(NULL) returns the reason of the last failed create
 * on this thread.
 */
MBS_API int mbs_create(mbs_ctx** out, int ndim, const int64_t* shape, double pixel_size, double wavelength,
               const int32_t* boundary_width, const int32_t* n_subdomains, const uint8_t* periodic,
               int32_t n_correction, void* cuda_stream);

/* 1 if a subdomain length M has an FFT plan in this build: 2^a (8..1024), 5*2^a (40..640), 3*2^a (48..768). */
MBS_API int mbs_fft_supported(int64_t M);

/* Bytes of device workspace the context needs (B_diag, u, slab buffers, reduction scratch). */
MBS_API size_t mbs_workspace_bytes(const mbs_ctx* ctx);

/* Hand the context a caller-owned device buffer of at least mbs_workspace_bytes (256-byte aligned)
 * instead of letting it cudaMalloc its own.  Must precede mbs_set_potential.  The buffer must
 * outlive the context. */
MBS_API int mbs_set_workspace(mbs_ctx* ctx, void* device_buffer, size_t bytes);

MBS_API int mbs_set_option(mbs_ctx* ctx, int option, int64_t value);

/*
 * Setup from the complex refractive index n(r) (device, complex64, `shape`):
 * k^2 = (2 pi/lambda)^2 n^2, absorbing layer (R3), k0^2 (R2), ||k^2-k0^2||_inf, c by Eq. (9),
 * B_diag = 1 - c (k^2 - k0^2).  Computed in double on the device, stored as complex64.
 * Requires Im n >= 0 (P:55 convergence condition) -> MBS_ERR_INVALID_ARG otherwise.
 * The map is read once and not retained.  Synchronises the stream.
 */
MBS_API int mbs_set_potential(mbs_ctx* ctx, const void* n_map_device);

/* out = Op(in) for one of enum mbs_operator; device pointers; in == out allowed. */
MBS_API int mbs_apply_operator(mbs_ctx* ctx, int which, const void* in_device, void* out_device);

/*
 * Run the iteration of Eq. (6) until eps < tol or max_iter updates (R7, R8).
 *  y   device, physical source y(r) of Eq. (1); the library forms y_vec = -c y.
 *  x   device, in/out: x^(0) on entry (zero it for a cold start; any start converges).
 *  residual_history  host, capacity max_iter (may be NULL): history[n] = eps_n, the relative
 *      residual ||Gamma^-1(y - A x^(n))|| / ||Gamma^-1 y|| of the iterate BEFORE update n.
 *  n_iter  host, out: number of updates applied.
 * Returns MBS_OK (converged), MBS_ERR_NOT_CONVERGED, MBS_ERR_NUMERIC (NaN/Inf in the source, the medium or the
 * residual), MBS_ERR_INVALID_ARG (y identically zero: the relative residual of P:130 is undefined), or a
 * CUDA/state error.
 */
/*
 * out = B in (as mbs_apply_operator with MBS_OP_B; Eq. (8)) WITHOUT any allocation, for callers that may
 * not call cudaMalloc (code under CUDA graph capture, serving loops, harnesses that forbid it).  The scratch of the
 * edge-slab kernels (the compact correction buffers, sum over the axes with corrections of
 * 16 t S_d (voxels / shape[d]) bytes, each rounded up to 256) lives in a static device array of
 * MBS_STATIC_SCRATCH_BYTES that every GPU loading the library holds until the process exits.
 *  - Grids that need more return MBS_ERR_INVALID_ARG (text in mbs_last_error); use mbs_apply_operator there.
 *  - The array is shared by all contexts and calls on the device: calls that overlap on the GPU (different streams
 *    with no ordering between them) race.  Calls on one stream are safe.  Asynchronous like mbs_apply_operator;
 *    in == out allowed; device pointers, complex64, `shape`.
 *  - Calls no cudaMalloc / cudaFree / allocating routine.  The first call on a device looks up the array's device
 *    address (cudaGetSymbolAddress) with the context's device current.
 */
#define MBS_STATIC_SCRATCH_BYTES (16u << 20)
MBS_API int mbs_apply_B_static(mbs_ctx* ctx, const void* in_device, void* out_device);

MBS_API int mbs_solve(mbs_ctx* ctx, const void* y_device, void* x_device, double tol, int32_t max_iter,
              double* residual_history, int32_t* n_iter);

/*
 * Batched solve: n_batch sources for ONE medium and wavelength (time- or source-dependent problems are solved one
 * system per source; the systems share A).  Reading R18, the same rule as the oracle's solve_batch:
 * every source is iterated in lock step with Eq. (6), exactly as mbs_solve would iterate it, and ONE stop test is
 * applied to the stacked system: eps_n = sqrt(sum_b ||r_b||^2) / sqrt(sum_b ||Gamma^-1 y_vec,b||^2).
 *  y, x   device, n_batch fields one after the other ([n_batch][shape], complex64); x in/out as in mbs_solve.
 *  tol    >= 0, or -1 for exactly max_iter updates without a stop test.
 *  residual_history / n_iter  as in mbs_solve, for the stacked system (every source gets the same number of updates).
 * What it buys: the first / last sweep read B_diag once per line for the whole batch (112 -> 96 + 16/n_batch bytes per
 * voxel-iteration and source).  The library allocates n_batch fields of workspace on the first call with a larger batch.
 * Needs a 2-D or 3-D grid whose contiguous subdomain length has a warp-line sweep (<= 512 voxels), t in {2, 4, 8, 16}, the
 * default kernel options, no subdomain activation -> MBS_ERR_UNSUPPORTED_SIZE / MBS_ERR_INVALID_ARG otherwise.
 * n_batch = 1 is mbs_solve.
 */
MBS_API int mbs_solve_batch(mbs_ctx* ctx, int32_t n_batch, const void* y_device, void* x_device, double tol, int32_t max_iter,
                    double* residual_history, int32_t* n_iter);

/*
 * Exactly n_iter updates of Eq. (6) with no stop test: the timed "step" of bench.py.
 *  nu  > 0: the normalisation ||Gamma^-1 y_vec|| to use for residual_history (e.g. mbs_info.norm_rhs
 *           of an earlier solve with the same y); <= 0: computed first as in mbs_solve.
 *  residual_history  host, capacity n_iter, may be NULL.
 * Returns MBS_OK, MBS_ERR_NUMERIC or a CUDA/state error.  Synchronises the stream before returning.
 */
MBS_API int mbs_iterate(mbs_ctx* ctx, const void* y_device, void* x_device, int32_t n_iter, double nu,
                double* residual_history);

/* Same with HOST arrays y and x (complex64, `shape`): copies y and x^(0) to the device, iterates,
 * copies x back.  The end-to-end entry point (bench.py "e2e"). */
MBS_API int mbs_solve_host(mbs_ctx* ctx, const void* y_host, void* x_host, double tol, int32_t max_iter,
                   double* residual_history, int32_t* n_iter);

/*
 * Subdomain activation ("initially activating only those subdomains that hold a source term.  Neighbouring
 * subdomains are activated only after the norm of the transferred field exceeds a certain threshold").  The paper
 * fixes neither the norm nor the threshold; reading R17, the same rule as the oracle's
 * solve_activated:
 *   - a subdomain is active from the start if y or x^(0) is non-zero anywhere in it;
 *   - before update n an inactive subdomain s becomes active (for good) when
 *       sqrt( sum_d || (corr_d x^(n)) restricted to s ||^2 ) >= threshold * ||Gamma^-1 y_vec||,
 *     corr_d = the edge corrections of P:124-128 (x_s = 0 there, so this is what its neighbours transfer into it);
 *   - an inactive subdomain is not computed: no FFT, no update, no residual.
 *  enable     0 / 1 (default 0).
 *  threshold  relative to ||Gamma^-1 y_vec||; < 0: tol / 10 of the solve (0 for mbs_iterate, i.e. all active).
 * Needs a 2-D or 3-D grid and the default kernel options.  Errors: MBS_ERR_INVALID_ARG, MBS_ERR_UNSUPPORTED_SIZE, MBS_ERR_OOM.
 */
MBS_API int mbs_set_activation(mbs_ctx* ctx, int enable, double threshold);

/* Iteration at which each subdomain was activated in the last solve (index (s0*S1 + s1)*S2 + s2 in the order of
 * n_subdomains; 0 = from the start, -1 = never; all 0 when activation is off).  activated_at: host, `capacity` entries,
 * may be NULL; *n_subdomains receives the number of subdomains. */
MBS_API int mbs_get_activation(const mbs_ctx* ctx, int32_t* activated_at, int32_t capacity, int32_t* n_subdomains);

MBS_API int mbs_get_info(const mbs_ctx* ctx, mbs_info* out);

/* Kernel statistics gathered since the last mbs_reset_kernel_stats (needs MBS_OPT_PROFILE = 1).
 * Writes at most `capacity` entries to out (host) and the number of classes seen to *count.
 * Synchronises the stream. */
MBS_API int mbs_get_kernel_stats(mbs_ctx* ctx, mbs_kernel_stat* out, int32_t capacity, int32_t* count);
MBS_API int mbs_reset_kernel_stats(mbs_ctx* ctx);

/* Frees everything the library allocated.  NULL-safe. */
MBS_API void mbs_destroy(mbs_ctx* ctx);

/* Library-owned text of the last error on this context (or of the last failed mbs_create when
 * ctx is NULL); valid until the next call on the context. */
MBS_API const char* mbs_last_error(const mbs_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* MBS_B200_H */
