// api.cu -- the C ABI of include/mbs.h: context, host-side setup (Eq. (9), K_t, tables), operator
// application and the solve loop with its device-side stop flag.  Every step of the hot path runs
// in the CUDA kernels of kernels.cu / fft_inst.cu; there is no CPU fallback.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <complex>
#include <mutex>
#include <string>
#include <vector>

#include "mbs_internal.h"

using namespace mbs;

typedef std::complex<double> cd;

// Per-kernel device timing (MBS_OPT_PROFILE): every launch is bracketed by a pair of CUDA events on
// the context's stream; pairs are resolved after the next stream synchronisation.
struct KernelClass {
    std::string name;
    int64_t launches = 0;
    double ms = 0, bytes = 0;
};
struct Profiler {
    std::vector<KernelClass> classes;
    std::vector<cudaEvent_t> pool;           // 2 events per pending launch
    std::vector<int> pending;                // class index of each pending launch
    int find(const char* name) {
        for (size_t i = 0; i < classes.size(); ++i)
            if (classes[i].name == name) return (int)i;
        classes.push_back(KernelClass{name});
        return (int)classes.size() - 1;
    }
};

struct mbs_ctx {
    int ndim = 0;
    int first = 0;  // first real axis of the internal 3-D description
    GridDesc g{};
    int W[3] = {0, 0, 0};
    double h = 0, wavelength = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 148;

    // workspace
    void* ws = nullptr;
    size_t ws_bytes = 0;
    bool ws_owned = false;
    cf* bdiag = nullptr;
    cf* u = nullptr;
    CorrBufs cx{};  // edge corrections of the current operand
    CorrBufs ds{};  // fused path: d = x - u' at the slab voxels of the non-contiguous axes
    double* partials = nullptr;
    unsigned char* ymask = nullptr;  // per grid row: the source row is not all zero

    // small library-owned device data
    DevState* state = nullptr;
    double* hist_dev = nullptr;
    int hist_cap = 0;
    float* Kh_dev = nullptr;
    cf* tw_dev[3] = {nullptr, nullptr, nullptr};
    float* p2_dev[3] = {nullptr, nullptr, nullptr};
    float* wtab_dev = nullptr;   // |p|^2 of the axes after the first one, per inner index of the kernel-multiply sweep
    const FftEntry* fft[3] = {nullptr, nullptr, nullptr};
    DevState* state_pinned = nullptr;  // 2 slots for polling
    cudaEvent_t ev_poll[2] = {nullptr, nullptr};
    cudaEvent_t ev_t0 = nullptr, ev_t1 = nullptr;
    cf* host_y = nullptr;  // device staging of mbs_solve_host
    cf* host_x = nullptr;

    // scalars
    cd c = 0, k02 = 0;
    double v_max = 0, norm_A12 = 0, beta = 0.5, alpha = 0.75, norm_rhs = 0, last_solve_ms = 0;
    int sum_a = 0;
    double y_row_fraction = 1.0;     // fraction of the grid rows of the last source that are not all zero (sweep 1 skips the rest)
    bool potential_set = false;
    std::vector<double> Kh;  // t*t

    // options
    int fused = 1;
    int check_interval = 0;  // 0 = automatic
    int use_graph = -1;      // -1 = automatic
    int use_tma = 1;         // TMA-fed strided sweeps
    int use_line = 1;        // warp-line first / last sweeps

    int profile = 0;
    Profiler prof;

    // split iterate x = x_ref + delta (lifts the complex64 residual floor on small grids; see recenter())
    int refine = -1;                 // MBS_OPT_REFINE: -1 automatic (grids of <= 2^21 voxels), 0 off, 1 on
    cf* delta = nullptr;             // owned: the small part of the iterate
    cf* dref = nullptr;              // owned: r_ref = B d_ref (complex128 path) or d_ref = x_ref - (L+I)^-1 (B x_ref + y_vec)
    double* bdiag64 = nullptr;       // owned: B_diag in complex128 (grids that may use the split iterate)
    double* Kh64_dev = nullptr;      // owned: K_t / h^2 in double
    double* tw64_dev[3] = {nullptr, nullptr, nullptr};   // owned: double twiddle tables per axis
    double* f64buf[2] = {nullptr, nullptr};              // owned: complex128 work arrays
    bool split = false;              // the running solve iterates on delta
    double split_eps = 1.0;          // eps at the last re-centering
    int n_recenter = 0;

    // batched solves (R18): n sources share the medium; their u and compact buffers live here
    int batch_n = 1;                 // sources of the running mbs_solve_batch (1: plain solve)
    int batch_cap = 0;
    cf* batch_u = nullptr;
    CorrBufs batch_cx{}, batch_ds{};
    unsigned char* batch_mask = nullptr;

    // subdomain activation (R17)
    int activation = 0;
    bool act_all = false;            // every subdomain of the running solve is active: back to the plain kernels
    double act_threshold = -1.0;     // relative to nu; < 0: tol / 10 of the solve
    ActivationState act{};
    void* act_mem = nullptr;
    int n_sub = 1;
    std::vector<int32_t> act_iter_host;

    // CUDA graph of one poll interval of iterations (small grids are launch-bound)
    cudaGraphExec_t graph_exec = nullptr;
    cudaStream_t cap_stream = nullptr;   // capture happens on a private stream (the caller's may be the default stream)
    const void* graph_y = nullptr;
    const void* graph_x = nullptr;
    int graph_batch = 0, graph_fused = -1, graph_tma = -1, graph_line = -1, graph_split = -1;
    int64_t launches_per_batch = 0;

    int64_t launches = 0;
    std::string err;
};

static thread_local std::string g_create_error;

static int fail(mbs_ctx* ctx, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf;
    else g_create_error = buf;
    return code;
}

#define MBS_CUDA(ctx, expr)                                                                          \
    do {                                                                                             \
        cudaError_t e__ = (expr);                                                                    \
        if (e__ != cudaSuccess)                                                                      \
            return fail(ctx, e__ == cudaErrorMemoryAllocation ? MBS_ERR_OOM : MBS_ERR_CUDA, "%s: %s", #expr, \
                        cudaGetErrorString(e__));                                                    \
    } while (0)

#define MBS_TRY(expr)                    \
    do {                                 \
        int rc__ = (expr);               \
        if (rc__ != MBS_OK) return rc__; \
    } while (0)

// Resolve the pending event pairs (the stream must have been synchronised).
static void prof_drain(mbs_ctx* c) {
    Profiler& p = c->prof;
    for (size_t i = 0; i < p.pending.size(); ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, p.pool[2 * i], p.pool[2 * i + 1]) == cudaSuccess) p.classes[p.pending[i]].ms += ms;
    }
    p.pending.clear();
}

// Brackets one kernel launch: counts it and, in profile mode, records the event pair around it.
struct KernelScope {
    mbs_ctx* c;
    int slot = -1;
    KernelScope(mbs_ctx* ctx, const char* name, double bytes) : c(ctx) {
        c->launches++;
        if (!c->profile) return;
        Profiler& p = c->prof;
        if (p.pending.size() >= 8192) {
            cudaStreamSynchronize(c->stream);
            prof_drain(c);
        }
        const int k = p.find(name);
        p.classes[k].launches++;
        p.classes[k].bytes += bytes;
        slot = (int)p.pending.size();
        while (p.pool.size() < 2 * (size_t)(slot + 1)) {
            cudaEvent_t e = nullptr;
            cudaEventCreate(&e);
            p.pool.push_back(e);
        }
        p.pending.push_back(k);
        cudaEventRecord(p.pool[2 * slot], c->stream);
    }
    ~KernelScope() {
        if (slot >= 0) cudaEventRecord(c->prof.pool[2 * slot + 1], c->stream);
    }
};

// ---------------------------------------------------------------------------------------------
// host-side small linear algebra: sigma_max of the t x t matrix K_t, cyclic Jacobi on K^T K
// ---------------------------------------------------------------------------------------------
static double second_derivative_kernel(int m) {
    // band-limited second derivative on the infinite grid, units 1/h^2 (R4)
    if (m == 0) return -M_PI * M_PI / 3.0;
    return -2.0 * ((m % 2 == 0) ? 1.0 : -1.0) / ((double)m * (double)m);
}

static double sigma_max(const std::vector<double>& K, int t) {
    std::vector<double> A((size_t)t * t, 0.0);  // A = K^T K
    for (int i = 0; i < t; ++i)
        for (int j = 0; j < t; ++j) {
            double s = 0;
            for (int k = 0; k < t; ++k) s += K[(size_t)k * t + i] * K[(size_t)k * t + j];
            A[(size_t)i * t + j] = s;
        }
    for (int sweep = 0; sweep < 100; ++sweep) {
        double off = 0;
        for (int i = 0; i < t; ++i)
            for (int j = i + 1; j < t; ++j) off += A[(size_t)i * t + j] * A[(size_t)i * t + j];
        if (off < 1e-30) break;
        for (int p = 0; p < t; ++p)
            for (int q = p + 1; q < t; ++q) {
                const double apq = A[(size_t)p * t + q];
                if (fabs(apq) < 1e-300) continue;
                const double app = A[(size_t)p * t + p], aqq = A[(size_t)q * t + q];
                const double theta = (aqq - app) / (2.0 * apq);
                const double tt = (theta >= 0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                const double cs = 1.0 / sqrt(tt * tt + 1.0), sn = tt * cs;
                for (int k = 0; k < t; ++k) {
                    const double akp = A[(size_t)k * t + p], akq = A[(size_t)k * t + q];
                    A[(size_t)k * t + p] = cs * akp - sn * akq;
                    A[(size_t)k * t + q] = sn * akp + cs * akq;
                }
                for (int k = 0; k < t; ++k) {
                    const double apk = A[(size_t)p * t + k], aqk = A[(size_t)q * t + k];
                    A[(size_t)p * t + k] = cs * apk - sn * aqk;
                    A[(size_t)q * t + k] = sn * apk + cs * aqk;
                }
            }
    }
    double mx = 0;
    for (int i = 0; i < t; ++i) mx = std::max(mx, A[(size_t)i * t + i]);
    return sqrt(mx);
}

// ---------------------------------------------------------------------------------------------
// workspace layout
// ---------------------------------------------------------------------------------------------
static size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

// A captured graph holds the device pointers of the launches it recorded: drop it whenever one of them changes
// (workspace, residual-history buffer).
static void invalidate_graph(mbs_ctx* c) {
    if (c->graph_exec) {
        cudaGraphExecDestroy(c->graph_exec);
        c->graph_exec = nullptr;
    }
}

static size_t corr_elems(const GridDesc& g, int ax) {
    if (g.a[ax] == 0 || g.t == 0) return 0;
    return (size_t)(g.voxels / g.N[ax]) * g.S[ax] * 2 * g.t;
}

static size_t layout_workspace(mbs_ctx* c, char* base) {
    size_t off = 0;
    auto take = [&](size_t bytes) {
        char* p = base ? base + off : nullptr;
        off += align_up(bytes);
        return p;
    };
    const GridDesc& g = c->g;
    c->bdiag = (cf*)take(sizeof(cf) * g.voxels);
    c->u = (cf*)take(sizeof(cf) * g.voxels);
    for (int ax = 0; ax < 3; ++ax) {
        const size_t n = corr_elems(g, ax);
        c->cx.buf[ax] = n ? (cf*)take(sizeof(cf) * n) : nullptr;
    }
    for (int ax = 0; ax < 3; ++ax) {
        const size_t n = corr_elems(g, ax);
        c->ds.buf[ax] = n ? (cf*)take(sizeof(cf) * n) : nullptr;
    }
    c->partials = (double*)take(sizeof(double) * MBS_MAX_PARTIALS * 5);
    c->ymask = (unsigned char*)take((size_t)(g.voxels / g.N[2]));
    return off;
}

// ---------------------------------------------------------------------------------------------
// create / destroy
// ---------------------------------------------------------------------------------------------
extern "C" int mbs_fft_supported(int64_t M) { return (M > 0 && M < (1 << 30) && fft_lookup((int)M)) ? 1 : 0; }

extern "C" int mbs_create(mbs_ctx** out, int ndim, const int64_t* shape, double pixel_size, double wavelength,
                          const int32_t* boundary_width, const int32_t* n_subdomains, const uint8_t* periodic,
                          int32_t n_correction, void* cuda_stream) {
    if (!out) return fail(nullptr, MBS_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (ndim < 1 || ndim > 3) return fail(nullptr, MBS_ERR_INVALID_ARG, "ndim must be 1, 2 or 3 (got %d)", ndim);
    if (!shape || !boundary_width || !n_subdomains) return fail(nullptr, MBS_ERR_INVALID_ARG, "NULL array argument");
    if (!(pixel_size > 0) || !(wavelength > 0))
        return fail(nullptr, MBS_ERR_INVALID_ARG, "pixel_size and wavelength must be positive");
    if (n_correction < 0) return fail(nullptr, MBS_ERR_INVALID_ARG, "n_correction must be >= 0");

    mbs_ctx* c = new (std::nothrow) mbs_ctx();
    if (!c) return fail(nullptr, MBS_ERR_OOM, "host allocation failed");
    c->ndim = ndim;
    c->first = 3 - ndim;
    c->h = pixel_size;
    c->wavelength = wavelength;
    c->stream = (cudaStream_t)cuda_stream;
    GridDesc& g = c->g;
    g.t = n_correction;
    g.voxels = 1;
    for (int d = 0; d < 3; ++d) { g.N[d] = g.M[d] = g.S[d] = 1; g.a[d] = 0; g.per[d] = 1; c->W[d] = 0; }
    int rc = MBS_OK;
    for (int d = 0; d < ndim && rc == MBS_OK; ++d) {
        const int ax = c->first + d;
        const int64_t N = shape[d];
        const int S = n_subdomains[d], W = boundary_width[d];
        const int per = periodic ? (periodic[d] ? 1 : 0) : 0;
        if (N < 1 || N > (1 << 30)) rc = fail(nullptr, MBS_ERR_INVALID_ARG, "shape[%d] = %lld out of range", d, (long long)N);
        else if (S < 1 || N % S != 0) rc = fail(nullptr, MBS_ERR_INVALID_ARG, "shape[%d] = %lld is not divisible by n_subdomains = %d", d, (long long)N, S);
        else if (W < 0 || 2 * (int64_t)W > N) rc = fail(nullptr, MBS_ERR_INVALID_ARG, "boundary_width[%d] = %d does not fit in %lld voxels", d, W, (long long)N);
        else {
            const int64_t M = N / S;
            g.N[ax] = (int)N; g.S[ax] = S; g.M[ax] = (int)M; g.per[ax] = per; c->W[ax] = W;
            g.a[ax] = (S >= 2) ? 2 : (per ? 0 : 1);
            g.voxels *= N;
            if (g.a[ax] > 0 && n_correction == 0)
                rc = fail(nullptr, MBS_ERR_INVALID_ARG, "n_correction = 0 is legal only when every axis is periodic with one subdomain (axis %d is not)", d);
            else if (g.a[ax] > 0 && 2 * (int64_t)n_correction > M)
                rc = fail(nullptr, MBS_ERR_INVALID_ARG, "2*n_correction = %d exceeds the subdomain length %lld of axis %d", 2 * n_correction, (long long)M, d);
            else if (!fft_lookup((int)M))
                rc = fail(nullptr, MBS_ERR_UNSUPPORTED_SIZE, "no FFT plan for subdomain length %lld (axis %d); supported: 8..1024 powers of two, 40..640 (5*2^k) and 48..768 (3*2^k)", (long long)M, d);
            else c->fft[ax] = fft_lookup((int)M);
        }
    }
    if (rc == MBS_OK && g.voxels >= (1LL << 31)) rc = fail(nullptr, MBS_ERR_INVALID_ARG, "grid has %lld voxels; the limit is 2^31 - 1", g.voxels);
    if (rc != MBS_OK) { delete c; return rc; }
    c->sum_a = g.a[0] + g.a[1] + g.a[2];
    c->n_sub = g.S[0] * g.S[1] * g.S[2];

    // K_t / h^2 and ||A_12|| (R4, R5)
    const int t = g.t;
    c->Kh.assign((size_t)t * t, 0.0);
    std::vector<double> K((size_t)t * t);
    for (int a = 0; a < t; ++a)
        for (int b = 0; b < t; ++b) K[(size_t)a * t + b] = second_derivative_kernel(t + b - a);
    for (size_t i = 0; i < K.size(); ++i) c->Kh[i] = K[i] / (pixel_size * pixel_size);
    c->norm_A12 = t > 0 ? sigma_max(K, t) / (pixel_size * pixel_size) : 0.0;

    auto cleanup_fail = [&](int code, const char* what, cudaError_t e) {
        g_create_error = std::string(what) + ": " + cudaGetErrorString(e);
        mbs_destroy(c);
        return code;
    };
    cudaError_t e;
    int dev = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return cleanup_fail(MBS_ERR_CUDA, "cudaGetDevice", e);
    if ((e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
        return cleanup_fail(MBS_ERR_CUDA, "cudaDeviceGetAttribute", e);
    if ((e = cudaMalloc(&c->state, sizeof(DevState))) != cudaSuccess) return cleanup_fail(MBS_ERR_OOM, "cudaMalloc(state)", e);
    if ((e = cudaMemset(c->state, 0, sizeof(DevState))) != cudaSuccess) return cleanup_fail(MBS_ERR_CUDA, "cudaMemset", e);
    if ((e = cudaMallocHost(&c->state_pinned, 2 * sizeof(DevState))) != cudaSuccess)
        return cleanup_fail(MBS_ERR_OOM, "cudaMallocHost", e);
    for (int i = 0; i < 2; ++i)
        if ((e = cudaEventCreateWithFlags(&c->ev_poll[i], cudaEventDisableTiming)) != cudaSuccess)
            return cleanup_fail(MBS_ERR_CUDA, "cudaEventCreate", e);
    if ((e = cudaEventCreate(&c->ev_t0)) != cudaSuccess || (e = cudaEventCreate(&c->ev_t1)) != cudaSuccess)
        return cleanup_fail(MBS_ERR_CUDA, "cudaEventCreate", e);
    if (t > 0) {
        std::vector<float> Kf(c->Kh.begin(), c->Kh.end());
        if ((e = cudaMalloc(&c->Kh_dev, sizeof(float) * Kf.size())) != cudaSuccess) return cleanup_fail(MBS_ERR_OOM, "cudaMalloc(Kh)", e);
        if ((e = cudaMemcpy(c->Kh_dev, Kf.data(), sizeof(float) * Kf.size(), cudaMemcpyHostToDevice)) != cudaSuccess)
            return cleanup_fail(MBS_ERR_CUDA, "cudaMemcpy(Kh)", e);
    }
    // twiddle tables W_M^n (double precision, rounded once) and p_d^2 = (2 pi fftfreq(M, h))^2 (R9)
    for (int ax = c->first; ax < 3; ++ax) {
        const int M = g.M[ax];
        std::vector<cf> tw(M);
        std::vector<float> p2(M);
        for (int n = 0; n < M; ++n) {
            const double ang = 2.0 * M_PI * (double)n / (double)M;
            tw[n] = make_float2((float)cos(ang), (float)(-sin(ang)));
            const int f = (n < (M + 1) / 2) ? n : n - M;   // numpy fftfreq ordering (Nyquist negative for even M)
            const double p = 2.0 * M_PI * (double)f / ((double)M * pixel_size);
            p2[n] = (float)(p * p);
        }
        if ((e = cudaMalloc(&c->tw_dev[ax], sizeof(cf) * M)) != cudaSuccess) return cleanup_fail(MBS_ERR_OOM, "cudaMalloc(tw)", e);
        if ((e = cudaMalloc(&c->p2_dev[ax], sizeof(float) * M)) != cudaSuccess) return cleanup_fail(MBS_ERR_OOM, "cudaMalloc(p2)", e);
        if ((e = cudaMemcpy(c->tw_dev[ax], tw.data(), sizeof(cf) * M, cudaMemcpyHostToDevice)) != cudaSuccess ||
            (e = cudaMemcpy(c->p2_dev[ax], p2.data(), sizeof(float) * M, cudaMemcpyHostToDevice)) != cudaSuccess)
            return cleanup_fail(MBS_ERR_CUDA, "cudaMemcpy(tables)", e);
    }
    if (ndim >= 2) {
        // per-line part of |p|^2 for the kernel-multiply sweep along the first axis (one float per inner index)
        long long inner = 1;
        for (int ax = c->first + 1; ax < 3; ++ax) inner *= g.N[ax];
        std::vector<float> wt((size_t)inner);
        std::vector<std::vector<double>> p2d(3);
        for (int ax = c->first + 1; ax < 3; ++ax) {
            const int M = g.M[ax];
            p2d[ax].resize(M);
            for (int n = 0; n < M; ++n) {
                const int f = (n < (M + 1) / 2) ? n : n - M;
                const double p = 2.0 * M_PI * (double)f / ((double)M * pixel_size);
                p2d[ax][n] = (double)(float)(p * p);      // the same rounded values as the per-axis tables
            }
        }
        for (long long ii = 0; ii < inner; ++ii) {
            const int i2 = (int)(ii % g.N[2]);
            float w = (float)p2d[2][i2 % g.M[2]];
            if (c->first == 0) w += (float)p2d[1][(int)((ii / g.N[2]) % g.M[1])];
            wt[(size_t)ii] = w;
        }
        if ((e = cudaMalloc(&c->wtab_dev, sizeof(float) * wt.size())) != cudaSuccess) return cleanup_fail(MBS_ERR_OOM, "cudaMalloc(wtab)", e);
        if ((e = cudaMemcpy(c->wtab_dev, wt.data(), sizeof(float) * wt.size(), cudaMemcpyHostToDevice)) != cudaSuccess)
            return cleanup_fail(MBS_ERR_CUDA, "cudaMemcpy(wtab)", e);
    }
    c->ws_bytes = layout_workspace(c, nullptr);
    *out = c;
    return MBS_OK;
}

static void free_batch(mbs_ctx* c) {
    if (c->batch_u) cudaFree(c->batch_u);
    for (int ax = 0; ax < 3; ++ax) {
        if (c->batch_cx.buf[ax]) cudaFree(c->batch_cx.buf[ax]);
        if (c->batch_ds.buf[ax]) cudaFree(c->batch_ds.buf[ax]);
        c->batch_cx.buf[ax] = c->batch_ds.buf[ax] = nullptr;
    }
    if (c->batch_mask) cudaFree(c->batch_mask);
    c->batch_u = nullptr; c->batch_mask = nullptr; c->batch_cap = 0;
}

extern "C" void mbs_destroy(mbs_ctx* c) {
    if (!c) return;
    if (c->ws_owned && c->ws) cudaFree(c->ws);
    if (c->state) cudaFree(c->state);
    if (c->hist_dev) cudaFree(c->hist_dev);
    if (c->Kh_dev) cudaFree(c->Kh_dev);
    if (c->wtab_dev) cudaFree(c->wtab_dev);
    for (int ax = 0; ax < 3; ++ax) {
        if (c->tw_dev[ax]) cudaFree(c->tw_dev[ax]);
        if (c->p2_dev[ax]) cudaFree(c->p2_dev[ax]);
    }
    if (c->state_pinned) cudaFreeHost(c->state_pinned);
    for (int i = 0; i < 2; ++i)
        if (c->ev_poll[i]) cudaEventDestroy(c->ev_poll[i]);
    if (c->ev_t0) cudaEventDestroy(c->ev_t0);
    if (c->ev_t1) cudaEventDestroy(c->ev_t1);
    if (c->host_y) cudaFree(c->host_y);
    if (c->host_x) cudaFree(c->host_x);
    for (cudaEvent_t e : c->prof.pool) cudaEventDestroy(e);
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    if (c->act_mem) cudaFree(c->act_mem);
    free_batch(c);
    if (c->delta) cudaFree(c->delta);
    if (c->dref) cudaFree(c->dref);
    if (c->bdiag64) cudaFree(c->bdiag64);
    if (c->Kh64_dev) cudaFree(c->Kh64_dev);
    for (int i = 0; i < 3; ++i) if (c->tw64_dev[i]) cudaFree(c->tw64_dev[i]);
    for (int i = 0; i < 2; ++i) if (c->f64buf[i]) cudaFree(c->f64buf[i]);
    delete c;
}

extern "C" const char* mbs_last_error(const mbs_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

extern "C" size_t mbs_workspace_bytes(const mbs_ctx* c) { return c ? c->ws_bytes : 0; }

extern "C" int mbs_set_workspace(mbs_ctx* c, void* device_buffer, size_t bytes) {
    if (!c) return MBS_ERR_INVALID_ARG;
    if (!device_buffer || bytes < c->ws_bytes) return fail(c, MBS_ERR_INVALID_ARG, "workspace needs %zu bytes, got %zu", c->ws_bytes, bytes);
    if (((uintptr_t)device_buffer & 255) != 0) return fail(c, MBS_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    if (c->ws_owned && c->ws) cudaFree(c->ws);
    invalidate_graph(c);
    c->ws = device_buffer;
    c->ws_owned = false;
    layout_workspace(c, (char*)c->ws);
    c->potential_set = false;
    return MBS_OK;
}

static int ensure_workspace(mbs_ctx* c) {
    if (c->ws) return MBS_OK;
    MBS_CUDA(c, cudaMalloc(&c->ws, c->ws_bytes));
    c->ws_owned = true;
    layout_workspace(c, (char*)c->ws);
    return MBS_OK;
}

extern "C" int mbs_set_option(mbs_ctx* c, int option, int64_t value) {
    if (!c) return MBS_ERR_INVALID_ARG;
    switch (option) {
        case MBS_OPT_FUSED: c->fused = value ? 1 : 0; return MBS_OK;
        case MBS_OPT_CHECK_INTERVAL:
            if (value < 0 || value > 4096) return fail(c, MBS_ERR_INVALID_ARG, "check interval must be in [0, 4096]");
            c->check_interval = (int)value;
            return MBS_OK;
        case MBS_OPT_USE_GRAPH: c->use_graph = value ? 1 : 0; return MBS_OK;
        case MBS_OPT_PROFILE: c->profile = value ? 1 : 0; return MBS_OK;
        case MBS_OPT_TMA: c->use_tma = value ? 1 : 0; return MBS_OK;
        case MBS_OPT_LINE: c->use_line = value == 2 ? 2 : (value ? 1 : 0); return MBS_OK;
        case MBS_OPT_REFINE: c->refine = value < 0 ? -1 : (value ? 1 : 0); invalidate_graph(c); return MBS_OK;
        default: return fail(c, MBS_ERR_INVALID_ARG, "unknown option %d", option);
    }
}

// ---------------------------------------------------------------------------------------------
// subdomain activation
// ---------------------------------------------------------------------------------------------
static bool fused_available(const mbs_ctx* c);
static bool activation_effective(const mbs_ctx* c) {
    return c->activation && !c->act_all && c->ndim >= 2 && c->fused && fused_available(c) && c->use_line && c->fft[2]->line &&
           slab_pass_supported(c->g.t);
}

extern "C" int mbs_set_activation(mbs_ctx* c, int enable, double threshold) {
    if (!c) return MBS_ERR_INVALID_ARG;
    if (enable && c->ndim < 2) return fail(c, MBS_ERR_INVALID_ARG, "subdomain activation needs a 2-D or 3-D grid");
    if (enable && !(c->fft[2]->line && slab_pass_supported(c->g.t)))
        return fail(c, MBS_ERR_UNSUPPORTED_SIZE, "subdomain activation needs the warp-line sweeps (contiguous subdomain length <= 512... and t in {2, 4, 8, 16})");
    if (enable && !c->act_mem) {
        const size_t ints = (size_t)3 * c->n_sub + 2;
        const size_t bytes = align_up(sizeof(int) * ints) + sizeof(double) * (size_t)c->n_sub * 6 * ACT_CHUNKS;
        MBS_CUDA(c, cudaMalloc(&c->act_mem, bytes));
        MBS_CUDA(c, cudaMemset(c->act_mem, 0, bytes));
        int* ip = (int*)c->act_mem;
        c->act.flags = ip; c->act.list = ip + c->n_sub; c->act.act_iter = ip + 2 * c->n_sub;
        c->act.n_act = ip + 3 * c->n_sub; c->act.ticket = (unsigned int*)(ip + 3 * c->n_sub + 1);
        c->act.partials = (double*)((char*)c->act_mem + align_up(sizeof(int) * ints));
    }
    invalidate_graph(c);
    c->activation = enable ? 1 : 0;
    c->act_threshold = threshold;
    return MBS_OK;
}

extern "C" int mbs_get_activation(const mbs_ctx* c, int32_t* activated_at, int32_t capacity, int32_t* n_subdomains) {
    if (!c || !n_subdomains) return MBS_ERR_INVALID_ARG;
    *n_subdomains = c->n_sub;
    for (int i = 0; i < c->n_sub && i < capacity && activated_at; ++i)
        activated_at[i] = i < (int)c->act_iter_host.size() ? c->act_iter_host[i] : 0;
    return MBS_OK;
}

// ---------------------------------------------------------------------------------------------
// set_potential (a0 of the scope table)
// ---------------------------------------------------------------------------------------------
// grids on which the split iterate may run (small, L2-resident: configs 1 and 2) get the double-precision tables
static bool split_grid(const mbs_ctx* c) { return c->refine == 1 || (c->refine < 0 && c->g.voxels <= (1LL << 21)); }

extern "C" int mbs_set_potential(mbs_ctx* c, const void* n_map_device) {
    if (!c) return MBS_ERR_INVALID_ARG;
    if (!n_map_device) return fail(c, MBS_ERR_INVALID_ARG, "n_map is NULL");
    invalidate_graph(c);                              // the scale factor c is recorded by value in the launches
    c->potential_set = false;
    MBS_TRY(ensure_workspace(c));
    const GridDesc& g = c->g;
    SetupParams sp{};
    sp.n_map = (const cf*)n_map_device;
    const double kw = 2.0 * M_PI / c->wavelength;
    sp.kw2 = kw * kw;
    sp.beta = c->beta;
    for (int d = 0; d < 3; ++d) sp.W[d] = c->W[d];
    int nblocks = (int)std::min<long long>((g.voxels + 255) / 256, (long long)std::min(MBS_MAX_PARTIALS, c->num_sms * 8));
    std::vector<double> host(5 * (size_t)nblocks);
    const double vb = 8.0 * (double)g.voxels;
    { KernelScope ks(c, "setup_minmax", vb); MBS_CUDA(c, launch_setup(g, sp, 0, c->partials, nullptr, nblocks, c->stream)); }
    MBS_CUDA(c, cudaMemcpyAsync(host.data(), c->partials, sizeof(double) * 5 * nblocks, cudaMemcpyDeviceToHost, c->stream));
    MBS_CUDA(c, cudaStreamSynchronize(c->stream));
    double mn_re = INFINITY, mx_re = -INFINITY, mn_im = INFINITY, mx_im = -INFINITY, mn_n = INFINITY;
    for (int b = 0; b < nblocks; ++b) {
        mn_re = std::min(mn_re, host[5 * b + 0]); mx_re = std::max(mx_re, host[5 * b + 1]);
        mn_im = std::min(mn_im, host[5 * b + 2]); mx_im = std::max(mx_im, host[5 * b + 3]);
        mn_n = std::min(mn_n, host[5 * b + 4]);
    }
    if (!(mn_re == mn_re) || !std::isfinite(mn_re) || !std::isfinite(mx_re) || !std::isfinite(mx_im))
        return fail(c, MBS_ERR_NUMERIC, "refractive-index map contains NaN or Inf");
    if (mn_n < 0.0) return fail(c, MBS_ERR_INVALID_ARG, "Im n < 0 (gain) violates the convergence condition (min Im n = %g)", mn_n);
    // R2: k0^2 = centre of the bounding box of k^2
    c->k02 = cd(0.5 * (mn_re + mx_re), 0.5 * (mn_im + mx_im));
    sp.k02_re = c->k02.real();
    sp.k02_im = c->k02.imag();
    { KernelScope ks(c, "setup_vmax", vb); MBS_CUDA(c, launch_setup(g, sp, 1, c->partials, nullptr, nblocks, c->stream)); }
    MBS_CUDA(c, cudaMemcpyAsync(host.data(), c->partials, sizeof(double) * nblocks, cudaMemcpyDeviceToHost, c->stream));
    MBS_CUDA(c, cudaStreamSynchronize(c->stream));
    double v2 = 0;
    for (int b = 0; b < nblocks; ++b) v2 = std::max(v2, host[b]);
    c->v_max = sqrt(v2);
    const double denom = c->v_max + (double)c->sum_a * c->norm_A12;   // Eq. (9)
    if (!(denom > 0)) return fail(c, MBS_ERR_INVALID_ARG, "homogeneous medium without corrections: ||V|| = 0, nothing to scale");
    c->c = cd(0.0, -0.95 / denom);
    sp.c_re = c->c.real();
    sp.c_im = c->c.imag();
    if (split_grid(c) && !c->bdiag64) MBS_CUDA(c, cudaMalloc(&c->bdiag64, 2 * sizeof(double) * (size_t)g.voxels));
    sp.bdiag64 = c->bdiag64;
    { KernelScope ks(c, "setup_bdiag", 2 * vb); MBS_CUDA(c, launch_setup(g, sp, 2, nullptr, c->bdiag, nblocks, c->stream)); }
    MBS_CUDA(c, cudaStreamSynchronize(c->stream));
    c->potential_set = true;
    return MBS_OK;
}

// ---------------------------------------------------------------------------------------------
// building blocks
// ---------------------------------------------------------------------------------------------
static cf to_cf(cd z) { return make_float2((float)z.real(), (float)z.imag()); }

// edge corrections of (in - in2) into c->cx  (a2 / a7 of the scope table)
static int run_slabs(mbs_ctx* c, const cf* in, const cf* in2, bool in_loop, int axis_mask = 7, bool from_ds = false) {
    auto params = [&](int ax) {
        SlabParams sp{};
        sp.in = from_ds ? c->ds.buf[ax] : in; sp.in2 = in2; sp.out = c->cx.buf[ax]; sp.Kh = c->Kh_dev; sp.c = to_cf(c->c); sp.axis = ax;
        sp.compact_in = from_ds ? 1 : 0;
        sp.state = c->state; sp.check_done = in_loop ? 1 : 0;
        return sp;
    };
    if (c->cx.buf[0] && c->cx.buf[1] && (axis_mask & 3) == 3 && slab_pair_supported(c->g.t)) {
        // axes 0 and 1 in one launch
        const SlabParams pA = params(0), pB = params(1);
        KernelScope ks(c, "slab_ax01", (in2 ? 24.0 : 16.0) * ((double)corr_elems(c->g, 0) + (double)corr_elems(c->g, 1)));
        MBS_CUDA(c, launch_slab_pair(c->g, pA, pB, c->stream));
        axis_mask &= ~3;
    }
    for (int ax = 0; ax < 3; ++ax) {
        if (!c->cx.buf[ax] || !((axis_mask >> ax) & 1)) continue;
        const SlabParams sp = params(ax);
        static const char* names[3] = {"slab_ax0", "slab_ax1", "slab_ax2"};
        KernelScope ks(c, names[ax], (in2 ? 24.0 : 16.0) * (double)corr_elems(c->g, ax));
        MBS_CUDA(c, launch_slab(c->g, sp, c->stream));
    }
    return MBS_OK;
}

static PointwiseParams pw_defaults(mbs_ctx* c, bool in_loop) {
    PointwiseParams p{};
    p.s1 = 1.f; p.s2 = 0.f; p.alpha = (float)c->alpha;
    p.ysc = make_float2(0.f, 0.f);
    p.partials = c->partials; p.hist = c->hist_dev; p.state = c->state;
    p.check_done = in_loop ? 1 : 0;
    return p;
}

static SymbolParams make_symbol(const mbs_ctx* c, int inverse) {
    const GridDesc& g = c->g;
    SymbolParams sp{};
    const cd ck = c->c * c->k02;
    sp.A0 = (float)(ck.real() + 1.0);
    sp.B0 = (float)ck.imag();
    sp.cr = (float)c->c.real();
    sp.ci = (float)c->c.imag();
    sp.scale = (float)(1.0 / ((double)g.M[0] * g.M[1] * g.M[2]));   // 1/M of the inverse transforms (R9)
    sp.inverse = inverse;
    return sp;
}

// FFT sweep along the contiguous axis, in place on buf
static int run_fft_contig(mbs_ctx* c, cf* buf, int mode, int inverse, bool in_loop) {
    const GridDesc& g = c->g;
    ContigGeom cg{};
    const FftEntry* e = c->fft[2];
    cg.n_lines = g.voxels / g.M[2];
    cg.n_tiles = (cg.n_lines + e->CC - 1) / e->CC;
    SymbolParams s2 = make_symbol(c, inverse);
    s2.tab_axis = c->p2_dev[2];
    static const char* names[3] = {"fft_contig_fwd", "fft_contig_inv", "fft_contig_mid"};
    KernelScope ks(c, names[mode], 16.0 * (double)g.voxels);
    MBS_CUDA(c, e->contig(buf, buf, cg, s2, c->tw_dev[2], mode, in_loop ? &c->state->done : nullptr, c->num_sms, c->stream));
    return MBS_OK;
}

// FFT sweep along strided axis ax (0 or 1), in place on buf
// n_rep > 1: `buf` holds n_rep fields one after the other (batched solves): the batch is one more outer dimension
static int run_fft_strided(mbs_ctx* c, cf* buf, int ax, int mode, int inverse, bool in_loop, int n_rep = 1) {
    const GridDesc& g = c->g;
    const FftEntry* e = c->fft[ax];
    StridedGeom sg{};
    long long inner = 1, outer = n_rep;
    for (int d = ax + 1; d < 3; ++d) inner *= g.N[d];
    for (int d = 0; d < ax; ++d) outer *= g.N[d];
    sg.stride = inner; sg.outer_stride = (long long)g.N[ax] * inner; sg.n_outer = (int)outer; sg.n_seg = g.S[ax];
    const int cs = (mode == FFT_MID) ? e->CSM : e->CS;
    sg.inner = (int)inner; sg.tiles_inner = (int)((inner + cs - 1) / cs);
    sg.n_tiles = outer * g.S[ax] * sg.tiles_inner;
    if (in_loop && n_rep == 1 && activation_effective(c) && g.M[2] % cs == 0) {
        // visit only the tiles of the active subdomains (their list lives in device memory)
        sg.act_list = c->act.list; sg.n_act = c->act.n_act; sg.axis = ax;
        sg.tps2 = g.M[2] / cs; sg.tiles_per_sub = (ax == 1 ? g.M[0] : g.M[1]) * sg.tps2;
        sg.S1 = g.S[1]; sg.S2 = g.S[2]; sg.M0 = g.M[0]; sg.M1 = g.M[1]; sg.row_tiles = g.N[2] / cs;
    }
    SymbolParams s2 = make_symbol(c, inverse);
    s2.tab_axis = c->p2_dev[ax];
    if (mode == FFT_MID) {
        // line-invariant part of |p|^2 from the axes after `ax`
        if (ax == 0) { s2.tabA = c->p2_dev[1]; s2.Ma = g.M[1]; s2.tabB = c->p2_dev[2]; s2.Mb = g.M[2]; s2.Nb = g.N[2]; }
        else { s2.tabA = nullptr; s2.Ma = 1; s2.tabB = c->p2_dev[2]; s2.Mb = g.M[2]; s2.Nb = g.N[2]; }
        if (ax == c->first) s2.wtab = c->wtab_dev;
    }
    static const char* names[2][3] = {{"fft_strided_fwd_ax0", "fft_strided_inv_ax0", "fft_strided_mid_ax0"},
                                      {"fft_strided_fwd_ax1", "fft_strided_inv_ax1", "fft_strided_mid_ax1"}};
    KernelScope ks(c, names[ax][mode], 16.0 * (double)g.voxels * n_rep);
    MBS_CUDA(c, e->strided(buf, sg, s2, c->tw_dev[ax], mode, in_loop ? &c->state->done : nullptr, c->num_sms, c->use_tma,
                           c->stream));
    return MBS_OK;
}

// the sweeps between the first and the last one: strided forward, kernel multiply, strided inverse (a3-a5)
static int run_middle_sweeps(mbs_ctx* c, cf* buf, int inverse, bool in_loop, int n_rep = 1) {
    if (c->ndim == 3) MBS_TRY(run_fft_strided(c, buf, 1, FFT_FWD, inverse, in_loop, n_rep));
    MBS_TRY(run_fft_strided(c, buf, c->first, FFT_MID, inverse, in_loop, n_rep));
    if (c->ndim == 3) MBS_TRY(run_fft_strided(c, buf, 1, FFT_INV, inverse, in_loop, n_rep));
    return MBS_OK;
}

// (L+I)^-1 (inverse = 1) or (L+I) (inverse = 0) in place on buf  (a3-a5 of the scope table)
static int run_propagator(mbs_ctx* c, cf* buf, int inverse, bool in_loop) {
    if (c->ndim == 1) return run_fft_contig(c, buf, FFT_MID, inverse, in_loop);
    MBS_TRY(run_fft_contig(c, buf, FFT_FWD, inverse, in_loop));
    MBS_TRY(run_middle_sweeps(c, buf, inverse, in_loop));
    return run_fft_contig(c, buf, FFT_INV, inverse, in_loop);
}

// out = s1 * [B_diag (in - in2) + ysc*y - corr(in - in2)] + s2*w
static int run_B(mbs_ctx* c, const cf* in, const cf* in2, const cf* y, cf ysc, cf* out, float s1, const cf* w, float s2,
                 int reduce, bool in_loop) {
    MBS_TRY(run_slabs(c, in, in2, in_loop));
    PointwiseParams p = pw_defaults(c, in_loop);
    p.in = in; p.in2 = in2; p.bdiag = c->bdiag; p.y = y; p.ysc = ysc; p.out = out; p.s1 = s1; p.w = w; p.s2 = s2;
    p.corr = c->cx; p.reduce = reduce;
    const int n_arrays = 2 + (in2 ? 1 : 0) + (y ? 1 : 0) + (w ? 1 : 0) + (out ? 1 : 0);
    KernelScope ks(c, y ? "pointwise_Bx_plus_y" : "pointwise_B", 8.0 * n_arrays * (double)c->g.voxels);
    MBS_CUDA(c, launch_pointwise(c->g, p, c->num_sms, c->stream));
    return MBS_OK;
}

// one iteration of Eq. (6), unfused: one kernel per step of P:122-128
static int run_iteration_unfused(mbs_ctx* c, const cf* y, cf* x) {
    const cf ysc = to_cf(-c->c);                                                   // y_vec = -c y
    MBS_TRY(run_B(c, x, nullptr, y, ysc, c->u, 1.f, nullptr, 0.f, RED_NONE, true));  // u = B x + y_vec
    MBS_TRY(run_propagator(c, c->u, 1, true));                                     // u' = (L+I)^-1 u
    MBS_TRY(run_slabs(c, x, c->u, true));                                          // corr(x - u')
    PointwiseParams p = pw_defaults(c, true);                                      // r = B (x - u'); x -= alpha r
    p.in = x; p.in2 = c->u; p.bdiag = c->bdiag; p.out = x; p.corr = c->cx; p.update = 1; p.reduce = RED_RESIDUAL;
    KernelScope ks(c, "pointwise_update", 32.0 * (double)c->g.voxels);
    MBS_CUDA(c, launch_pointwise(c->g, p, c->num_sms, c->stream));
    return MBS_OK;
}

// The fused path needs whole grid rows inside one tile of the contiguous-axis kernel.
static bool fused_available(const mbs_ctx* c) { return c->fft[2]->fused != nullptr && c->fft[2]->CC % c->g.S[2] == 0; }

// one iteration of Eq. (6), fused sweeps (112 B/voxel ledger of DESIGN.md section 5)
static int run_iteration_fused(mbs_ctx* c, const cf* y, cf* x) {
    const GridDesc& g = c->g;
    const FftEntry* e = c->fft[2];
    if (c->split) {   // split iterate: the sweeps run on delta with no source; the last sweep adds d_ref (recenter())
        y = nullptr;
        x = c->delta;
    }
    const int e0 = g.a[0] > 0, e1 = g.a[1] > 0;
    const int* done = &c->state->done;
    FusedParams p{};
    p.x = x; p.bdiag = c->bdiag; p.y = y; p.ymask = c->ymask; p.ysc = to_cf(-c->c); p.u = c->u;
    p.N0 = g.N[0]; p.S0 = g.S[0];
    p.N1 = g.N[1]; p.N2 = g.N[2]; p.S2 = g.S[2]; p.a2 = g.a[2]; p.per2 = g.per[2]; p.t = g.t;
    p.e0 = e0; p.e1 = e1; p.M0 = g.M[0]; p.M1 = g.M[1]; p.S1 = g.S[1];
    p.cx0 = c->cx.buf[0]; p.cx1 = c->cx.buf[1]; p.ds0 = c->ds.buf[0]; p.ds1 = c->ds.buf[1];
    p.Kh = c->Kh_dev; p.c = to_cf(c->c); p.alpha = (float)c->alpha;
    p.sp = make_symbol(c, 1); p.sp.tab_axis = c->p2_dev[2];
    p.n_lines = g.voxels / g.M[2];
    p.n_tiles = (p.n_lines + e->CC - 1) / e->CC;
    p.partials = c->partials; p.state = c->state; p.hist = c->hist_dev; p.reduce_mode = RED_RESIDUAL;
    p.dref = (c->split && !c->bdiag64) ? c->dref : nullptr;
    p.rref = (c->split && c->bdiag64) ? c->dref : nullptr;
    p.line_variant = c->use_line == 2 ? 1 : 0;
    const double vb = 8.0 * (double)g.voxels;
    if (c->ndim == 1) {
        p.slot0 = 0; p.finish = 1;
        p.n_total = e->fused_blocks(FUSED_1D, g.t, p.n_tiles, c->num_sms);
        KernelScope ks(c, "fused_1d", (3.0 + c->y_row_fraction) * vb);
        MBS_CUDA(c, e->fused(p, c->tw_dev[2], FUSED_1D, done, c->num_sms, c->stream));
        return MBS_OK;
    }
    const int mask01 = (e0 ? 1 : 0) | (e1 ? 2 : 0);
    const bool act_on = activation_effective(c);
    if (act_on) {
        // before the update, activate the inactive subdomains whose transferred norm reached the threshold
        KernelScope ks(c, "activation_step", 0.0);
        MBS_CUDA(c, launch_activation_step(g, c->act, x, c->Kh_dev, to_cf(c->c), c->state, c->stream));
        p.active = c->act.flags;
    }
    if (mask01) MBS_TRY(run_slabs(c, x, nullptr, true, mask01));                      // corr_0(x), corr_1(x)
    if (c->use_line && e->line) {
        // warp-line sweeps: corr_2(x) inside sweep 1; corr_2(d) through the compact buffers like axes 0 and 1
        const int e2 = g.a[2] > 0 ? 1 : 0;
        p.ds2 = c->ds.buf[2];
        {
            KernelScope ks(c, "line_sweep1", (3.0 + c->y_row_fraction) * vb);     // all-zero rows of y are not read
            MBS_CUDA(c, e->line(p, c->tw_dev[2], LINE_S1, done, c->num_sms, c->stream));
        }
        MBS_TRY(run_middle_sweeps(c, c->u, 1, true));
        const int nb5 = e->line_blocks(LINE_S5, g.t, p.line_variant, p.n_lines, c->num_sms);
        if (nb5 < 1) return fail(c, MBS_ERR_CUDA, "line sweep: occupancy query failed");
        const int mask = mask01 | (e2 ? 4 : 0);
        p.slot0 = 0; p.n_total = nb5; p.finish = mask ? 0 : 1;
        {
            KernelScope ks(c, "line_sweep5", 4 * vb);
            MBS_CUDA(c, e->line(p, c->tw_dev[2], LINE_S5, done, c->num_sms, c->stream));
        }
        if (mask && slab_pass_supported(g.t)) {
            // one pass per axis: corr_ax(d) from the compact d, applied in the same kernel; the last pass finishes
            int slot = nb5, last_ax = (mask & 4) ? 2 : ((mask & 2) ? 1 : 0);
            for (int ax = 0; ax < 3; ++ax) {
                if (!((mask >> ax) & 1)) continue;
                SlabPassParams sp{};
                sp.ds = c->ds.buf[ax]; sp.u = c->u; sp.x = x; sp.Kh = c->Kh_dev; sp.c = to_cf(c->c); sp.axis = ax;
                sp.e1 = e1; sp.e2 = e2; sp.alpha = (float)c->alpha; sp.partials = c->partials; sp.slot0 = slot;
                sp.finish = (ax == last_ax) ? 1 : 0; sp.state = c->state; sp.hist = c->hist_dev;
                sp.active = act_on ? c->act.flags : nullptr;
                static const char* names[3] = {"slab_pass_ax0", "slab_pass_ax1", "slab_pass_ax2"};
                KernelScope ks(c, names[ax], 40.0 * (double)corr_elems(g, ax));
                MBS_CUDA(c, launch_slab_pass(g, sp, c->stream));
                slot += slab_pass_blocks(g, ax);
            }
        } else if (mask) {
            MBS_TRY(run_slabs(c, nullptr, nullptr, true, mask, true));                // corr_d(d) from the compact d
            FixupParams f{};
            f.x = x; f.u = c->u; f.cx0 = c->cx.buf[0]; f.cx1 = c->cx.buf[1]; f.cx2 = c->cx.buf[2];
            f.e0 = e0; f.e1 = e1; f.e2 = e2; f.alpha = (float)c->alpha;
            f.partials = c->partials; f.slot0 = nb5; f.reduce_mode = RED_RESIDUAL; f.state = c->state; f.hist = c->hist_dev;
            f.check_done = 1;
            const double vox = (double)corr_elems(g, 0) + (double)corr_elems(g, 1) + (double)corr_elems(g, 2);
            KernelScope ks(c, "fixup_slab_voxels", 32.0 * vox);
            MBS_CUDA(c, launch_fixup(g, f, fixup_blocks(g, e0, e1, e2, c->num_sms), c->stream));
        }
        return MBS_OK;
    }
    {
        KernelScope ks(c, "fused_sweep1", (3.0 + c->y_row_fraction) * vb);           // reads x, B_diag, y (non-empty rows); writes u
        MBS_CUDA(c, e->fused(p, c->tw_dev[2], FUSED_S1, done, c->num_sms, c->stream));
    }
    MBS_TRY(run_middle_sweeps(c, c->u, 1, true));
    const int nb5 = e->fused_blocks(FUSED_S5, g.t, p.n_tiles, c->num_sms);
    if (nb5 < 1) return fail(c, MBS_ERR_CUDA, "fused sweep: occupancy query failed");
    p.slot0 = 0; p.n_total = nb5; p.finish = mask01 ? 0 : 1;
    {
        KernelScope ks(c, "fused_sweep5", 4 * vb);                                    // reads u, x, B_diag; writes x
        MBS_CUDA(c, e->fused(p, c->tw_dev[2], FUSED_S5, done, c->num_sms, c->stream));
    }
    if (mask01) {
        MBS_TRY(run_slabs(c, nullptr, nullptr, true, mask01, true));                  // corr_0(d), corr_1(d) from the compact d
        FixupParams f{};
        f.x = x; f.u = c->u; f.cx0 = c->cx.buf[0]; f.cx1 = c->cx.buf[1]; f.cx2 = nullptr; f.e0 = e0; f.e1 = e1; f.e2 = 0;
        f.alpha = (float)c->alpha;
        f.partials = c->partials; f.slot0 = nb5; f.reduce_mode = RED_RESIDUAL; f.state = c->state; f.hist = c->hist_dev;
        f.check_done = 1;
        const double rows = (double)corr_elems(g, 0) + (double)corr_elems(g, 1);
        KernelScope ks(c, "fixup_slab_rows", 40.0 * rows);
        MBS_CUDA(c, launch_fixup(g, f, fixup_blocks(g, e0, e1, 0, c->num_sms), c->stream));
    }
    return MBS_OK;
}

// ---------------------------------------------------------------------------------------------
// Batched solves (one system per source, the same A; reading R18 of DESIGN.md section 3).  x and y hold n sources
// one after the other.  Every source runs Eq. (6) exactly as a plain solve; the warp-line sweeps take the sources
// of a batch one after the other on the same line, so B_diag is read from DRAM once per line and iteration instead of
// once per source (112 -> 96 + 16/n bytes per voxel-iteration and source); the strided sweeps see the batch as one more
// outer dimension; one residual of the stacked system decides the stop.
// ---------------------------------------------------------------------------------------------
static bool batch_available(const mbs_ctx* c) {
    return c->ndim >= 2 && c->fused && fused_available(c) && c->use_line && c->fft[2]->line && slab_pass_supported(c->g.t);
}

static int ensure_batch(mbs_ctx* c, int n) {
    if (n <= c->batch_cap) return MBS_OK;
    free_batch(c);
    const GridDesc& g = c->g;
    MBS_CUDA(c, cudaMalloc(&c->batch_u, sizeof(cf) * (size_t)n * (size_t)g.voxels));
    for (int ax = 0; ax < 3; ++ax) {
        const size_t ne = corr_elems(g, ax);
        if (!ne) continue;
        MBS_CUDA(c, cudaMalloc(&c->batch_cx.buf[ax], sizeof(cf) * ne * n));
        MBS_CUDA(c, cudaMalloc(&c->batch_ds.buf[ax], sizeof(cf) * ne * n));
    }
    MBS_CUDA(c, cudaMalloc(&c->batch_mask, (size_t)n * (size_t)(g.voxels / g.N[2])));
    c->batch_cap = n;
    return MBS_OK;
}

static int run_iteration_batch(mbs_ctx* c, const cf* y, cf* x) {
    const GridDesc& g = c->g;
    const FftEntry* e = c->fft[2];
    const int nb = c->batch_n;
    const int e0 = g.a[0] > 0, e1 = g.a[1] > 0, e2 = g.a[2] > 0 ? 1 : 0;
    const int* done = &c->state->done;
    const double vb = 8.0 * (double)g.voxels;
    FusedParams p{};
    p.x = x; p.bdiag = c->bdiag; p.y = y; p.ymask = c->batch_mask; p.ysc = to_cf(-c->c); p.u = c->batch_u;
    p.N0 = g.N[0]; p.S0 = g.S[0];
    p.N1 = g.N[1]; p.N2 = g.N[2]; p.S2 = g.S[2]; p.a2 = g.a[2]; p.per2 = g.per[2]; p.t = g.t;
    p.e0 = e0; p.e1 = e1; p.M0 = g.M[0]; p.M1 = g.M[1]; p.S1 = g.S[1];
    p.cx0 = c->batch_cx.buf[0]; p.cx1 = c->batch_cx.buf[1];
    p.ds0 = c->batch_ds.buf[0]; p.ds1 = c->batch_ds.buf[1]; p.ds2 = c->batch_ds.buf[2];
    p.Kh = c->Kh_dev; p.c = to_cf(c->c); p.alpha = (float)c->alpha;
    p.n_lines = g.voxels / g.M[2];
    p.partials = c->partials; p.state = c->state; p.hist = c->hist_dev; p.reduce_mode = RED_RESIDUAL;
    p.line_variant = c->use_line == 2 ? 1 : 0;
    p.n_batch = nb; p.batch_stride = g.voxels; p.mask_stride = g.voxels / g.N[2];
    for (int ax = 0; ax < 3; ++ax) p.cstride[ax] = (long long)corr_elems(g, ax);
    // corr_0(x), corr_1(x) of every source
    for (int ax = 0; ax < 2; ++ax) {
        if (!c->batch_cx.buf[ax]) continue;
        SlabParams sp{};
        sp.in = x; sp.out = c->batch_cx.buf[ax]; sp.Kh = c->Kh_dev; sp.c = to_cf(c->c); sp.axis = ax;
        sp.state = c->state; sp.check_done = 1;
        sp.n_batch = nb; sp.in_stride = g.voxels; sp.out_stride = (long long)corr_elems(g, ax);
        static const char* names[2] = {"slab_ax0", "slab_ax1"};
        KernelScope ks(c, names[ax], 16.0 * (double)corr_elems(g, ax) * nb);
        MBS_CUDA(c, launch_slab(g, sp, c->stream));
    }
    {
        KernelScope ks(c, "line_sweep1", (2.0 + c->y_row_fraction) * vb * nb + vb);      // B_diag once per batch
        MBS_CUDA(c, e->line(p, c->tw_dev[2], LINE_S1, done, c->num_sms, c->stream));
    }
    MBS_TRY(run_middle_sweeps(c, c->batch_u, 1, true, nb));
    const int nb5 = e->line_blocks(LINE_S5, g.t, p.line_variant, p.n_lines, c->num_sms);
    if (nb5 < 1) return fail(c, MBS_ERR_CUDA, "line sweep: occupancy query failed");
    const int mask = (e0 ? 1 : 0) | (e1 ? 2 : 0) | (e2 ? 4 : 0);
    p.slot0 = 0; p.n_total = nb5; p.finish = mask ? 0 : 1;
    {
        KernelScope ks(c, "line_sweep5", 3 * vb * nb + vb);
        MBS_CUDA(c, e->line(p, c->tw_dev[2], LINE_S5, done, c->num_sms, c->stream));
    }
    int slot = nb5;
    const int last_ax = (mask & 4) ? 2 : ((mask & 2) ? 1 : 0);
    for (int ax = 0; ax < 3; ++ax) {
        if (!((mask >> ax) & 1)) continue;
        SlabPassParams sp{};
        sp.ds = c->batch_ds.buf[ax]; sp.u = c->batch_u; sp.x = x; sp.Kh = c->Kh_dev; sp.c = to_cf(c->c); sp.axis = ax;
        sp.e1 = e1; sp.e2 = e2; sp.alpha = (float)c->alpha; sp.partials = c->partials; sp.slot0 = slot;
        sp.finish = (ax == last_ax) ? 1 : 0; sp.state = c->state; sp.hist = c->hist_dev;
        sp.n_batch = nb; sp.ds_stride = (long long)corr_elems(g, ax); sp.vox_stride = g.voxels;
        static const char* names[3] = {"slab_pass_ax0", "slab_pass_ax1", "slab_pass_ax2"};
        KernelScope ks(c, names[ax], 40.0 * (double)corr_elems(g, ax) * nb);
        MBS_CUDA(c, launch_slab_pass(g, sp, c->stream));
        slot += slab_pass_blocks(g, ax);
    }
    return MBS_OK;
}

static int run_iteration(mbs_ctx* c, const cf* y, cf* x) {
    if (c->batch_n > 1) return run_iteration_batch(c, y, x);
    return (c->fused && fused_available(c)) ? run_iteration_fused(c, y, x) : run_iteration_unfused(c, y, x);
}

// ---------------------------------------------------------------------------------------------
// apply_operator
// ---------------------------------------------------------------------------------------------
extern "C" int mbs_apply_operator(mbs_ctx* c, int which, const void* in_device, void* out_device) {
    if (!c) return MBS_ERR_INVALID_ARG;
    if (!c->potential_set) return fail(c, MBS_ERR_STATE, "mbs_set_potential has not been called");
    if (!in_device || !out_device) return fail(c, MBS_ERR_INVALID_ARG, "NULL array argument");
    const cf* in = (const cf*)in_device;
    cf* out = (cf*)out_device;
    const cf zero = make_float2(0.f, 0.f);
    switch (which) {
        case MBS_OP_B:
            return run_B(c, in, nullptr, nullptr, zero, out, 1.f, nullptr, 0.f, RED_NONE, false);
        case MBS_OP_PROPAGATOR:
            if (in != out) MBS_CUDA(c, cudaMemcpyAsync(out, in, sizeof(cf) * c->g.voxels, cudaMemcpyDeviceToDevice, c->stream));
            return run_propagator(c, out, 1, false);
        case MBS_OP_A:
            // A in = (L+I) in - B in
            MBS_CUDA(c, cudaMemcpyAsync(c->u, in, sizeof(cf) * c->g.voxels, cudaMemcpyDeviceToDevice, c->stream));
            MBS_TRY(run_propagator(c, c->u, 0, false));
            return run_B(c, in, nullptr, nullptr, zero, out, -1.f, c->u, 1.f, RED_NONE, false);
        case MBS_OP_PRECOND_A:
            // Gamma^-1 A in = B (in - (L+I)^-1 B in)
            MBS_TRY(run_B(c, in, nullptr, nullptr, zero, c->u, 1.f, nullptr, 0.f, RED_NONE, false));
            MBS_TRY(run_propagator(c, c->u, 1, false));
            return run_B(c, in, c->u, nullptr, zero, out, 1.f, nullptr, 0.f, RED_NONE, false);
        default:
            return fail(c, MBS_ERR_INVALID_ARG, "unknown operator %d", which);
    }
}

// ---------------------------------------------------------------------------------------------
// solve
// ---------------------------------------------------------------------------------------------
// ---------------------------------------------------------------------------------------------
// Split iterate ("a compensated (hi + lo) x in the small, L2-resident configs").  The residual of Eq. (6),
// r = B (x - (L+I)^-1 (B x + y_vec)), is a cancellation: the fp32 FFT of a field of size |x| leaves noise of about
// 3e-7 |x| in it, a floor of (1-3)e-7 ||x|| / ||Gamma^-1 y|| under the relative residual (above config 1's tol of 1e-6).
// Writing x = x_ref + delta with x_ref frozen, linearity gives
//     x - (L+I)^-1 (B x + y_vec) = [x_ref - (L+I)^-1 (B x_ref + y_vec)] + [delta - (L+I)^-1 B delta] = d_ref + (delta - u'),
// the same d as Eq. (6) in exact arithmetic, so the iteration, its residuals and its iteration count are unchanged; but
// the FFT now acts on delta only and its rounding noise scales with |delta|, which shrinks as the iteration converges.
// d_ref is computed once per re-centering (x_ref += delta, delta = 0), a few times per solve, when the residual has
// dropped by two orders of magnitude.  Costs two extra arrays; the sweeps move the same bytes (the last sweep reads
// d_ref, the first one reads no source).  Used on grids of <= 2^21 voxels (configs 1 and 2) unless MBS_OPT_REFINE says otherwise.
// ---------------------------------------------------------------------------------------------
static bool split_effective(const mbs_ctx* c) {
    const bool want = c->refine == 1 || (c->refine < 0 && c->g.voxels <= (1LL << 21));
    return want && c->fused && fused_available(c) && !c->activation && c->batch_n == 1;
}

// double tables and work arrays of refine_f64.cu (once per context)
static int ensure_f64_tables(mbs_ctx* c) {
    const GridDesc& g = c->g;
    if (!c->Kh64_dev && g.t > 0) {
        MBS_CUDA(c, cudaMalloc(&c->Kh64_dev, sizeof(double) * c->Kh.size()));
        MBS_CUDA(c, cudaMemcpy(c->Kh64_dev, c->Kh.data(), sizeof(double) * c->Kh.size(), cudaMemcpyHostToDevice));
    }
    for (int ax = c->first; ax < 3; ++ax) {
        if (c->tw64_dev[ax]) continue;
        const int M = g.M[ax];
        std::vector<double> tw(2 * (size_t)M);
        for (int n = 0; n < M; ++n) {
            const double ang = 2.0 * M_PI * (double)n / (double)M;
            tw[2 * n] = cos(ang);
            tw[2 * n + 1] = -sin(ang);
        }
        MBS_CUDA(c, cudaMalloc(&c->tw64_dev[ax], sizeof(double) * tw.size()));
        MBS_CUDA(c, cudaMemcpy(c->tw64_dev[ax], tw.data(), sizeof(double) * tw.size(), cudaMemcpyHostToDevice));
    }
    for (int i = 0; i < 2; ++i)
        if (!c->f64buf[i]) MBS_CUDA(c, cudaMalloc(&c->f64buf[i], 2 * sizeof(double) * (size_t)g.voxels));
    return MBS_OK;
}

static int recenter(mbs_ctx* c, const cf* y, cf* x, bool add_delta) {
    const size_t bytes = sizeof(cf) * (size_t)c->g.voxels;
    const double vb = 8.0 * (double)c->g.voxels;
    if (c->bdiag64) {
        // mixed-precision refinement: the residual of the frozen part in complex128 (refine_f64.cu)
        if (add_delta) {                                      // x_ref <- x_ref + delta
            PointwiseParams p = pw_defaults(c, false);
            p.in = x; p.w = c->delta; p.s1 = 1.f; p.s2 = 1.f; p.out = x;
            KernelScope ks(c, "recenter_add", 3 * vb);
            MBS_CUDA(c, launch_pointwise(c->g, p, c->num_sms, c->stream));
        }
        MBS_TRY(ensure_f64_tables(c));
        RefineF64 r{};
        r.bdiag = c->bdiag64; r.Kh = c->Kh64_dev;
        for (int ax = 0; ax < 3; ++ax) r.tw[ax] = c->tw64_dev[ax];
        r.buf[0] = c->f64buf[0]; r.buf[1] = c->f64buf[1];
        r.c_re = c->c.real(); r.c_im = c->c.imag(); r.k02_re = c->k02.real(); r.k02_im = c->k02.imag(); r.h = c->h;
        r.first_axis = c->first;
        {
            KernelScope ks(c, "recenter_rref_f64", 3 * vb);
            c->launches += 2 * c->ndim + 4;                   // (the scope counted one of the 2 ndim + 5 launches)
            MBS_CUDA(c, launch_rref_f64(c->g, r, x, y, c->dref, c->stream));
        }
        MBS_CUDA(c, cudaMemsetAsync(c->delta, 0, bytes, c->stream));
        c->n_recenter++;
        return MBS_OK;
    }
    if (add_delta) {                                          // x_ref <- x_ref + delta
        PointwiseParams p = pw_defaults(c, false);
        p.in = x; p.w = c->delta; p.s1 = 1.f; p.s2 = 1.f; p.out = x;
        KernelScope ks(c, "recenter_add", 3 * vb);
        MBS_CUDA(c, launch_pointwise(c->g, p, c->num_sms, c->stream));
    }
    // u = (L+I)^-1 (B x_ref + y_vec)
    MBS_TRY(run_B(c, x, nullptr, y, to_cf(-c->c), c->u, 1.f, nullptr, 0.f, RED_NONE, false));
    MBS_TRY(run_propagator(c, c->u, 1, false));
    {                                                         // d_ref = x_ref - u
        PointwiseParams p = pw_defaults(c, false);
        p.in = x; p.in2 = c->u; p.out = c->dref;
        KernelScope ks(c, "recenter_dref", 3 * vb);
        MBS_CUDA(c, launch_pointwise(c->g, p, c->num_sms, c->stream));
    }
    {                                                         // ||x_ref||^2 -> DevState.xnorm2 (size of the rounding floor)
        PointwiseParams p = pw_defaults(c, false);
        p.in = x; p.reduce = RED_XNORM;
        KernelScope ks(c, "recenter_norm", vb);
        MBS_CUDA(c, launch_pointwise(c->g, p, c->num_sms, c->stream));
    }
    MBS_CUDA(c, cudaMemsetAsync(c->delta, 0, bytes, c->stream));
    c->n_recenter++;
    return MBS_OK;
}

// Reset the device state for a new solve and (nu <= 0) compute nu = || B (L+I)^-1 y_vec ||
static int begin_solve(mbs_ctx* c, const cf* y, const cf* x, double tol, int32_t max_iter, double nu) {
    c->act_all = false;
    if (c->activation && (!activation_effective(c) || c->batch_n > 1))
        return fail(c, MBS_ERR_INVALID_ARG, "subdomain activation needs the default kernel options (fused warp-line sweeps) and a single source");
    DevState init{};
    init.iter = 0; init.done = 0; init.max_iter = max_iter; init.ticket = 0; init.tol = tol;
    init.nu2 = nu > 0 ? nu * nu : 0.0; init.last_sum = 0;
    init.n_active = c->n_sub; init.n_sub = c->n_sub; init.xnorm2 = 0.0;
    c->state_pinned[0] = init;
    MBS_CUDA(c, cudaMemcpyAsync(c->state, &c->state_pinned[0], sizeof(DevState), cudaMemcpyHostToDevice, c->stream));
    const long long rows = c->g.voxels / c->g.N[2];
    {
        KernelScope ks(c, "source_row_mask", 8.0 * (double)c->g.voxels * c->batch_n);
        MBS_CUDA(c, launch_row_mask(y, c->batch_n > 1 ? c->batch_mask : c->ymask, rows * c->batch_n, c->g.N[2], c->stream));
    }
    if (!(nu > 0)) {
        // nu^2 = sum over the sources of ||B (L+I)^-1 y_vec,b||^2 (one source: the plain normalisation of P:130)
        double nu2_sum = 0.0;
        for (int b = 0; b < c->batch_n; ++b) {
            const cf* yb = y + (size_t)b * (size_t)c->g.voxels;
            { KernelScope ks(c, "scale_copy", 16.0 * (double)c->g.voxels); MBS_CUDA(c, launch_scale_copy(yb, c->u, to_cf(-c->c), c->g.voxels, c->stream)); }
            MBS_TRY(run_propagator(c, c->u, 1, false));
            MBS_TRY(run_B(c, c->u, nullptr, nullptr, make_float2(0.f, 0.f), nullptr, 1.f, nullptr, 0.f, RED_NU2, false));
            if (c->batch_n > 1) {
                DevState st{};
                MBS_CUDA(c, cudaMemcpyAsync(&st, c->state, sizeof(DevState), cudaMemcpyDeviceToHost, c->stream));
                MBS_CUDA(c, cudaStreamSynchronize(c->stream));
                nu2_sum += st.nu2;
            }
        }
        if (c->batch_n > 1)
            MBS_CUDA(c, cudaMemcpy(&c->state->nu2, &nu2_sum, sizeof(double), cudaMemcpyHostToDevice));   // (the stream is idle here)
    }
    if (c->activation) {
        // an inactive subdomain contributes d = 0: the compact d buffers must not hold values of an earlier solve
        for (int ax = 0; ax < 3; ++ax)
            if (c->ds.buf[ax]) MBS_CUDA(c, cudaMemsetAsync(c->ds.buf[ax], 0, sizeof(cf) * corr_elems(c->g, ax), c->stream));
        const double thr = c->act_threshold >= 0 ? c->act_threshold : (tol > 0 ? 0.1 * tol : 0.0);
        c->act.thr2 = thr * thr;
        KernelScope ks(c, "activation_init", 16.0 * (double)c->g.voxels);
        MBS_CUDA(c, launch_activation_init(c->g, c->act, y, x, c->state, c->stream));
    }
    c->split = false;
    if (split_effective(c)) {
        const size_t bytes = sizeof(cf) * (size_t)c->g.voxels;
        if (!c->delta) { invalidate_graph(c); MBS_CUDA(c, cudaMalloc(&c->delta, bytes)); }
        if (!c->dref) MBS_CUDA(c, cudaMalloc(&c->dref, bytes));
        c->n_recenter = 0;
        MBS_TRY(recenter(c, y, const_cast<cf*>(x), false));   // x_ref = x^(0), delta = 0
        c->split = true;
        c->split_eps = 1.0;
    }
    MBS_CUDA(c, cudaStreamSynchronize(c->stream));   // state_pinned[0] is reused by the poll loop
    {
        // rows of y the first sweep has to read (byte ledger of the sparse-source row of SURVEY 8(d))
        const size_t rows = (size_t)(c->g.voxels / c->g.N[2]) * (size_t)c->batch_n;
        std::vector<unsigned char> m(rows);
        MBS_CUDA(c, cudaMemcpy(m.data(), c->batch_n > 1 ? c->batch_mask : c->ymask, rows, cudaMemcpyDeviceToHost));
        size_t nz = 0;
        for (size_t i = 0; i < rows; ++i) nz += m[i] ? 1 : 0;
        c->y_row_fraction = rows ? (double)nz / (double)rows : 1.0;
    }
    if (!(nu > 0)) {
        // the relative residual of P:130 divides by ||Gamma^-1 y_vec||: a zero (or non-finite) source has none
        DevState st{};
        MBS_CUDA(c, cudaMemcpy(&st, c->state, sizeof(DevState), cudaMemcpyDeviceToHost));
        if (!(st.nu2 > 0) || !std::isfinite(st.nu2))
            return fail(c, st.nu2 == 0 ? MBS_ERR_INVALID_ARG : MBS_ERR_NUMERIC,
                        st.nu2 == 0 ? "the source y is identically zero: ||Gamma^-1 y|| = 0 and the relative residual is undefined"
                                    : "non-finite ||Gamma^-1 y||: the source or the medium holds NaN/Inf");
    }
    return MBS_OK;
}

// iteration at which each subdomain was activated (all 0 when activation is off), for mbs_get_activation
static int fetch_activation(mbs_ctx* c) {
    c->act_iter_host.assign((size_t)c->n_sub, 0);
    if (c->activation)
        MBS_CUDA(c, cudaMemcpy(c->act_iter_host.data(), c->act.act_iter, sizeof(int32_t) * (size_t)c->n_sub, cudaMemcpyDeviceToHost));
    return MBS_OK;
}

static int ensure_history(mbs_ctx* c, int32_t max_iter) {
    if (c->hist_cap < max_iter) {
        invalidate_graph(c);
        if (c->hist_dev) cudaFree(c->hist_dev);
        c->hist_dev = nullptr;
        c->hist_cap = 0;
        MBS_CUDA(c, cudaMalloc(&c->hist_dev, sizeof(double) * (size_t)max_iter));
        c->hist_cap = max_iter;
    }
    return MBS_OK;
}

// Enqueue `batch` iterations: as individual launches, or (graphs on, not profiling) as one replay of a CUDA graph
// captured from the same launches.  The graph is rebuilt when the arrays, the batch or the kernel options change.
static bool graphs_enabled(const mbs_ctx* c) {
    return !c->profile && c->batch_n == 1 && (c->use_graph == 1 || (c->use_graph < 0 && c->g.voxels <= (1LL << 25)));
}

static int enqueue_batch(mbs_ctx* c, const cf* y, cf* x, int batch, bool allow_graph) {
    const bool graph_on = allow_graph && graphs_enabled(c);
    if (!graph_on) {
        for (int i = 0; i < batch; ++i) MBS_TRY(run_iteration(c, y, x));
        return MBS_OK;
    }
    const bool stale = !c->graph_exec || c->graph_y != y || c->graph_x != x || c->graph_batch != batch || c->graph_split != (int)c->split ||
                       c->graph_fused != c->fused || c->graph_tma != c->use_tma || c->graph_line != c->use_line;
    if (stale) {
        if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
        if (!c->cap_stream) MBS_CUDA(c, cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
        MBS_CUDA(c, cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
        int rc = MBS_OK;
        const int64_t launches0 = c->launches;
        cudaStream_t user_stream = c->stream;
        c->stream = c->cap_stream;                    // every launch site enqueues on c->stream
        for (int i = 0; i < batch && rc == MBS_OK; ++i) rc = run_iteration(c, y, x);
        c->stream = user_stream;
        const int64_t captured = c->launches - launches0;
        c->launches = launches0;                      // counted per replay below
        cudaGraph_t graph = nullptr;
        const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
        if (rc != MBS_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (e != cudaSuccess) return fail(c, MBS_ERR_CUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(e));
        const cudaError_t e2 = cudaGraphInstantiate(&c->graph_exec, graph, 0);
        cudaGraphDestroy(graph);
        if (e2 != cudaSuccess) { c->graph_exec = nullptr; return fail(c, MBS_ERR_CUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e2)); }
        c->graph_y = y; c->graph_x = x; c->graph_batch = batch; c->graph_split = (int)c->split;
        c->graph_fused = c->fused; c->graph_tma = c->use_tma; c->graph_line = c->use_line;
        c->launches_per_batch = captured;
    }
    MBS_CUDA(c, cudaGraphLaunch(c->graph_exec, c->stream));
    c->launches += c->launches_per_batch;
    return MBS_OK;
}

// iterations enqueued between two looks at the device stop flag (and per CUDA-graph replay)
static int poll_interval(const mbs_ctx* c) {
    if (c->check_interval > 0) return c->check_interval;
    return (int)std::max<long long>(1, std::min<long long>(64, (64LL << 20) / std::max<long long>(1, c->g.voxels)));
}

// The iteration loop behind mbs_solve, mbs_solve_host (stop test on: tol >= 0) and mbs_iterate (no stop test: tol < 0,
// `nu` > 0 reuses a known normalisation).
static int solve_device(mbs_ctx* c, const cf* y, cf* x, double tol, int32_t max_iter, double nu, double* residual_history,
                        int32_t* n_iter) {
    if (!c->potential_set) return fail(c, MBS_ERR_STATE, "mbs_set_potential has not been called");
    if (!y || !x) return fail(c, MBS_ERR_INVALID_ARG, "NULL array argument");
    if (max_iter < 1) return fail(c, MBS_ERR_INVALID_ARG, "max_iter must be >= 1");
    if (n_iter) *n_iter = 0;
    MBS_TRY(ensure_history(c, max_iter));
    MBS_TRY(begin_solve(c, y, x, tol, max_iter, nu));

    const int interval = poll_interval(c);
    MBS_CUDA(c, cudaEventRecord(c->ev_t0, c->stream));
    int enqueued = 0;
    int slot = 0;
    bool pending[2] = {false, false};
    int final_done = 0;
    while (true) {
        // enqueue one batch, then look at the poll of the PREVIOUS batch (one batch of lookahead keeps the GPU busy)
        // the first batch is enqueued launch by launch (it also warms the per-kernel attribute caches); later batches
        // replay a graph of a full interval: kernels past max_iter return at once on the device flag
        const bool first = (enqueued == 0);
        const int batch = (first || !graphs_enabled(c)) ? std::min(interval, max_iter - enqueued)
                                                        : (enqueued < max_iter ? interval : 0);
        if (batch > 0 && !final_done) {
            MBS_TRY(enqueue_batch(c, y, x, batch, !first));
            enqueued += batch;
            MBS_CUDA(c, cudaMemcpyAsync(&c->state_pinned[slot], c->state, sizeof(DevState), cudaMemcpyDeviceToHost, c->stream));
            MBS_CUDA(c, cudaEventRecord(c->ev_poll[slot], c->stream));
            pending[slot] = true;
        }
        const int prev = slot ^ 1;
        if (pending[prev]) {
            MBS_CUDA(c, cudaEventSynchronize(c->ev_poll[prev]));
            pending[prev] = false;
            const DevState& st = c->state_pinned[prev];
            if (st.done) { final_done = st.done; break; }
            if (c->activation && !c->act_all && st.n_active == st.n_sub) {
                // every subdomain is awake: the rest of the solve runs the plain kernels (no flags, no activation step)
                c->act_all = true;
                invalidate_graph(c);
            }
            if (c->split && st.iter > 0 && st.nu2 > 0 && c->n_recenter < 64) {
                // split iterate: re-centre as the residual falls (what is enqueued here runs after the batch already in
                // flight; in exact arithmetic it changes nothing).  With the double-precision residual (bdiag64) every
                // re-centring removes the complex64 rounding accumulated in delta: once per factor 2 of the residual.  The
                // complex64 fallback draws a fresh fp32 rounding of (L+I)^-1 (B x_ref + y_vec) each time, a one-off
                // perturbation of the size of the plain floor, about 2.4e-7 ||x|| / nu: once per decade and
                // only while eps is 30 x above that floor.
                const double eps = sqrt(st.last_sum / st.nu2);
                bool go;
                if (c->bdiag64) {
                    go = eps < 0.5 * c->split_eps;
                } else {
                    const double floor_plain = 2.4e-7 * sqrt(st.xnorm2 / st.nu2);
                    go = eps < 0.1 * c->split_eps && eps > 30.0 * floor_plain;
                }
                if (go) {
                    MBS_TRY(recenter(c, y, x, true));
                    c->split_eps = eps;
                }
            }
        }
        if (batch <= 0 || enqueued >= max_iter) {
            // nothing more to enqueue: drain the last poll
            if (pending[slot]) {
                MBS_CUDA(c, cudaEventSynchronize(c->ev_poll[slot]));
                pending[slot] = false;
                final_done = c->state_pinned[slot].done;
            }
            break;
        }
        slot ^= 1;
    }
    if (c->split) {
        // x = x_ref + delta (kernels that were enqueued past the stop returned at once and left delta alone)
        PointwiseParams p = pw_defaults(c, false);
        p.in = x; p.w = c->delta; p.s1 = 1.f; p.s2 = 1.f; p.out = x;
        KernelScope ks(c, "recenter_add", 24.0 * (double)c->g.voxels);
        MBS_CUDA(c, launch_pointwise(c->g, p, c->num_sms, c->stream));
        c->split = false;
    }
    MBS_CUDA(c, cudaEventRecord(c->ev_t1, c->stream));
    MBS_CUDA(c, cudaStreamSynchronize(c->stream));
    DevState fin{};
    MBS_CUDA(c, cudaMemcpy(&fin, c->state, sizeof(DevState), cudaMemcpyDeviceToHost));
    float ms = 0.f;
    MBS_CUDA(c, cudaEventElapsedTime(&ms, c->ev_t0, c->ev_t1));
    c->last_solve_ms = ms;
    prof_drain(c);
    c->norm_rhs = sqrt(fin.nu2);
    MBS_TRY(fetch_activation(c));
    if (n_iter) *n_iter = fin.iter;
    if (residual_history && fin.iter > 0)
        MBS_CUDA(c, cudaMemcpy(residual_history, c->hist_dev, sizeof(double) * (size_t)fin.iter, cudaMemcpyDeviceToHost));
    if (fin.done == 1) return MBS_OK;
    if (fin.done == 3) return fail(c, MBS_ERR_NUMERIC, "non-finite residual at iteration %d", fin.iter - 1);
    if (tol < 0) return MBS_OK;                       // mbs_iterate: exactly max_iter updates were asked for
    return fail(c, MBS_ERR_NOT_CONVERGED, "residual did not reach tol = %g within %d iterations", tol, max_iter);
}

extern "C" int mbs_solve(mbs_ctx* c, const void* y_device, void* x_device, double tol, int32_t max_iter,
                         double* residual_history, int32_t* n_iter) {
    if (!c) return MBS_ERR_INVALID_ARG;
    if (!(tol >= 0)) return fail(c, MBS_ERR_INVALID_ARG, "tol must be >= 0");
    return solve_device(c, (const cf*)y_device, (cf*)x_device, tol, max_iter, 0.0, residual_history, n_iter);
}

extern "C" int mbs_solve_batch(mbs_ctx* c, int32_t n_batch, const void* y_device, void* x_device, double tol, int32_t max_iter,
                               double* residual_history, int32_t* n_iter) {
    if (!c) return MBS_ERR_INVALID_ARG;
    if (n_batch < 1 || n_batch > 64) return fail(c, MBS_ERR_INVALID_ARG, "n_batch must be in [1, 64] (got %d)", n_batch);
    if (!(tol >= 0) && !(tol == -1.0)) return fail(c, MBS_ERR_INVALID_ARG, "tol must be >= 0 (or -1: exactly max_iter updates, no stop test)");
    if (n_batch == 1) return solve_device(c, (const cf*)y_device, (cf*)x_device, tol, max_iter, 0.0, residual_history, n_iter);
    if (!batch_available(c))
        return fail(c, MBS_ERR_UNSUPPORTED_SIZE, "batched solves need a 2-D or 3-D grid whose contiguous subdomain length has a warp-line sweep "
                                                 "(up to 512 voxels), t in {2, 4, 8, 16} and the default kernel options");
    if (c->activation) return fail(c, MBS_ERR_INVALID_ARG, "subdomain activation and batched solves are exclusive");
    MBS_TRY(ensure_batch(c, n_batch));
    c->batch_n = n_batch;
    const int rc = solve_device(c, (const cf*)y_device, (cf*)x_device, tol, max_iter, 0.0, residual_history, n_iter);
    c->batch_n = 1;
    return rc;
}

extern "C" int mbs_iterate(mbs_ctx* c, const void* y_device, void* x_device, int32_t n_iter, double nu,
                           double* residual_history) {
    if (!c) return MBS_ERR_INVALID_ARG;
    if (n_iter < 1) return fail(c, MBS_ERR_INVALID_ARG, "n_iter must be >= 1");
    return solve_device(c, (const cf*)y_device, (cf*)x_device, -1.0, n_iter, nu, residual_history, nullptr);
}

extern "C" int mbs_get_kernel_stats(mbs_ctx* c, mbs_kernel_stat* out, int32_t capacity, int32_t* count) {
    if (!c || !count) return MBS_ERR_INVALID_ARG;
    MBS_CUDA(c, cudaStreamSynchronize(c->stream));
    prof_drain(c);
    const int n = (int)c->prof.classes.size();
    *count = n;
    for (int i = 0; i < n && i < capacity && out; ++i) {
        const KernelClass& k = c->prof.classes[i];
        memset(&out[i], 0, sizeof out[i]);
        snprintf(out[i].name, sizeof out[i].name, "%s", k.name.c_str());
        out[i].launches = k.launches;
        out[i].total_ms = k.ms;
        out[i].algorithmic_bytes = k.bytes;
    }
    return MBS_OK;
}

extern "C" int mbs_reset_kernel_stats(mbs_ctx* c) {
    if (!c) return MBS_ERR_INVALID_ARG;
    MBS_CUDA(c, cudaStreamSynchronize(c->stream));
    prof_drain(c);
    c->prof.classes.clear();
    return MBS_OK;
}

extern "C" int mbs_solve_host(mbs_ctx* c, const void* y_host, void* x_host, double tol, int32_t max_iter,
                              double* residual_history, int32_t* n_iter) {
    if (!c) return MBS_ERR_INVALID_ARG;
    if (!y_host || !x_host) return fail(c, MBS_ERR_INVALID_ARG, "NULL array argument");
    const size_t bytes = sizeof(cf) * (size_t)c->g.voxels;
    if (!c->host_y) MBS_CUDA(c, cudaMalloc(&c->host_y, bytes));
    if (!c->host_x) MBS_CUDA(c, cudaMalloc(&c->host_x, bytes));
    MBS_CUDA(c, cudaMemcpyAsync(c->host_y, y_host, bytes, cudaMemcpyHostToDevice, c->stream));
    MBS_CUDA(c, cudaMemcpyAsync(c->host_x, x_host, bytes, cudaMemcpyHostToDevice, c->stream));
    if (!(tol >= 0)) return fail(c, MBS_ERR_INVALID_ARG, "tol must be >= 0");
    const int rc = solve_device(c, c->host_y, c->host_x, tol, max_iter, 0.0, residual_history, n_iter);
    if (rc != MBS_OK && rc != MBS_ERR_NOT_CONVERGED) return rc;
    const std::string keep = c->err;
    MBS_CUDA(c, cudaMemcpyAsync(x_host, c->host_x, bytes, cudaMemcpyDeviceToHost, c->stream));
    MBS_CUDA(c, cudaStreamSynchronize(c->stream));
    c->err = keep;
    return rc;
}

extern "C" int mbs_get_info(const mbs_ctx* c, mbs_info* out) {
    if (!c || !out) return MBS_ERR_INVALID_ARG;
    memset(out, 0, sizeof *out);
    out->c_re = c->c.real(); out->c_im = c->c.imag();
    out->k02_re = c->k02.real(); out->k02_im = c->k02.imag();
    out->v_max = c->v_max; out->norm_A12 = c->norm_A12; out->sum_a = c->sum_a; out->ndim = c->ndim;
    out->voxels = c->g.voxels;
    for (int d = 0; d < c->ndim; ++d) out->subdomain_shape[d] = c->g.M[c->first + d];
    out->alpha = c->alpha; out->norm_rhs = c->norm_rhs;
    const double per_voxel = c->ndim == 3 ? 112.0 : (c->ndim == 2 ? 80.0 : 32.0);
    out->algorithmic_bytes_per_iteration = per_voxel * (double)c->g.voxels;
    // the same ledger when the all-zero rows of the source are not read ("source stored sparsely": 104 B)
    out->sparse_source_bytes_per_iteration = (per_voxel - 8.0 * (1.0 - c->y_row_fraction)) * (double)c->g.voxels;
    out->workspace_bytes = c->ws_bytes;
    out->kernel_launches = c->launches;
    out->last_solve_ms = c->last_solve_ms;
    return MBS_OK;
}

// ---------------------------------------------------------------------------------------------
// mbs_apply_B_static: the scattering operator B = I - V (Eq. (8)) for callers that may not allocate
// (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  The edge-slab kernels need scratch:
// the compact correction buffers corr_d(in) that the pointwise pass then subtracts.  mbs_apply_operator keeps them in
// the context's workspace; this variant keeps them in a file-scope device array of MBS_STATIC_SCRATCH_BYTES, which
// every GPU that loads the library holds until the process exits.  Same kernels, same launch geometry, same results.
//  - no cudaMalloc / cudaFree / allocating library call on this path (and no event creation: launches are not profiled);
//  - the array is shared by every call and every context on the device and keeps the last call's contents: the slab
//    kernels overwrite every slot they later read, and the range in use is cleared first all the same; two calls that
//    overlap on the GPU (different streams, no ordering between them) race on it;
//  - in host code `g_static_scratch` is only the host-side stand-in of the symbol: its device address is looked up once
//    per device with cudaGetSymbolAddress, with that device current, and that pointer is what the kernels get.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_static_scratch[MBS_STATIC_SCRATCH_BYTES];

static int static_scratch_address(mbs_ctx* c, unsigned char** out) {
    constexpr int MAX_DEV = 64;
    static unsigned char* addr[MAX_DEV] = {nullptr};
    static std::mutex mu;
    int dev = 0;
    MBS_CUDA(c, cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEV) return fail(c, MBS_ERR_INVALID_ARG, "device ordinal %d out of range", dev);
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void* p = nullptr;
        MBS_CUDA(c, cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p || ((uintptr_t)p & 255) != 0) return fail(c, MBS_ERR_CUDA, "cudaGetSymbolAddress returned an unusable address");
        addr[dev] = (unsigned char*)p;
    }
    *out = addr[dev];
    return MBS_OK;
}

extern "C" int mbs_apply_B_static(mbs_ctx* c, const void* in_device, void* out_device) {
    if (!c) return MBS_ERR_INVALID_ARG;
    if (!c->potential_set) return fail(c, MBS_ERR_STATE, "mbs_set_potential has not been called");
    if (!in_device || !out_device) return fail(c, MBS_ERR_INVALID_ARG, "NULL array argument");
    const GridDesc& g = c->g;
    size_t off[3] = {0, 0, 0}, need = 0;
    for (int ax = 0; ax < 3; ++ax) {
        off[ax] = need;
        need += align_up(sizeof(cf) * corr_elems(g, ax));
    }
    if (need > (size_t)MBS_STATIC_SCRATCH_BYTES)
        return fail(c, MBS_ERR_INVALID_ARG,
                    "mbs_apply_B_static: the edge corrections of this grid need %zu bytes of scratch, the static array holds %zu "
                    "(MBS_STATIC_SCRATCH_BYTES); use mbs_apply_operator", need, (size_t)MBS_STATIC_SCRATCH_BYTES);
    unsigned char* base = nullptr;
    MBS_TRY(static_scratch_address(c, &base));
    if (need) MBS_CUDA(c, cudaMemsetAsync(base, 0, need, c->stream));
    CorrBufs cb{};
    for (int ax = 0; ax < 3; ++ax) cb.buf[ax] = corr_elems(g, ax) ? reinterpret_cast<cf*>(base + off[ax]) : nullptr;
    for (int ax = 0; ax < 3; ++ax) {
        if (!cb.buf[ax]) continue;
        SlabParams sp{};
        sp.in = (const cf*)in_device; sp.in2 = nullptr; sp.out = cb.buf[ax]; sp.Kh = c->Kh_dev; sp.c = to_cf(c->c); sp.axis = ax;
        sp.compact_in = 0; sp.state = c->state; sp.check_done = 0;
        c->launches++;
        MBS_CUDA(c, launch_slab(g, sp, c->stream));
    }
    PointwiseParams p = pw_defaults(c, false);
    p.in = (const cf*)in_device; p.bdiag = c->bdiag; p.out = (cf*)out_device; p.corr = cb; p.reduce = RED_NONE;
    c->launches++;
    MBS_CUDA(c, launch_pointwise(g, p, c->num_sms, c->stream));
    return MBS_OK;
}
