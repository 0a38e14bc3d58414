// fft_inst.cu -- instantiates the FFT tile kernels for ONE subdomain length; compiled once per
// size with -DMBS_FFT_SIZE=<M> (build.py) so the sizes build in parallel.
#include "fft_plans.h"
#include "mbs_internal.h"
#include "fused_kernels.cuh"
#include "fft_tma.cuh"
#include "line_kernels.cuh"
#include "line_fast.cuh"

#ifndef MBS_FFT_SIZE
#error "compile with -DMBS_FFT_SIZE=<M>"
#endif

namespace mbs {
namespace {

using PL = FftPlan<MBS_FFT_SIZE>::type;
// tile widths: CS voxels per tile row of the strided sweeps, CC lines per tile of the contiguous sweeps
#ifdef MBS_CS
constexpr int CS = MBS_CS;
#else
constexpr int CS = FftPlan<MBS_FFT_SIZE>::CS;
#endif
#ifdef MBS_CC
constexpr int CC = MBS_CC;
#else
constexpr int CC = FftPlan<MBS_FFT_SIZE>::CC;
#endif
// the kernel-multiply sweep (two FFTs per tile) may use a narrower tile than the single-FFT sweeps
#ifdef MBS_CSM
constexpr int CSM = MBS_CSM;
#else
constexpr int CSM = FftPlan<MBS_FFT_SIZE>::CSM;
#endif
template <int MODE> constexpr int cs_of() { return MODE == FFT_MID ? CSM : CS; }
template <int MODE> constexpr int nts_of() { return PL::T * cs_of<MODE>(); }
constexpr int NTC = PL::T * CC;

template <int MODE>
__global__ void __launch_bounds__(nts_of<MODE>()) k_fft_strided(cf* __restrict__ data, const StridedGeom g, const SymbolParams sp,
                                                    const cf* __restrict__ tw, const int* __restrict__ done) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (done && *done) return;
    fft_strided_body<PL, cs_of<MODE>(), MODE>(data, g, sp, tw, threadIdx.x, blockIdx.x, gridDim.x, reinterpret_cast<cf*>(smem_raw));
}

// TMA-fed variant (fft_tma.cuh): persistent CTAs, NSTAGE shared-memory stages
template <class F, class = void> struct plan_nstage { static constexpr int value = 0; };
template <class F> struct plan_nstage<F, std::void_t<decltype(F::NSTAGE)>> { static constexpr int value = F::NSTAGE; };
template <int MODE>
constexpr int tma_stages() {
    const size_t stage = (size_t)PL::M * cs_of<MODE>() * sizeof(cf);
    const size_t budget = 220 * 1024;
#ifdef MBS_NSTAGE_MID
    if (MODE == FFT_MID) return stage * MBS_NSTAGE_MID <= budget ? MBS_NSTAGE_MID : 0;
#endif
#ifdef MBS_NSTAGE
    if (MODE != FFT_MID) return stage * MBS_NSTAGE <= budget ? MBS_NSTAGE : 0;
#endif
    constexpr int fixed = plan_nstage<FftPlan<MBS_FFT_SIZE>>::value;
    if (MODE != FFT_MID && fixed >= 2 && stage * fixed <= budget) return fixed;
    return stage * 3 <= budget ? 3 : (stage * 2 <= budget ? 2 : 0);
}
template <int MODE> constexpr int nstage_of() { return tma_stages<MODE>() >= 2 ? tma_stages<MODE>() : 2; }

#ifndef MBS_MID_MINB
#define MBS_MID_MINB 1
#endif
template <int MODE>
__global__ void __launch_bounds__(nts_of<MODE>(), MODE == FFT_MID ? MBS_MID_MINB : 1) k_fft_strided_tma(const __grid_constant__ CUtensorMap tmap, const StridedGeom g,
                                                        const SymbolParams sp, const cf* __restrict__ tw,
                                                        const int* __restrict__ done) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    if (done && *done) return;
    if constexpr (tma_stages<MODE>() >= 2)
        fft_strided_tma_body<PL, cs_of<MODE>(), MODE, nstage_of<MODE>()>(&tmap, g, sp, tw, reinterpret_cast<cf*>(smem_raw));
}

template <int MODE>
__global__ void __launch_bounds__(NTC) k_fft_contig(const cf* src, cf* dst, const ContigGeom g,
                                                   const SymbolParams sp, const cf* __restrict__ tw,
                                                   const int* __restrict__ done) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (done && *done) return;
    fft_contig_body<PL, CC, MODE>(src, dst, g, sp, tw, threadIdx.x, blockIdx.x, gridDim.x, reinterpret_cast<cf*>(smem_raw));
}

// the fused tile kernels move lines as pairs of voxels (128-bit accesses): odd subdomain lengths (63, 315) run unfused
constexpr bool fused_ok() { return PL::M % 2 == 0; }
template <int MODE>
__global__ void __launch_bounds__(NTC) k_fused(const FusedParams p, const cf* __restrict__ tw, const int* __restrict__ done) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[32];
    if (done && *done) return;
    if constexpr (fused_ok()) fused_contig_body<PL, CC, MODE>(p, tw, reinterpret_cast<cf*>(smem_raw), red);
}

// warp-line variant of the first / last sweep (line_kernels.cuh): 8 warps per CTA, each warp owns whole lines
constexpr bool line_ok() { return PL::T <= 32 && 32 % PL::T == 0; }
constexpr int LINE_WARPS = 8;
// resident CTAs per SM the compiler must allow: sweep 1 keeps <= 85 registers (24 warps per SM); sweep 5 holds x and
// B_diag of a line in registers across the FFT (<= 128 registers, 16 warps per SM)
#ifndef MBS_LINE_MINB_S1
#define MBS_LINE_MINB_S1 3
#endif
// FAST: the variant with t = 8 known at compile time (line_fast.cuh), chosen on the host when the context has t = 8.
// Measured A/B on one box (profiles/r02_line_kernels.md): with two or more lines per warp (T <= 16, e.g. the 256-long lines
// of config 3) the first sweep gains 12 %; with one 512-long line per warp it loses 10 % (it no longer fits the 80 registers
// that three CTAs per SM allow), while the last sweep gains 3 % there and loses 3 % at T = 16.  So: first sweep for T <= 16,
// last sweep for T = 32.
template <int MODE> constexpr bool line_fast_avail() {
    if constexpr (line_ok())
        return line_fast_ok<PL, 8>() && !line_stage_b<PL, MODE>() && (MODE == LINE_S1 ? PL::T <= 16 : PL::T == 32);
    else
        return false;
}
template <int MODE, bool ACT = false, bool FAST = false>
__global__ void __launch_bounds__(LINE_WARPS * 32, MODE == LINE_S1 ? MBS_LINE_MINB_S1 : 2) k_line(const FusedParams p, const cf* __restrict__ tw,
                                                                         const int* __restrict__ done) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[32];
    if (done && *done) return;
    if constexpr (FAST) {
        if constexpr (line_fast_avail<MODE>()) line_body_fast<PL, LINE_WARPS, MODE, ACT, 8>(p, tw, reinterpret_cast<cf*>(smem_raw), red);
    } else {
        if constexpr (line_ok()) line_body<PL, LINE_WARPS, MODE, ACT>(p, tw, reinterpret_cast<cf*>(smem_raw), red);
    }
}

// Opt in to the dynamic shared memory a kernel needs and query its occupancy; cached per (kernel, size).
// (The attribute must be raised again when a later launch needs more than the size it was set to.)
template <class K>
cudaError_t prepare(K kernel, int nthreads, size_t smem, int* blocks_per_sm) {
    struct Entry { const void* fn; int dev; size_t smem; size_t attr; int bps; };
    static thread_local Entry cache[32];
    static thread_local int n_cached = 0;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);              // function attributes are per device
    if (e != cudaSuccess) return e;
    size_t attr = 0;
    for (int i = 0; i < n_cached; ++i) {
        if (cache[i].fn != (const void*)kernel || cache[i].dev != dev) continue;
        if (cache[i].smem == smem) { *blocks_per_sm = cache[i].bps; return cudaSuccess; }
        if (cache[i].attr > attr) attr = cache[i].attr;
    }
    if (smem > attr) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr = smem;
    }
    int bps = 1;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kernel, nthreads, smem);
    if (e != cudaSuccess) return e;
    if (bps < 1) bps = 1;
    if (n_cached < 32) cache[n_cached++] = Entry{(const void*)kernel, dev, smem, attr, bps};
    *blocks_per_sm = bps;
    return cudaSuccess;
}

template <int MODE>
cudaError_t run_strided_tma(cf* data, const StridedGeom& g, const SymbolParams& sp, const cf* tw, const int* done,
                            int num_sms, cudaStream_t st) {
    CUtensorMap map;
    cudaError_t e = make_strided_tensor_map(&map, data, g, PL::M, cs_of<MODE>());
    if (e != cudaSuccess) return e;
    const size_t smem = tma_smem_bytes<PL, cs_of<MODE>(), nstage_of<MODE>()>();
    int bps = 1;
    e = prepare(k_fft_strided_tma<MODE>, nts_of<MODE>(), smem, &bps);
    if (e != cudaSuccess) return e;
    long long nb = (long long)num_sms * bps;
    if (nb > g.n_tiles) nb = g.n_tiles;
    if (nb < 1) return cudaSuccess;
    k_fft_strided_tma<MODE><<<(unsigned)nb, nts_of<MODE>(), smem, st>>>(map, g, sp, tw, done);
    return cudaGetLastError();
}

template <int MODE>
cudaError_t run_strided(cf* data, const StridedGeom& g, const SymbolParams& sp, const cf* tw, const int* done,
                        int num_sms, cudaStream_t st) {
    const size_t smem = sizeof(cf) * strided_smem_elems<PL, cs_of<MODE>()>();
    int bps = 1;
    cudaError_t e = prepare(k_fft_strided<MODE>, nts_of<MODE>(), smem, &bps);
    if (e != cudaSuccess) return e;
    long long nb = (long long)num_sms * bps;
    if (nb > g.n_tiles) nb = g.n_tiles;
    if (nb < 1) return cudaSuccess;
    k_fft_strided<MODE><<<(unsigned)nb, nts_of<MODE>(), smem, st>>>(data, g, sp, tw, done);
    return cudaGetLastError();
}

template <int MODE>
cudaError_t run_contig(const cf* src, cf* dst, const ContigGeom& g, const SymbolParams& sp, const cf* tw,
                       const int* done, int num_sms, cudaStream_t st) {
    const size_t smem = sizeof(cf) * contig_smem_elems<PL, CC>();
    int bps = 1;
    cudaError_t e = prepare(k_fft_contig<MODE>, NTC, smem, &bps);
    if (e != cudaSuccess) return e;
    long long nb = (long long)num_sms * bps;
    if (nb > g.n_tiles) nb = g.n_tiles;
    if (nb < 1) return cudaSuccess;
    k_fft_contig<MODE><<<(unsigned)nb, NTC, smem, st>>>(src, dst, g, sp, tw, done);
    return cudaGetLastError();
}

template <int MODE>
cudaError_t fused_grid(int t, long long n_tiles, int num_sms, int* nb_out, size_t* smem_out) {
    const size_t smem = sizeof(cf) * fused_smem_elems<PL, CC>(t);
    int bps = 1;
    cudaError_t e = prepare(k_fused<MODE>, NTC, smem, &bps);
    if (e != cudaSuccess) return e;
    long long nb = (long long)num_sms * bps;
    if (nb > n_tiles) nb = n_tiles;
    if (nb > MBS_MAX_PARTIALS / 2) nb = MBS_MAX_PARTIALS / 2;
    if (nb < 1) nb = 1;
    *nb_out = (int)nb;
    *smem_out = smem;
    return cudaSuccess;
}

template <int MODE>
cudaError_t run_fused(const FusedParams& p, const cf* tw, const int* done, int num_sms, cudaStream_t st) {
    int nb = 1;
    size_t smem = 0;
    cudaError_t e = fused_grid<MODE>(p.t, p.n_tiles, num_sms, &nb, &smem);
    if (e != cudaSuccess) return e;
    k_fused<MODE><<<(unsigned)nb, NTC, smem, st>>>(p, tw, done);
    return cudaGetLastError();
}

cudaError_t fused_entry(const FusedParams& p, const cf* tw, int mode, const int* done, int num_sms, cudaStream_t st) {
    switch (mode) {
        case FUSED_S1: return run_fused<FUSED_S1>(p, tw, done, num_sms, st);
        case FUSED_S5: return run_fused<FUSED_S5>(p, tw, done, num_sms, st);
        default: return run_fused<FUSED_1D>(p, tw, done, num_sms, st);
    }
}

int fused_blocks_entry(int mode, int t, long long n_tiles, int num_sms) {
    int nb = 1;
    size_t smem = 0;
    cudaError_t e;
    switch (mode) {
        case FUSED_S1: e = fused_grid<FUSED_S1>(t, n_tiles, num_sms, &nb, &smem); break;
        case FUSED_S5: e = fused_grid<FUSED_S5>(t, n_tiles, num_sms, &nb, &smem); break;
        default: e = fused_grid<FUSED_1D>(t, n_tiles, num_sms, &nb, &smem); break;
    }
    return e == cudaSuccess ? nb : -1;
}

typedef void (*LineKernel)(const FusedParams, const cf*, const int*);
template <int MODE>
LineKernel line_kernel(bool act, bool fast) {
    if (fast) return act ? k_line<MODE, true, true> : k_line<MODE, false, true>;
    return act ? k_line<MODE, true, false> : k_line<MODE, false, false>;
}

// grid of the plain (not ACT) kernel of the variant the context's t selects; the ACT kernels are launched on the same grid
// (the number of residual partials is fixed by line_blocks())
template <int MODE>
cudaError_t line_grid(int t, int variant, long long n_lines, int num_sms, int* nb_out, size_t* smem_out, bool* fast_out) {
    if constexpr (!line_ok()) {
        return cudaErrorNotSupported;
    } else {
        const bool fast = line_fast_avail<MODE>() && t == 8 && variant == 0;
        const size_t smem = line_smem_bytes<PL, LINE_WARPS, MODE>(t);
        int bps = 1;
        cudaError_t e = prepare(line_kernel<MODE>(false, fast), LINE_WARPS * 32, smem, &bps);
        if (e != cudaSuccess) return e;
        const long long units = (n_lines + (32 / PL::T) - 1) / (32 / PL::T);
        long long nb = (long long)num_sms * bps;
        const long long need = (units + LINE_WARPS - 1) / LINE_WARPS;
        if (nb > need) nb = need;
        if (nb > MBS_MAX_PARTIALS / 2) nb = MBS_MAX_PARTIALS / 2;
        if (nb < 1) nb = 1;
        *nb_out = (int)nb;
        *smem_out = smem;
        *fast_out = fast;
        return cudaSuccess;
    }
}

template <int MODE>
cudaError_t line_launch(const FusedParams& p, const cf* tw, const int* done, int num_sms, cudaStream_t st) {
    int nb = 1, bps = 1;
    size_t smem = 0;
    bool fast = false;
    cudaError_t e = line_grid<MODE>(p.t, p.line_variant, p.n_lines, num_sms, &nb, &smem, &fast);
    if (e != cudaSuccess) return e;
    const bool ext = p.active != nullptr || p.n_batch > 1;        // activation and batches run the extended instantiations
    const LineKernel k = line_kernel<MODE>(ext, fast);
    if (ext && (e = prepare(k, LINE_WARPS * 32, smem, &bps)) != cudaSuccess) return e;
    k<<<(unsigned)nb, LINE_WARPS * 32, smem, st>>>(p, tw, done);
    return cudaGetLastError();
}

cudaError_t line_entry(const FusedParams& p, const cf* tw, int mode, const int* done, int num_sms, cudaStream_t st) {
    return mode == LINE_S1 ? line_launch<LINE_S1>(p, tw, done, num_sms, st) : line_launch<LINE_S5>(p, tw, done, num_sms, st);
}

int line_blocks_entry(int mode, int t, int variant, long long n_lines, int num_sms) {
    int nb = 1;
    size_t smem = 0;
    bool fast = false;
    cudaError_t e = (mode == LINE_S1) ? line_grid<LINE_S1>(t, variant, n_lines, num_sms, &nb, &smem, &fast)
                                      : line_grid<LINE_S5>(t, variant, n_lines, num_sms, &nb, &smem, &fast);
    return e == cudaSuccess ? nb : -1;
}

cudaError_t strided_entry(cf* data, const StridedGeom& g, const SymbolParams& sp, const cf* tw, int mode,
                          const int* done, int num_sms, int use_tma, cudaStream_t st) {
    // TMA needs 16-byte multiples for the global strides (inner even) and a 16-byte aligned base
    if (use_tma && g.inner % 2 == 0 && (reinterpret_cast<uintptr_t>(data) & 15) == 0) {
        if (mode == FFT_FWD && tma_stages<FFT_FWD>() >= 2) return run_strided_tma<FFT_FWD>(data, g, sp, tw, done, num_sms, st);
        if (mode == FFT_INV && tma_stages<FFT_INV>() >= 2) return run_strided_tma<FFT_INV>(data, g, sp, tw, done, num_sms, st);
        if (mode == FFT_MID && tma_stages<FFT_MID>() >= 2) return run_strided_tma<FFT_MID>(data, g, sp, tw, done, num_sms, st);
    }
    switch (mode) {
        case FFT_FWD: return run_strided<FFT_FWD>(data, g, sp, tw, done, num_sms, st);
        case FFT_INV: return run_strided<FFT_INV>(data, g, sp, tw, done, num_sms, st);
        default: return run_strided<FFT_MID>(data, g, sp, tw, done, num_sms, st);
    }
}

cudaError_t contig_entry(const cf* src, cf* dst, const ContigGeom& g, const SymbolParams& sp, const cf* tw, int mode,
                         const int* done, int num_sms, cudaStream_t st) {
    switch (mode) {
        case FFT_FWD: return run_contig<FFT_FWD>(src, dst, g, sp, tw, done, num_sms, st);
        case FFT_INV: return run_contig<FFT_INV>(src, dst, g, sp, tw, done, num_sms, st);
        default: return run_contig<FFT_MID>(src, dst, g, sp, tw, done, num_sms, st);
    }
}

}  // namespace

#define MBS_CAT2(a, b) a##b
#define MBS_CAT(a, b) MBS_CAT2(a, b)
extern const FftEntry MBS_CAT(g_fft_entry_, MBS_FFT_SIZE) = {
    MBS_FFT_SIZE, CS, CSM, CC, strided_entry, contig_entry, fused_ok() ? fused_entry : nullptr,
    fused_ok() ? fused_blocks_entry : nullptr,
    line_ok() ? line_entry : nullptr, line_ok() ? line_blocks_entry : nullptr};

}  // namespace mbs
