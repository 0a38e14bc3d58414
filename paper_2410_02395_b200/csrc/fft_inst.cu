// fft_inst.cu -- instantiates the FFT tile kernels for ONE subdomain length; compiled once per
// size with -DMBS_FFT_SIZE=<M> (build.py) so the sizes build in parallel.
#include "fft_plans.h"
#include "mbs_internal.h"

#ifndef MBS_FFT_SIZE
#error "compile with -DMBS_FFT_SIZE=<M>"
#endif

namespace mbs {
namespace {

using PL = FftPlan<MBS_FFT_SIZE>::type;
constexpr int C = FftPlan<MBS_FFT_SIZE>::C;
constexpr int NT = PL::T * C;

template <int MODE>
__global__ void __launch_bounds__(NT) k_fft_strided(cf* __restrict__ data, const StridedGeom g, const SymbolParams sp,
                                                    const cf* __restrict__ tw, const int* __restrict__ done) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (done && *done) return;
    fft_strided_body<PL, C, MODE>(data, g, sp, tw, threadIdx.x, blockIdx.x, gridDim.x, reinterpret_cast<cf*>(smem_raw));
}

template <int MODE>
__global__ void __launch_bounds__(NT) k_fft_contig(const cf* src, cf* dst, const ContigGeom g,
                                                   const SymbolParams sp, const cf* __restrict__ tw,
                                                   const int* __restrict__ done) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (done && *done) return;
    fft_contig_body<PL, C, MODE>(src, dst, g, sp, tw, threadIdx.x, blockIdx.x, gridDim.x, reinterpret_cast<cf*>(smem_raw));
}

template <class K>
cudaError_t prepare(K kernel, size_t smem, int* blocks_per_sm) {
    static thread_local const void* done_for[16];
    static thread_local int bps_for[16];
    static thread_local int n_done = 0;
    for (int i = 0; i < n_done; ++i)
        if (done_for[i] == (const void*)kernel) { *blocks_per_sm = bps_for[i]; return cudaSuccess; }
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int bps = 1;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kernel, NT, smem);
    if (e != cudaSuccess) return e;
    if (bps < 1) bps = 1;
    if (n_done < 16) { done_for[n_done] = (const void*)kernel; bps_for[n_done] = bps; ++n_done; }
    *blocks_per_sm = bps;
    return cudaSuccess;
}

template <int MODE>
cudaError_t run_strided(cf* data, const StridedGeom& g, const SymbolParams& sp, const cf* tw, const int* done,
                        int num_sms, cudaStream_t st) {
    const size_t smem = sizeof(cf) * strided_smem_elems<PL, C>();
    int bps = 1;
    cudaError_t e = prepare(k_fft_strided<MODE>, smem, &bps);
    if (e != cudaSuccess) return e;
    long long nb = (long long)num_sms * bps;
    if (nb > g.n_tiles) nb = g.n_tiles;
    if (nb < 1) return cudaSuccess;
    k_fft_strided<MODE><<<(unsigned)nb, NT, smem, st>>>(data, g, sp, tw, done);
    return cudaGetLastError();
}

template <int MODE>
cudaError_t run_contig(const cf* src, cf* dst, const ContigGeom& g, const SymbolParams& sp, const cf* tw,
                       const int* done, int num_sms, cudaStream_t st) {
    const size_t smem = sizeof(cf) * contig_smem_elems<PL, C>();
    int bps = 1;
    cudaError_t e = prepare(k_fft_contig<MODE>, smem, &bps);
    if (e != cudaSuccess) return e;
    long long nb = (long long)num_sms * bps;
    if (nb > g.n_tiles) nb = g.n_tiles;
    if (nb < 1) return cudaSuccess;
    k_fft_contig<MODE><<<(unsigned)nb, NT, smem, st>>>(src, dst, g, sp, tw, done);
    return cudaGetLastError();
}

cudaError_t strided_entry(cf* data, const StridedGeom& g, const SymbolParams& sp, const cf* tw, int mode,
                          const int* done, int num_sms, cudaStream_t st) {
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
extern const FftEntry MBS_CAT(g_fft_entry_, MBS_FFT_SIZE) = {MBS_FFT_SIZE, C, strided_entry, contig_entry};

}  // namespace mbs
