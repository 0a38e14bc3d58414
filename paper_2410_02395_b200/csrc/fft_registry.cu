// fft_registry.cu -- table of the FFT sizes built into the library.
#include "fft_plans.h"
#include "mbs_internal.h"

namespace mbs {
#define MBS_DECL_ENTRY(Mv) extern const FftEntry g_fft_entry_##Mv;
MBS_FOR_EACH_FFT_SIZE(MBS_DECL_ENTRY)

const FftEntry* fft_lookup(int M) {
#define MBS_CASE_ENTRY(Mv) if (M == Mv) return &g_fft_entry_##Mv;
    MBS_FOR_EACH_FFT_SIZE(MBS_CASE_ENTRY)
    return nullptr;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

cudaError_t make_strided_tensor_map(CUtensorMap* out, const cf* data, const StridedGeom& g, int M, int C) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return cudaErrorNotSupported;
    int nbox = 1;
    while (M % nbox != 0 || M / nbox > 256) ++nbox;   // as tma_nbox_of (fft_tma.cuh)
    const cuuint64_t dims[3] = {2ull * (cuuint64_t)g.inner, (cuuint64_t)g.n_seg * (cuuint64_t)M, (cuuint64_t)g.n_outer};
    const cuuint64_t strides[2] = {(cuuint64_t)g.stride * sizeof(cf), (cuuint64_t)g.outer_stride * sizeof(cf)};
    const cuuint32_t box[3] = {2u * (cuuint32_t)C, (cuuint32_t)(M / nbox), 1u};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<cf*>(data), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}
}  // namespace mbs
