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
}  // namespace mbs
