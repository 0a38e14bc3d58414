// mbs_internal.h -- shared declarations of the library's translation units (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/mbs.h"
#include "fft_kernels.cuh"

namespace mbs {

constexpr int MBS_MAX_T = 16;           // templated slab kernels; larger t uses the generic kernel
constexpr int MBS_MAX_PARTIALS = 4096;  // per-block partial sums of a reduction

// Grid description, always 3-D internally: a D < 3 problem has leading axes of length 1.
struct GridDesc {
    int N[3];   // grid
    int M[3];   // subdomain length
    int S[3];   // subdomain count
    int a[3];   // a_d of Eq. (9): 0 none, 1 wrap only, 2 wrap + transfer
    int per[3]; // periodic flag
    int t;      // correction points
    long long voxels;
};

// Compact edge-correction buffers, one per axis (nullptr when a_d = 0).
// axis 0: [S0*2t][N1][N2]; axis 1: [N0][S1*2t][N2]; axis 2: [N0*N1][S2*2t].
// Slot q of subdomain s: s*2t + e for the first t points (e < t), s*2t + t + (e - (M - t)) for the last t.
struct CorrBufs {
    cf* buf[3];
};

// Device-resident solver state (one per context).
struct DevState {
    int iter;               // updates applied so far in this solve
    int done;               // 0 running, 1 converged, 2 max_iter reached, 3 non-finite residual
    int max_iter;
    unsigned int ticket;    // last-block election counter of the reduction
    double tol;
    double nu2;             // ||Gamma^-1 y_vec||^2
    double last_sum;        // last reduced sum (for norm queries)
};

enum ReduceMode { RED_NONE = 0, RED_NU2 = 1, RED_RESIDUAL = 2, RED_PLAIN = 3 };

// Pointwise pass:  val = B_diag*(in - in2) + ysc*y - corr;   (each term optional)
//   update == 0:   out = s1*val + s2*w
//   update == 1:   x = in (the iterate), r = val, out = x - alpha*r   (a6-a9 of the scope table)
//   reduce != 0:   accumulate |val|^2 and finish according to ReduceMode.
struct PointwiseParams {
    const cf* in;
    const cf* in2;     // optional, subtracted from in before B_diag
    const cf* bdiag;   // optional (nullptr: factor 1)
    const cf* y;       // optional
    cf ysc;
    const cf* w;       // optional
    float s1, s2;
    cf* out;
    CorrBufs corr;     // subtracted where non-null
    int update;
    float alpha;
    int reduce;
    double* partials;
    double* hist;
    DevState* state;
    int check_done;    // 1: return immediately if state->done != 0
};

struct SlabParams {
    const cf* in;
    const cf* in2;     // optional: correction of (in - in2)
    cf* out;           // compact buffer of this axis
    const float* Kh;   // t x t, K_t / h^2, row-major (row a = last-edge index, column b = first-edge index)
    cf c;              // scale factor c of Eq. (9)
    int axis;
    const DevState* state;
    int check_done;
};

// launchers implemented in kernels.cu
cudaError_t launch_pointwise(const GridDesc& g, const PointwiseParams& p, int num_sms, cudaStream_t st);
cudaError_t launch_slab(const GridDesc& g, const SlabParams& p, cudaStream_t st);
cudaError_t launch_scale_copy(const cf* in, cf* out, cf scale, long long n, cudaStream_t st);

struct SetupParams {
    const cf* n_map;
    double kw2;          // (2 pi / lambda)^2
    double beta;         // absorber strength (R3)
    int W[3];
    double k02_re, k02_im;
    double c_re, c_im;
};
// pass 0: per-block min/max of Re k^2, Im k^2 and min Im n -> out[block*5 + {0..4}]
// pass 1: per-block max |k^2 - k0^2|^2                     -> out[block]
// pass 2: B_diag = 1 - c (k^2 - k0^2)                      -> bdiag
cudaError_t launch_setup(const GridDesc& g, const SetupParams& p, int pass, double* out, cf* bdiag, int nblocks,
                         cudaStream_t st);

// FFT registry (fft_inst.cu compiled once per size, fft_registry.cu)
struct FftEntry {
    int M;
    int C;   // lines per tile
    cudaError_t (*strided)(cf* data, const StridedGeom& g, const SymbolParams& sp, const cf* tw, int mode,
                           const int* done, int num_sms, cudaStream_t st);
    cudaError_t (*contig)(const cf* src, cf* dst, const ContigGeom& g, const SymbolParams& sp, const cf* tw, int mode,
                          const int* done, int num_sms, cudaStream_t st);
};
const FftEntry* fft_lookup(int M);

}  // namespace mbs
