// mbs_internal.h -- shared declarations of the library's translation units (not installed).
#pragma once
#include <cuda.h>
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
    int n_active;           // subdomain activation: active subdomains (= all of them when it is off)
    int n_sub;
    double xnorm2;          // ||x_ref||^2 at the last re-centering of the split iterate (api.cu recenter())
};

enum ReduceMode { RED_NONE = 0, RED_NU2 = 1, RED_RESIDUAL = 2, RED_PLAIN = 3, RED_XNORM = 4 };

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
    int compact_in;    // 1: `in` is already a compact [outer][S*2t][inner] buffer (fix-up of the fused sweep)
    const DevState* state;
    int check_done;
    // batched solves (R18): n_batch sources, `in` advances by in_stride and `out` by out_stride elements per source
    // (0 / 1 source: plain call)
    int n_batch;
    long long in_stride, out_stride;
};

// fix-up of the fused last sweep on the slab rows of axes 0 and 1 (kernels.cu: k_fixup)
struct FixupParams {
    cf* x;
    const cf* u;       // r_part on the slab rows
    const cf* cx0;     // corr_0(d), corr_1(d), compact
    const cf* cx1;
    const cf* cx2;     // corr_2(d), compact [N0*N1][S2*2t] (warp-line path; else nullptr)
    int e0, e1, e2;
    float alpha;
    double* partials;
    int slot0;         // first partial slot of this launch; slots below hold the fused sweep's partials
    int reduce_mode;
    DevState* state;
    double* hist;
    int check_done;
};

// launchers implemented in kernels.cu
cudaError_t launch_pointwise(const GridDesc& g, const PointwiseParams& p, int num_sms, cudaStream_t st);
cudaError_t launch_slab(const GridDesc& g, const SlabParams& p, cudaStream_t st);
bool slab_pair_supported(int t);   // launch_slab_pair: two axes in one launch (t = 2, 4, 8, 16)
cudaError_t launch_slab_pair(const GridDesc& g, const SlabParams& pA, const SlabParams& pB, cudaStream_t st);
// slab pass of one axis (kernels.cu: k_slab_pass): corr_ax(d) from the compact d, applied to u / x in the same kernel
struct SlabPassParams {
    const cf* ds;      // compact d of this axis, [outer][S*2t][inner]
    cf* u;             // r_part minus the corrections of the earlier axes, at the slab voxels
    cf* x;
    const float* Kh;
    cf c;
    int axis;
    int e1, e2;        // axes 1 / 2 have edge corrections (later passes exist)
    float alpha;
    double* partials;
    int slot0;         // first partial slot of this launch
    int finish;        // 1: this is the last pass: add all partials [0, slot0 + grid) and finish the iteration
    DevState* state;
    double* hist;
    const int* active; // subdomain activation: flags per subdomain (s0*S1 + s1)*S2 + s2, or nullptr (all active);
                       // the edge voxels of an inactive subdomain are left alone (no update, no residual)
    int n_batch;       // batched solves: sources (0 / 1: plain); ds advances by ds_stride, u and x by vox_stride per source
    long long ds_stride, vox_stride;
};
int slab_pass_blocks(const GridDesc& g, int ax);
bool slab_pass_supported(int t);
cudaError_t launch_slab_pass(const GridDesc& g, const SlabPassParams& p, cudaStream_t st);
int fixup_blocks(const GridDesc& g, int e0, int e1, int e2, int num_sms);
cudaError_t launch_fixup(const GridDesc& g, const FixupParams& p, int nblocks, cudaStream_t st);
cudaError_t launch_row_mask(const cf* y, unsigned char* mask, long long rows, int N2, cudaStream_t st);
cudaError_t launch_scale_copy(const cf* in, cf* out, cf scale, long long n, cudaStream_t st);

struct SetupParams {
    const cf* n_map;
    double kw2;          // (2 pi / lambda)^2
    double beta;         // absorber strength (R3)
    int W[3];
    double k02_re, k02_im;
    double c_re, c_im;
    double* bdiag64;     // optional (pass 2): B_diag also as complex128 (interleaved re, im) for refine_f64.cu
};
// pass 0: per-block min/max of Re k^2, Im k^2 and min Im n -> out[block*5 + {0..4}]
// pass 1: per-block max |k^2 - k0^2|^2                     -> out[block]
// pass 2: B_diag = 1 - c (k^2 - k0^2)                      -> bdiag
cudaError_t launch_setup(const GridDesc& g, const SetupParams& p, int pass, double* out, cf* bdiag, int nblocks,
                         cudaStream_t st);

// fused first / last sweep along the contiguous axis (fused_kernels.cuh)
enum FusedMode { FUSED_S1 = 0, FUSED_S5 = 1, FUSED_1D = 2 };
enum LineMode { LINE_S1 = 0, LINE_S5 = 1 };   // warp-line variant (line_kernels.cuh)

struct FusedParams {
    cf* x;               // iterate: read by S1; read and updated in place by S5 / 1D
    const cf* bdiag;     // B_diag = 1 - c (k^2 - k0^2)
    const cf* y;         // physical source (S1 / 1D) or nullptr
    const unsigned char* ymask;   // per grid row: 0 = the row of y is all zero (skip its load); nullptr = unknown
    cf ysc;              // y_vec = ysc * y = -c y
    cf* u;               // S1: output; S5: input u' lines, output r_part on slab rows
    int N0, N1, N2;      // grid extents (N2 = S2 * M)
    int S0;              // subdomains along axis 0
    int S2, a2, per2;    // subdomains, a_d and periodic flag of the last axis
    int t;               // correction points
    int e0, e1;          // 1 if axis 0 / 1 has edge corrections
    int M0, M1, S1;
    const cf* cx0;       // S1: corr_0(x), compact [S0*2t][N1][N2]
    const cf* cx1;       // S1: corr_1(x), compact [N0][S1*2t][N2]
    cf* ds0;             // S5: d at the axis-0 slab rows, same layouts
    cf* ds1;
    cf* ds2;             // warp-line S5: d at the 2t edge points of every line, compact [N0*N1][S2*2t]
    const float* Kh;     // K_t / h^2, t x t row-major
    cf c;                // scale factor of Eq. (9)
    float alpha;
    SymbolParams sp;     // 1D: Fourier kernel
    long long n_lines;   // voxels / M
    long long n_tiles;
    // reduction
    double* partials;
    int slot0, n_total, finish, reduce_mode;
    DevState* state;
    double* hist;
    const int* active;   // subdomain activation: flags per subdomain, or nullptr; lines of an inactive
                         // subdomain are skipped by the warp-line sweeps
    // batched solves (R18), warp-line sweeps only: n_batch sources share B_diag; x, y, u advance by batch_stride
    // elements per source, the compact buffers of axis d by cstride[d], ymask by mask_stride rows
    int n_batch;
    long long batch_stride, cstride[3], mask_stride;
    int line_variant;    // warp-line sweeps: 0 = the variant with t known at compile time when there is one (t = 8), 1 = generic
    const cf* rref;      // split iterate with the complex128 residual: r_ref = B d_ref, added to r = B_diag d - corr(d) of the
                         // small part d = delta - u' (instead of d_ref being added to d); or nullptr
    const cf* dref;      // split iterate (api.cu "refinement"): the sweeps run on the small part delta of x = x_ref + delta,
                         // and the last sweep adds d_ref = x_ref - (L+I)^-1 (B x_ref + y_vec) to d = delta - u'; or nullptr
};

// Subdomain activation (reading R17 of DESIGN.md section 3).  Device-resident: flags[n_sub], the list of
// the active subdomains in index order + its length (read by the strided sweeps), the iteration at which each
// subdomain was activated, per-block partial sums of the transferred norms.
struct ActivationState {
    int* flags;          // [n_sub]
    int* list;           // [n_sub] active subdomain indices, ascending
    int* n_act;          // [1]
    int* act_iter;       // [n_sub] iteration of activation, -1 = not yet
    double* partials;    // [n_sub][6][ACT_CHUNKS]
    unsigned int* ticket;
    double thr2;         // threshold^2 (relative to nu^2)
};
constexpr int ACT_CHUNKS = 8;
// flags from the source and the start vector (a subdomain is active from the start if y or x0 is non-zero in it)
cudaError_t launch_activation_init(const GridDesc& g, const ActivationState& a, const cf* y, const cf* x, DevState* state,
                                   cudaStream_t st);
// before update n: T_s^2 = sum_d ||corr_d(x)_s||^2 for every inactive subdomain s (what its active neighbours
// transfer into it); activates s when T_s^2 >= thr2 * nu^2; rebuilds the list.  Deterministic (fixed-order sums).
cudaError_t launch_activation_step(const GridDesc& g, const ActivationState& a, const cf* x, const float* Kh, cf c,
                                   DevState* state, cudaStream_t st);


// Double-precision residual of the frozen part of the split iterate (refine_f64.cu): everything the kernels need.
struct RefineF64 {
    const double* bdiag;   // B_diag as complex128 (interleaved)
    const double* Kh;      // K_t / h^2, t x t row-major, double
    const double* tw[3];   // per axis: exp(-2 pi i j / M_d), j in [0, M_d), complex128 (interleaved); nullptr for unit axes
    double* buf[2];        // two complex128 work arrays of the grid size
    double c_re, c_im, k02_re, k02_im, h;
    int first_axis;        // first real axis of the internal 3-D description
};
// rref = B (x - (L+I)^-1 (B x + y_vec)) evaluated in complex128, rounded once to complex64 (y may be nullptr)
cudaError_t launch_rref_f64(const GridDesc& g, const RefineF64& r, const cf* x, const cf* y, cf* rref, cudaStream_t st);

// FFT registry (fft_inst.cu compiled once per size, fft_registry.cu)
struct FftEntry {
    int M;
    int CS;  // voxels per tile row of the strided forward / inverse sweeps
    int CSM; // voxels per tile row of the strided kernel-multiply sweep
    int CC;  // lines per tile of the contiguous sweeps
    cudaError_t (*strided)(cf* data, const StridedGeom& g, const SymbolParams& sp, const cf* tw, int mode,
                           const int* done, int num_sms, int use_tma, cudaStream_t st);
    cudaError_t (*contig)(const cf* src, cf* dst, const ContigGeom& g, const SymbolParams& sp, const cf* tw, int mode,
                          const int* done, int num_sms, cudaStream_t st);
    // fused sweep (FusedMode); *blocks_out = grid size used (number of residual partials written)
    cudaError_t (*fused)(const FusedParams& p, const cf* tw, int mode, const int* done, int num_sms, cudaStream_t st);
    int (*fused_blocks)(int mode, int t, long long n_tiles, int num_sms);
    // warp-line variant of the first / last sweep (line_kernels.cuh); nullptr when a line does not fit in a warp
    cudaError_t (*line)(const FusedParams& p, const cf* tw, int mode, const int* done, int num_sms, cudaStream_t st);
    int (*line_blocks)(int mode, int t, int variant, long long n_lines, int num_sms);   // variant: FusedParams::line_variant
};
const FftEntry* fft_lookup(int M);

// Tensor map of `data` viewed as [n_outer][n_seg*M][inner] for the TMA-fed strided sweep (fft_registry.cu):
// float32 dims {2*inner, n_seg*M, n_outer}, box {2*C, M / ceil(M/256), 1}.
cudaError_t make_strided_tensor_map(CUtensorMap* out, const cf* data, const StridedGeom& g, int M, int C);

}  // namespace mbs
