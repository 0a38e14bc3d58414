// kernels.cu -- pointwise, edge-slab, reduction and setup kernels of the MBS iteration (sm_100a).
//
//   pointwise : B = I - V applied as  B_diag * u - corr(u)  (Eq. (8), P:126 step 3-5), the source
//               term y_vec = -c y, the difference x - u' and the alpha-update of Eq. (6),
//               and the residual partial sums of P:130 -- one vectorised pass, options by flags.
//   slab      : edge corrections C_ss u_s and A_{s,s+-1} u_{s+-1} of P:122-128 (steps 1, 2, 4, 5), written
//               to compact per-axis buffers without materialising halos: the neighbour's edge points are
//               read in place.
//   setup     : k^2 = (2 pi n / lambda)^2 + absorber, min/max, ||k^2 - k0^2||_inf and B_diag, in double.
#include <math_constants.h>

#include "mbs_internal.h"
#include "reduce.cuh"

namespace mbs {

// ---------------------------------------------------------------------------------------------
// pointwise pass
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int edge_slot(int i, int M, int t) {
    // slot within [0, 2t) of subdomain-local index e if it is an edge point, else -1; plus s*2t
    const int s = i / M;
    const int e = i - s * M;
    if (e < t) return s * 2 * t + e;
    if (e >= M - t) return s * 2 * t + t + (e - (M - t));
    return -1;
}

template <int VEC>
__device__ __forceinline__ void corr_gather(const GridDesc& g, const CorrBufs& cb, int i0, int i1, int i2, cf* acc) {
    if (cb.buf[0]) {
        const int q = edge_slot(i0, g.M[0], g.t);
        if (q >= 0) {
            const cf* src = cb.buf[0] + ((long long)q * g.N[1] + i1) * g.N[2] + i2;
#pragma unroll
            for (int v = 0; v < VEC; ++v) acc[v] = cadd(acc[v], src[v]);
        }
    }
    if (cb.buf[1]) {
        const int q = edge_slot(i1, g.M[1], g.t);
        if (q >= 0) {
            const cf* src = cb.buf[1] + ((long long)i0 * (g.S[1] * 2 * g.t) + q) * g.N[2] + i2;
#pragma unroll
            for (int v = 0; v < VEC; ++v) acc[v] = cadd(acc[v], src[v]);
        }
    }
    if (cb.buf[2]) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            const int q = edge_slot(i2 + v, g.M[2], g.t);
            if (q >= 0) acc[v] = cadd(acc[v], cb.buf[2][((long long)i0 * g.N[1] + i1) * (g.S[2] * 2 * g.t) + q]);
        }
    }
}

template <int VEC> struct VecT;
template <> struct VecT<1> { typedef float2 type; };
template <> struct VecT<2> { typedef float4 type; };

template <int VEC>
__device__ __forceinline__ void load_vec(const cf* p, cf* v) {
    typename VecT<VEC>::type raw = *reinterpret_cast<const typename VecT<VEC>::type*>(p);
    const cf* r = reinterpret_cast<const cf*>(&raw);
#pragma unroll
    for (int i = 0; i < VEC; ++i) v[i] = r[i];
}
template <int VEC>
__device__ __forceinline__ void store_vec(cf* p, const cf* v) {
    typename VecT<VEC>::type raw;
    cf* r = reinterpret_cast<cf*>(&raw);
#pragma unroll
    for (int i = 0; i < VEC; ++i) r[i] = v[i];
    *reinterpret_cast<typename VecT<VEC>::type*>(p) = raw;
}

constexpr int PW_THREADS = 256;

template <int VEC>
__global__ void __launch_bounds__(PW_THREADS) k_pointwise(const GridDesc g, const PointwiseParams p) {
    __shared__ double red[32];
    if (p.check_done && p.state->done) return;
    const int chunk_len = PW_THREADS * VEC;
    const int nchunks = (g.N[2] + chunk_len - 1) / chunk_len;
    const long long n_work = (long long)g.N[0] * g.N[1] * nchunks;
    float acc = 0.f;
    for (long long work = blockIdx.x; work < n_work; work += gridDim.x) {
        const int chunk = (int)(work % nchunks);
        const int row = (int)(work / nchunks);
        const int i1 = row % g.N[1];
        const int i0 = row / g.N[1];
        const int i2 = chunk * chunk_len + threadIdx.x * VEC;
        if (i2 >= g.N[2]) continue;
        const long long idx = (long long)row * g.N[2] + i2;
        cf a[VEC], val[VEC];
        load_vec<VEC>(p.in + idx, a);
#pragma unroll
        for (int v = 0; v < VEC; ++v) val[v] = a[v];
        if (p.in2) {
            cf b[VEC];
            load_vec<VEC>(p.in2 + idx, b);
#pragma unroll
            for (int v = 0; v < VEC; ++v) val[v] = csub(val[v], b[v]);
        }
        if (p.bdiag) {
            cf b[VEC];
            load_vec<VEC>(p.bdiag + idx, b);
#pragma unroll
            for (int v = 0; v < VEC; ++v) val[v] = cmul(b[v], val[v]);
        }
        if (p.y) {
            cf b[VEC];
            load_vec<VEC>(p.y + idx, b);
#pragma unroll
            for (int v = 0; v < VEC; ++v) val[v] = cadd(val[v], cmul(p.ysc, b[v]));
        }
        cf corr[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) corr[v] = make_float2(0.f, 0.f);
        corr_gather<VEC>(g, p.corr, i0, i1, i2, corr);
#pragma unroll
        for (int v = 0; v < VEC; ++v) val[v] = csub(val[v], corr[v]);
        if (p.reduce) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) acc += val[v].x * val[v].x + val[v].y * val[v].y;
        }
        cf o[VEC];
        if (p.update) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) o[v] = make_float2(a[v].x - p.alpha * val[v].x, a[v].y - p.alpha * val[v].y);
        } else {
#pragma unroll
            for (int v = 0; v < VEC; ++v) o[v] = cscale(val[v], p.s1);
            if (p.w) {
                cf b[VEC];
                load_vec<VEC>(p.w + idx, b);
#pragma unroll
                for (int v = 0; v < VEC; ++v) o[v] = make_float2(o[v].x + p.s2 * b[v].x, o[v].y + p.s2 * b[v].y);
            }
        }
        if (p.out) store_vec<VEC>(p.out + idx, o);
    }
    if (p.reduce) {
        const double bs = block_sum((double)acc, red);
        grid_reduce_finish(bs, p.partials, 0, (int)gridDim.x, 1, p.reduce, p.state, p.hist, red);
    }
}

cudaError_t launch_pointwise(const GridDesc& g, const PointwiseParams& p, int num_sms, cudaStream_t st) {
    const bool vec2 = (g.N[2] % 2 == 0);
    const int vec = vec2 ? 2 : 1;
    const int chunk_len = PW_THREADS * vec;
    const long long nchunks = (g.N[2] + chunk_len - 1) / chunk_len;
    const long long n_work = (long long)g.N[0] * g.N[1] * nchunks;
    long long nb = (long long)num_sms * 8;
    if (nb > MBS_MAX_PARTIALS) nb = MBS_MAX_PARTIALS;
    if (nb > n_work) nb = n_work;
    if (nb < 1) nb = 1;
    if (vec2) k_pointwise<2><<<(unsigned)nb, PW_THREADS, 0, st>>>(g, p);
    else k_pointwise<1><<<(unsigned)nb, PW_THREADS, 0, st>>>(g, p);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// edge-slab corrections.  One thread = one (outer, subdomain, side, inner) item and the
// t outputs of that edge:
//   side 1 (last t points of s):   corr[a] = c * sum_b Kh[a][b] (u_{s+1}[b]     - u_s[b])          = -l_s + l_{s+1}
//   side 0 (first t points of s):  corr[b] = c * sum_a Kh[a][b] (u_{s-1}[M-t+a] - u_s[M-t+a])      = -rho_s + rho_{s-1}
// A missing neighbour (non-periodic exterior face) contributes 0; periodic axes wrap.
// ---------------------------------------------------------------------------------------------
constexpr int SLAB_THREADS = 128;

// the items of one axis, spread over `nblocks` blocks of which this one is number `block`
template <int TT>
__device__ __forceinline__ void slab_items(const GridDesc& g, const SlabParams& p, const long long inner, const long long n_items,
                                           const float* Ks, const unsigned block, const unsigned nblocks) {
    const int t = (TT > 0) ? TT : g.t;
    const int ax = p.axis;
    const int S = g.S[ax], M = g.M[ax];
    const long long axis_stride = inner;
    // n_items = 2 voxels / M < 2^30 (mbs_create limits the grid to 2^31 - 1 voxels): 32-bit item arithmetic, no
    // 64-bit divisions in the loop (measured: 5-10 % on this kernel)
    const unsigned inner32 = (unsigned)inner, n32 = (unsigned)n_items, S32 = (unsigned)S;
    for (unsigned item = block * SLAB_THREADS + threadIdx.x; item < n32; item += nblocks * SLAB_THREADS) {
        const unsigned rest0 = item / inner32;
        const long long in_i = (long long)(item - rest0 * inner32);
        const int side = (int)(rest0 & 1u);
        const unsigned rest1 = rest0 >> 1;
        const unsigned o32 = rest1 / S32;
        const int s = (int)(rest1 - o32 * S32);
        const long long o = (long long)o32;
        // neighbour subdomain
        int nb = side ? s + 1 : s - 1;
        bool has_nb = true;
        if (nb < 0 || nb >= S) {
            if (g.per[ax]) nb = (nb + S) % S;
            else has_nb = false;
        }
        // side 1 reads the FIRST t points of own and neighbour; side 0 reads the LAST t points
        long long own0, nb0;
        if (p.compact_in) {   // input already in the compact [outer][S*2t][inner] layout
            own0 = ((o * S + s) * 2 * t + (side ? 0 : t)) * inner + in_i;
            nb0 = ((o * S + nb) * 2 * t + (side ? 0 : t)) * inner + in_i;
        } else {
            const long long base_o = o * (long long)g.N[ax] * inner + in_i;
            const long long off = side ? 0 : (long long)(M - t);
            own0 = base_o + ((long long)s * M + off) * axis_stride;
            nb0 = base_o + ((long long)nb * M + off) * axis_stride;
        }
        cf dv[TT];
#pragma unroll
        for (int q = 0; q < TT; ++q) {
            cf own = p.in[own0 + q * axis_stride];
            if (p.in2) own = csub(own, p.in2[own0 + q * axis_stride]);
            cf nbv = make_float2(0.f, 0.f);
            if (has_nb) {
                nbv = p.in[nb0 + q * axis_stride];
                if (p.in2) nbv = csub(nbv, p.in2[nb0 + q * axis_stride]);
            }
            dv[q] = csub(nbv, own);
        }
        cf* outp = p.out + ((o * S + s) * 2 * t + (long long)side * t) * inner + in_i;
#pragma unroll
        for (int e = 0; e < TT; ++e) {
            float sr = 0.f, si = 0.f;
#pragma unroll
            for (int q = 0; q < TT; ++q) {
                const float k = side ? Ks[e * TT + q] : Ks[q * TT + e];
                sr = fmaf(k, dv[q].x, sr);
                si = fmaf(k, dv[q].y, si);
            }
            outp[(long long)e * inner] = cmul(p.c, make_float2(sr, si));
        }
    }
}

// BATCH: batched solves (R18), one source after the other; a separate instantiation so that the plain kernels keep
// their code exactly (the loop and the parameter copy cost 25-60 % on these latency-bound kernels)
template <int TT, bool BATCH = false>
__global__ void __launch_bounds__(SLAB_THREADS) k_slab(const GridDesc g, const SlabParams p, const long long outer,
                                                       const long long inner, const long long n_items) {
    __shared__ float Ks[TT * TT];
    if (p.check_done && p.state->done) return;
    for (int i = threadIdx.x; i < TT * TT; i += SLAB_THREADS) Ks[i] = p.Kh[i];
    __syncthreads();
    if constexpr (BATCH) {
        SlabParams q = p;
        for (int b = 0; b < p.n_batch; ++b) {
            slab_items<TT>(g, q, inner, n_items, Ks, blockIdx.x, gridDim.x);
            q.in += p.in_stride; q.out += p.out_stride;
        }
    } else {
        slab_items<TT>(g, p, inner, n_items, Ks, blockIdx.x, gridDim.x);
    }
}

// Two axes in one launch (the corrections of different axes are independent): blocks [0, nbA) take the items of pA, the
// rest those of pB, so the tail of one axis overlaps the other and one launch gap disappears (it matters on small grids).
template <int TT>
__global__ void __launch_bounds__(SLAB_THREADS) k_slab_pair(const GridDesc g, const SlabParams pA, const SlabParams pB,
                                                            const long long innerA, const long long nA,
                                                            const long long innerB, const long long nB, const unsigned nbA) {
    __shared__ float Ks[TT * TT];
    if (pA.check_done && pA.state->done) return;
    for (int i = threadIdx.x; i < TT * TT; i += SLAB_THREADS) Ks[i] = pA.Kh[i];
    __syncthreads();
    if (blockIdx.x < nbA) slab_items<TT>(g, pA, innerA, nA, Ks, blockIdx.x, nbA);
    else slab_items<TT>(g, pB, innerB, nB, Ks, blockIdx.x - nbA, gridDim.x - nbA);
}

// ---------------------------------------------------------------------------------------------
// slab pass (fix-up of the warp-line last sweep): for one axis, corr_ax(d) from the compact d and its
// application in the same kernel.  At each of the t edge voxels an item owns:
//     r = u - corr_ax(d)          (u holds r_part = B_diag d, minus the corrections of the earlier axes)
// and then either the voxel is also an edge point of a LATER axis (its pass will finish it): u = r; or this is
// its last correction:  |r|^2 partial sum,  x <- x - alpha r        (a7-a9).
// Passes run in axis order 0, 1, 2 on the stream; the last one finishes the reduction and the stop test.
// ---------------------------------------------------------------------------------------------
template <int TT, bool ACT, bool BATCH>
__global__ void __launch_bounds__(SLAB_THREADS) k_slab_pass(const GridDesc g, const SlabPassParams p, const long long outer,
                                                            const long long inner, const long long n_items) {
    __shared__ float Ks[TT * TT];
    __shared__ double red[32];
    if (p.state->done) return;
    constexpr int t = TT;
    for (int i = threadIdx.x; i < TT * TT; i += SLAB_THREADS) Ks[i] = p.Kh[i];
    __syncthreads();
    const int ax = p.axis;
    const int S = g.S[ax], M = g.M[ax];
    float acc = 0.f;
    const int n_batch = BATCH ? p.n_batch : 1;            // batched solves (R18): one source after the other
    for (int bsrc = 0; bsrc < n_batch; ++bsrc) {
    const cf* __restrict__ ds = BATCH ? p.ds + bsrc * p.ds_stride : p.ds;
    cf* __restrict__ u = BATCH ? p.u + bsrc * p.vox_stride : p.u;      // u, x and ds are distinct arrays
    cf* __restrict__ x = BATCH ? p.x + bsrc * p.vox_stride : p.x;
    for (long long item = (long long)blockIdx.x * SLAB_THREADS + threadIdx.x; item < n_items;
         item += (long long)gridDim.x * SLAB_THREADS) {
        const long long in_i = item % inner;
        long long rest = item / inner;
        const int side = (int)(rest % 2);
        rest /= 2;
        const int s = (int)(rest % S);
        const long long o = rest / S;
        int nb = side ? s + 1 : s - 1;
        bool has_nb = true;
        if (nb < 0 || nb >= S) {
            if (g.per[ax]) nb = (nb + S) % S;
            else has_nb = false;
        }
        if constexpr (ACT) {
            // subdomain activation: the edge voxels of an inactive subdomain are left alone
            int s0, s1, s2;
            if (ax == 0) { s0 = s; s1 = (int)(in_i / g.N[2]) / g.M[1]; s2 = (int)(in_i % g.N[2]) / g.M[2]; }
            else if (ax == 1) { s0 = (int)o / g.M[0]; s1 = s; s2 = (int)in_i / g.M[2]; }
            else { s0 = (int)(o / g.N[1]) / g.M[0]; s1 = (int)(o % g.N[1]) / g.M[1]; s2 = s; }
            if (!p.active[(s0 * g.S[1] + s1) * g.S[2] + s2]) continue;
        }
        // side 1 (last t points of s) reads the FIRST t points of s and s+1; side 0 reads the LAST t points
        const long long own0 = ((o * S + s) * 2 * t + (side ? 0 : t)) * inner + in_i;
        const long long nb0 = ((o * S + nb) * 2 * t + (side ? 0 : t)) * inner + in_i;
        cf dv[TT];
#pragma unroll
        for (int q = 0; q < TT; ++q) {
            const cf own = ds[own0 + q * inner];
            cf nbv = make_float2(0.f, 0.f);
            if (has_nb) nbv = ds[nb0 + q * inner];
            dv[q] = make_float2(nbv.x - own.x, nbv.y - own.y);
        }
        // is the voxel an edge point of a later axis?  (constant over the t outputs of this item)
        bool later = false;
        long long vox0, vstride;                      // voxel index of output e: vox0 + e * vstride
        const int ia0 = s * M + (side ? M - t : 0);
        if (ax == 0) {
            const int i1 = (int)(in_i / g.N[2]), i2 = (int)(in_i - (long long)i1 * g.N[2]);
            later = (p.e1 && edge_slot(i1, g.M[1], t) >= 0) || (p.e2 && edge_slot(i2, g.M[2], t) >= 0);
            vox0 = (long long)ia0 * inner + in_i;
            vstride = inner;
        } else if (ax == 1) {
            later = p.e2 && edge_slot((int)in_i, g.M[2], t) >= 0;
            vox0 = (o * g.N[1] + ia0) * inner + in_i;
            vstride = inner;
        } else {
            vox0 = o * g.N[2] + ia0;
            vstride = 1;
        }
#pragma unroll
        for (int e = 0; e < TT; ++e) {
            float sr = 0.f, si = 0.f;
#pragma unroll
            for (int q = 0; q < TT; ++q) {
                const float k = side ? Ks[e * TT + q] : Ks[q * TT + e];
                sr = fmaf(k, dv[q].x, sr);
                si = fmaf(k, dv[q].y, si);
            }
            const cf corr = cmul(p.c, make_float2(sr, si));
            const long long vox = vox0 + e * vstride;
            const cf uu = u[vox];
            const cf r = make_float2(uu.x - corr.x, uu.y - corr.y);
            if (later) {
                u[vox] = r;
            } else {
                const cf xv = x[vox];
                acc += r.x * r.x + r.y * r.y;
                x[vox] = make_float2(xv.x - p.alpha * r.x, xv.y - p.alpha * r.y);
            }
        }
    }
    }
    const double bs = block_sum((double)acc, red);
    grid_reduce_finish(bs, p.partials, p.slot0, p.slot0 + (int)gridDim.x, p.finish, RED_RESIDUAL, p.state, p.hist, red);
}

// Slab pass of the LAST axis (the contiguous one): the t outputs of an item are contiguous voxels.  One thread per
// output (item, e) with e fastest: the TT threads of an item read the same 2 TT values of d (one 128-byte line, served by
// L1) and write TT contiguous voxels, instead of one thread writing 64 bytes per row with rows 8 N2 bytes apart.
template <int TT, bool ACT, bool BATCH>
__global__ void __launch_bounds__(SLAB_THREADS) k_slab_pass_contig(const GridDesc g, const SlabPassParams p, const unsigned n_items) {
    __shared__ float Ks[TT * TT];
    __shared__ double red[32];
    if (p.state->done) return;
    constexpr int t = TT;
    for (int i = threadIdx.x; i < TT * TT; i += SLAB_THREADS) Ks[i] = p.Kh[i];
    __syncthreads();
    const unsigned S = (unsigned)g.S[2];
    const int M = g.M[2];
    const unsigned n_out = n_items * TT;              // <= voxels < 2^31 (2t <= M)
    float acc = 0.f;
    const int n_batch = BATCH ? p.n_batch : 1;            // batched solves (R18): one source after the other
    for (int bsrc = 0; bsrc < n_batch; ++bsrc) {
    const cf* __restrict__ ds = BATCH ? p.ds + bsrc * p.ds_stride : p.ds;
    cf* __restrict__ u = BATCH ? p.u + bsrc * p.vox_stride : p.u;      // u, x and ds are distinct arrays
    cf* __restrict__ x = BATCH ? p.x + bsrc * p.vox_stride : p.x;
    for (unsigned w = blockIdx.x * SLAB_THREADS + threadIdx.x; w < n_out; w += gridDim.x * SLAB_THREADS) {
        const unsigned item = w / TT;
        const int e = (int)(w - item * TT);
        const int side = (int)(item & 1u);
        const unsigned rest = item >> 1;
        const unsigned o = rest / S;                  // grid row i0 * N1 + i1
        const int s = (int)(rest - o * S);
        if constexpr (ACT) {
            const int i0 = (int)(o / (unsigned)g.N[1]), i1 = (int)(o - (unsigned)i0 * (unsigned)g.N[1]);
            if (!p.active[((i0 / g.M[0]) * g.S[1] + i1 / g.M[1]) * g.S[2] + s]) continue;
        }
        int nb = side ? s + 1 : s - 1;
        bool has_nb = true;
        if (nb < 0 || nb >= (int)S) {
            if (g.per[2]) nb = (nb + (int)S) % (int)S;
            else has_nb = false;
        }
        // side 1 (last t points of s) reads the FIRST t points of s and s+1; side 0 reads the LAST t points
        const cf* own = ds + ((long long)(o * S + (unsigned)s) * 2 * t + (side ? 0 : t));
        const cf* nbp = ds + ((long long)(o * S + (unsigned)nb) * 2 * t + (side ? 0 : t));
        float sr = 0.f, si = 0.f;
#pragma unroll
        for (int q = 0; q < TT; ++q) {
            const cf ov = own[q];
            cf nv = make_float2(0.f, 0.f);
            if (has_nb) nv = nbp[q];
            const float k = side ? Ks[e * TT + q] : Ks[q * TT + e];
            sr = fmaf(k, nv.x - ov.x, sr);
            si = fmaf(k, nv.y - ov.y, si);
        }
        const cf corr = cmul(p.c, make_float2(sr, si));
        const long long vox = (long long)o * g.N[2] + s * M + (side ? M - t : 0) + e;
        const cf uu = u[vox];
        const cf r = make_float2(uu.x - corr.x, uu.y - corr.y);
        const cf xv = x[vox];
        acc += r.x * r.x + r.y * r.y;
        x[vox] = make_float2(xv.x - p.alpha * r.x, xv.y - p.alpha * r.y);
    }
    }
    const double bs = block_sum((double)acc, red);
    grid_reduce_finish(bs, p.partials, p.slot0, p.slot0 + (int)gridDim.x, p.finish, RED_RESIDUAL, p.state, p.hist, red);
}

// The pass of the contiguous axis runs one thread per output (k_slab_pass_contig) while it is latency-bound: measured 6 %
// faster at config 3 (131 072 items) and 5-12 % slower at configs 4 and 5 (1.6 M and 4.2 M items) than one thread per item.
static bool slab_pass_contig(const GridDesc& g, int ax) {
    return ax == 2 && (long long)g.N[0] * g.N[1] * g.S[2] * 2 <= (1LL << 18);
}

int slab_pass_blocks(const GridDesc& g, int ax) {
    long long outer = 1, inner = 1;
    for (int d = 0; d < ax; ++d) outer *= g.N[d];
    for (int d = ax + 1; d < 3; ++d) inner *= g.N[d];
    const long long n_items = outer * g.S[ax] * 2 * inner;
    const long long n_threads = slab_pass_contig(g, ax) ? n_items * g.t : n_items;    // one thread per output there
    long long nb = (n_threads + SLAB_THREADS - 1) / SLAB_THREADS;
    if (nb > 1024) nb = 1024;
    return (int)(nb < 1 ? 1 : nb);
}

bool slab_pass_supported(int t) { return t == 2 || t == 4 || t == 8 || t == 16; }

cudaError_t launch_slab_pass(const GridDesc& g, const SlabPassParams& p, cudaStream_t st) {
    const int ax = p.axis;
    long long outer = 1, inner = 1;
    for (int d = 0; d < ax; ++d) outer *= g.N[d];
    for (int d = ax + 1; d < 3; ++d) inner *= g.N[d];
    const long long n_items = outer * g.S[ax] * 2 * inner;
    const int nb = slab_pass_blocks(g, ax);
#define MBS_SLAB_PASS(TTv)                                                                                                  \
    if (contig && p.n_batch > 1) k_slab_pass_contig<TTv, false, true><<<nb, SLAB_THREADS, 0, st>>>(g, p, (unsigned)n_items);      \
    else if (contig && p.active) k_slab_pass_contig<TTv, true, false><<<nb, SLAB_THREADS, 0, st>>>(g, p, (unsigned)n_items);      \
    else if (contig) k_slab_pass_contig<TTv, false, false><<<nb, SLAB_THREADS, 0, st>>>(g, p, (unsigned)n_items);                 \
    else if (p.n_batch > 1) k_slab_pass<TTv, false, true><<<nb, SLAB_THREADS, 0, st>>>(g, p, outer, inner, n_items);              \
    else if (p.active) k_slab_pass<TTv, true, false><<<nb, SLAB_THREADS, 0, st>>>(g, p, outer, inner, n_items);                   \
    else k_slab_pass<TTv, false, false><<<nb, SLAB_THREADS, 0, st>>>(g, p, outer, inner, n_items)
    const bool contig = slab_pass_contig(g, ax);
    switch (g.t) {
        case 2: MBS_SLAB_PASS(2); break;
        case 4: MBS_SLAB_PASS(4); break;
        case 8: MBS_SLAB_PASS(8); break;
        case 16: MBS_SLAB_PASS(16); break;
        default: return cudaErrorNotSupported;
    }
#undef MBS_SLAB_PASS
    return cudaGetLastError();
}

// generic t (any value): one thread per output element
__global__ void __launch_bounds__(SLAB_THREADS) k_slab_generic(const GridDesc g, const SlabParams p,
                                                               const long long outer, const long long inner,
                                                               const long long n_items) {
    if (p.check_done && p.state->done) return;
    const int t = g.t;
    const int ax = p.axis;
    const int S = g.S[ax], M = g.M[ax];
    for (long long item = (long long)blockIdx.x * SLAB_THREADS + threadIdx.x; item < n_items * t;
         item += (long long)gridDim.x * SLAB_THREADS) {
        const long long in_i = item % inner;
        long long rest = item / inner;
        const int e = (int)(rest % t);
        rest /= t;
        const int side = (int)(rest % 2);
        rest /= 2;
        const int s = (int)(rest % S);
        const long long o = rest / S;
        int nb = side ? s + 1 : s - 1;
        bool has_nb = true;
        if (nb < 0 || nb >= S) {
            if (g.per[ax]) nb = (nb + S) % S;
            else has_nb = false;
        }
        long long own0, nb0;
        if (p.compact_in) {
            own0 = ((o * S + s) * 2 * t + (side ? 0 : t)) * inner + in_i;
            nb0 = ((o * S + nb) * 2 * t + (side ? 0 : t)) * inner + in_i;
        } else {
            const long long base_o = o * (long long)g.N[ax] * inner + in_i;
            const long long off = side ? 0 : (long long)(M - t);
            own0 = base_o + ((long long)s * M + off) * inner;
            nb0 = base_o + ((long long)nb * M + off) * inner;
        }
        float sr = 0.f, si = 0.f;
        for (int q = 0; q < t; ++q) {
            cf own = p.in[own0 + q * inner];
            if (p.in2) own = csub(own, p.in2[own0 + q * inner]);
            cf nbv = make_float2(0.f, 0.f);
            if (has_nb) {
                nbv = p.in[nb0 + q * inner];
                if (p.in2) nbv = csub(nbv, p.in2[nb0 + q * inner]);
            }
            const float k = side ? p.Kh[e * t + q] : p.Kh[q * t + e];
            sr = fmaf(k, nbv.x - own.x, sr);
            si = fmaf(k, nbv.y - own.y, si);
        }
        p.out[((o * S + s) * 2 * t + (long long)side * t + e) * inner + in_i] = cmul(p.c, make_float2(sr, si));
    }
}

cudaError_t launch_slab(const GridDesc& g, const SlabParams& p, cudaStream_t st) {
    const int ax = p.axis;
    long long outer = 1, inner = 1;
    for (int d = 0; d < ax; ++d) outer *= g.N[d];
    for (int d = ax + 1; d < 3; ++d) inner *= g.N[d];
    const long long n_items = outer * g.S[ax] * 2 * inner;
    long long nb = (n_items + SLAB_THREADS - 1) / SLAB_THREADS;
    if (nb > 65535LL * 16) nb = 65535LL * 16;
    if (nb < 1) nb = 1;
    switch (g.t) {
#define MBS_SLAB(TTv)                                                                                          \
    if (p.n_batch > 1) k_slab<TTv, true><<<(unsigned)nb, SLAB_THREADS, 0, st>>>(g, p, outer, inner, n_items);     \
    else k_slab<TTv, false><<<(unsigned)nb, SLAB_THREADS, 0, st>>>(g, p, outer, inner, n_items)
        case 2: MBS_SLAB(2); break;
        case 4: MBS_SLAB(4); break;
        case 8: MBS_SLAB(8); break;
        case 16: MBS_SLAB(16); break;
#undef MBS_SLAB
        default: {
            long long nb2 = (n_items * g.t + SLAB_THREADS - 1) / SLAB_THREADS;
            if (nb2 > 65535LL * 16) nb2 = 65535LL * 16;
            k_slab_generic<<<(unsigned)nb2, SLAB_THREADS, 0, st>>>(g, p, outer, inner, n_items);
        }
    }
    return cudaGetLastError();
}

static void slab_geom(const GridDesc& g, int ax, long long* inner, long long* n_items, long long* nb) {
    long long outer = 1;
    *inner = 1;
    for (int d = 0; d < ax; ++d) outer *= g.N[d];
    for (int d = ax + 1; d < 3; ++d) *inner *= g.N[d];
    *n_items = outer * g.S[ax] * 2 * *inner;
    *nb = (*n_items + SLAB_THREADS - 1) / SLAB_THREADS;
    if (*nb > 65535LL * 8) *nb = 65535LL * 8;
    if (*nb < 1) *nb = 1;
}

bool slab_pair_supported(int t) { return t == 2 || t == 4 || t == 8 || t == 16; }

cudaError_t launch_slab_pair(const GridDesc& g, const SlabParams& pA, const SlabParams& pB, cudaStream_t st) {
    long long iA, nA, bA, iB, nB, bB;
    slab_geom(g, pA.axis, &iA, &nA, &bA);
    slab_geom(g, pB.axis, &iB, &nB, &bB);
    const unsigned nb = (unsigned)(bA + bB);
    switch (g.t) {
        case 2: k_slab_pair<2><<<nb, SLAB_THREADS, 0, st>>>(g, pA, pB, iA, nA, iB, nB, (unsigned)bA); break;
        case 4: k_slab_pair<4><<<nb, SLAB_THREADS, 0, st>>>(g, pA, pB, iA, nA, iB, nB, (unsigned)bA); break;
        case 8: k_slab_pair<8><<<nb, SLAB_THREADS, 0, st>>>(g, pA, pB, iA, nA, iB, nB, (unsigned)bA); break;
        case 16: k_slab_pair<16><<<nb, SLAB_THREADS, 0, st>>>(g, pA, pB, iA, nA, iB, nB, (unsigned)bA); break;
        default: return cudaErrorNotSupported;
    }
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// fix-up of the fused last sweep: on every row that lies in a slab of axis 0 or 1,
//   r = r_part - corr_0(d) - corr_1(d),  |r|^2 partial sums,  x <- x - alpha r      (a7-a9)
// r_part = B_diag d - corr_2(d) was left in u by the fused sweep; corr_0(d), corr_1(d) are in the compact
// buffers.  Rows are enumerated without a list: set A = {i0 edge of axis 0} x all i1, then
// set B = {i0 not an edge of axis 0} x {i1 edge of axis 1}.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int edge_index(int q, int M, int t) {   // q in [0, S*2t) -> grid index
    const int s = q / (2 * t), e = q - s * 2 * t;
    return s * M + (e < t ? e : M - 2 * t + e);
}

template <int VEC>
__global__ void __launch_bounds__(PW_THREADS) k_fixup(const GridDesc g, const FixupParams p) {
    __shared__ double red[32];
    if (p.check_done && p.state->done) return;
    const int t = g.t;
    const int nE0 = p.e0 ? g.S[0] * 2 * t : 0, nE1 = p.e1 ? g.S[1] * 2 * t : 0;
    const long long rowsA = (long long)nE0 * g.N[1];
    const long long rowsB = (long long)(g.N[0] - nE0) * nE1;
    const int chunk_len = PW_THREADS * VEC;
    const int nchunks = (g.N[2] + chunk_len - 1) / chunk_len;
    const long long n_work = (rowsA + rowsB) * nchunks;
    float acc = 0.f;
    for (long long work = blockIdx.x; work < n_work; work += gridDim.x) {
        const int chunk = (int)(work % nchunks);
        const long long rid = work / nchunks;
        int i0, i1, q0 = -1, q1 = -1;
        if (rid < rowsA) {
            q0 = (int)(rid / g.N[1]);
            i1 = (int)(rid - (long long)q0 * g.N[1]);
            i0 = edge_index(q0, g.M[0], t);
            if (p.e1) q1 = edge_slot(i1, g.M[1], t);
        } else {
            const long long rb = rid - rowsA;
            const int k0 = (int)(rb / nE1);          // k0-th non-edge index of axis 0
            q1 = (int)(rb - (long long)k0 * nE1);
            i1 = edge_index(q1, g.M[1], t);
            if (p.e0) {
                const int w = g.M[0] - 2 * t;
                const int s = k0 / w;
                i0 = s * g.M[0] + t + (k0 - s * w);
            } else {
                i0 = k0;
            }
        }
        const int i2 = chunk * chunk_len + threadIdx.x * VEC;
        if (i2 >= g.N[2]) continue;
        const long long idx = ((long long)i0 * g.N[1] + i1) * g.N[2] + i2;
        cf r[VEC], xv[VEC];
        load_vec<VEC>(p.u + idx, r);
        load_vec<VEC>(p.x + idx, xv);
        if (q0 >= 0) {
            cf cc[VEC];
            load_vec<VEC>(p.cx0 + ((long long)q0 * g.N[1] + i1) * g.N[2] + i2, cc);
#pragma unroll
            for (int v = 0; v < VEC; ++v) r[v] = csub(r[v], cc[v]);
        }
        if (q1 >= 0) {
            cf cc[VEC];
            load_vec<VEC>(p.cx1 + ((long long)i0 * nE1 + q1) * g.N[2] + i2, cc);
#pragma unroll
            for (int v = 0; v < VEC; ++v) r[v] = csub(r[v], cc[v]);
        }
        if (p.e2) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                const int q2 = edge_slot(i2 + v, g.M[2], t);
                if (q2 >= 0) r[v] = csub(r[v], p.cx2[((long long)i0 * g.N[1] + i1) * (g.S[2] * 2 * t) + q2]);
            }
        }
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            acc += r[v].x * r[v].x + r[v].y * r[v].y;
            xv[v] = make_float2(xv[v].x - p.alpha * r[v].x, xv[v].y - p.alpha * r[v].y);
        }
        store_vec<VEC>(p.x + idx, xv);
    }
    if (p.e2) {
        // set C: the 2t edge points of every line on the rows that are in no slab of axis 0 or 1
        const int E2 = g.S[2] * 2 * t;
        const int w0 = p.e0 ? g.M[0] - 2 * t : g.M[0], w1 = p.e1 ? g.M[1] - 2 * t : g.M[1];
        const long long n0 = (long long)g.S[0] * w0, n1 = (long long)g.S[1] * w1;
        const long long n_items = n0 * n1 * E2;
        for (long long item = (long long)blockIdx.x * PW_THREADS + threadIdx.x; item < n_items;
             item += (long long)gridDim.x * PW_THREADS) {
            const int q2 = (int)(item % E2);
            const long long rr = item / E2;
            const int k1 = (int)(rr % n1), k0 = (int)(rr / n1);
            const int s0 = k0 / w0, s1 = k1 / w1;
            const int i0 = s0 * g.M[0] + (p.e0 ? t : 0) + (k0 - s0 * w0);
            const int i1 = s1 * g.M[1] + (p.e1 ? t : 0) + (k1 - s1 * w1);
            const int i2 = edge_index(q2, g.M[2], t);
            const long long row = (long long)i0 * g.N[1] + i1;
            const long long idx = row * g.N[2] + i2;
            const cf r = csub(p.u[idx], p.cx2[row * E2 + q2]);
            const cf xv = p.x[idx];
            acc += r.x * r.x + r.y * r.y;
            p.x[idx] = make_float2(xv.x - p.alpha * r.x, xv.y - p.alpha * r.y);
        }
    }
    const double bs = block_sum((double)acc, red);
    grid_reduce_finish(bs, p.partials, p.slot0, p.slot0 + (int)gridDim.x, 1, p.reduce_mode, p.state, p.hist, red);
}

int fixup_blocks(const GridDesc& g, int e0, int e1, int e2, int num_sms) {
    const int vec = (g.N[2] % 2 == 0) ? 2 : 1;
    const int chunk_len = PW_THREADS * vec;
    const long long nchunks = (g.N[2] + chunk_len - 1) / chunk_len;
    const long long nE0 = e0 ? g.S[0] * 2 * g.t : 0, nE1 = e1 ? g.S[1] * 2 * g.t : 0;
    long long n_work = (nE0 * g.N[1] + (g.N[0] - nE0) * nE1) * nchunks;
    if (e2) n_work += ((g.N[0] - nE0) * (g.N[1] - nE1) * g.S[2] * 2 * g.t + PW_THREADS - 1) / PW_THREADS;
    long long nb = (long long)num_sms * 8;
    if (nb > MBS_MAX_PARTIALS / 2) nb = MBS_MAX_PARTIALS / 2;
    if (nb > n_work) nb = n_work;
    return (int)(nb < 1 ? 1 : nb);
}

cudaError_t launch_fixup(const GridDesc& g, const FixupParams& p, int nblocks, cudaStream_t st) {
    if (g.N[2] % 2 == 0) k_fixup<2><<<nblocks, PW_THREADS, 0, st>>>(g, p);
    else k_fixup<1><<<nblocks, PW_THREADS, 0, st>>>(g, p);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// mask[row] = 1 if the row of y (N2 contiguous voxels) holds a non-zero value.  Point, line and plane
// sources leave almost every row empty; the fused first sweep skips the load of y there.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_row_mask(const cf* __restrict__ y, unsigned char* __restrict__ mask,
                                                  const long long rows, const int N2) {
    const int lane = threadIdx.x & 31;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long row = warp0; row < rows; row += nwarps) {
        const cf* yr = y + row * N2;
        bool nz = false;
        for (int i = lane; i < N2; i += 32) {
            const cf v = yr[i];
            nz = nz || (v.x != 0.f) || (v.y != 0.f);
        }
        nz = __any_sync(0xffffffffu, nz);
        if (lane == 0) mask[row] = nz ? 1 : 0;
    }
}

cudaError_t launch_row_mask(const cf* y, unsigned char* mask, long long rows, int N2, cudaStream_t st) {
    long long nb = (rows + 7) / 8;
    if (nb > 148 * 16) nb = 148 * 16;
    if (nb < 1) nb = 1;
    k_row_mask<<<(unsigned)nb, 256, 0, st>>>(y, mask, rows, N2);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// out = scale * in
// ---------------------------------------------------------------------------------------------
__global__ void k_scale_copy(const cf* __restrict__ in, cf* __restrict__ out, const cf scale, const long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        out[i] = cmul(scale, in[i]);
}

cudaError_t launch_scale_copy(const cf* in, cf* out, cf scale, long long n, cudaStream_t st) {
    long long nb = (n + 255) / 256;
    if (nb > 148 * 32) nb = 148 * 32;
    k_scale_copy<<<(unsigned)nb, 256, 0, st>>>(in, out, scale, n);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// Subdomain activation ("initially activating only those subdomains that hold a source term.  Neighbouring
// subdomains are activated only after the norm of the transferred field exceeds a certain threshold"; reading R17).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int subdomain_of(const GridDesc& g, int i0, int i1, int i2) {
    return ((i0 / g.M[0]) * g.S[1] + i1 / g.M[1]) * g.S[2] + i2 / g.M[2];
}

// flags[s] = 1 if y or x is non-zero anywhere in subdomain s (flags are zeroed before the launch)
__global__ void __launch_bounds__(256) k_activation_mark(const GridDesc g, const cf* __restrict__ y, const cf* __restrict__ x,
                                                         int* __restrict__ flags) {
    const long long rows = g.voxels / g.N[2];
    const int lane = threadIdx.x & 31;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long row = warp0; row < rows; row += nwarps) {
        const int i1 = (int)(row % g.N[1]), i0 = (int)(row / g.N[1]);
        const cf* yr = y + row * g.N[2];
        const cf* xr = x + row * g.N[2];
        for (int s2 = 0; s2 < g.S[2]; ++s2) {
            bool nz = false;
            for (int i = s2 * g.M[2] + lane; i < (s2 + 1) * g.M[2]; i += 32) {
                const cf a = yr[i], b = xr[i];
                nz = nz || a.x != 0.f || a.y != 0.f || b.x != 0.f || b.y != 0.f;
            }
            if (__any_sync(0xffffffffu, nz) && lane == 0) flags[subdomain_of(g, i0, i1, s2 * g.M[2])] = 1;
        }
    }
}

// list of the active subdomains in ascending order, their number, and the activation iteration of the initial set
__global__ void k_activation_list(const int n_sub, int* flags, int* list, int* n_act, int* act_iter, DevState* state,
                                  const int init) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    int n = 0;
    for (int s = 0; s < n_sub; ++s) {
        if (init) act_iter[s] = flags[s] ? 0 : -1;
        if (flags[s]) list[n++] = s;
    }
    *n_act = n;
    state->n_active = n;
    state->n_sub = n_sub;
}

// One block per (subdomain s, face f = axis*2 + side, chunk): partial sum of |corr_axis(x)|^2 over the t edge points of
// that face of an INACTIVE s whose neighbour across the face is ACTIVE (x_s = 0, so corr is what the neighbour transfers):
//   side 0 (first t points of s):  corr[b] = c sum_a Kh[a][b] x_{s-1}[M-t+a]
//   side 1 (last  t points of s):  corr[a] = c sum_b Kh[a][b] x_{s+1}[b]            (kernels above)
// The last block to finish adds the partials per subdomain in a fixed order, activates s when
// T_s^2 >= thr2 * nu^2, and rebuilds the list.
template <int TT>
__global__ void __launch_bounds__(256) k_activation_step(const GridDesc g, const ActivationState a, const cf* __restrict__ x,
                                                         const float* __restrict__ Kh, const cf c, DevState* state) {
    __shared__ float Ks[TT * TT];
    __shared__ double red[32];
    __shared__ int s_last;
    if (state->done) return;
    const int n_sub = g.S[0] * g.S[1] * g.S[2];
    if (*a.n_act == n_sub) return;                    // everything is active: nothing to decide
    const int t = TT;
    for (int i = threadIdx.x; i < TT * TT; i += blockDim.x) Ks[i] = Kh[i];
    __syncthreads();
    const int ch = blockIdx.x % ACT_CHUNKS;
    const int f = (blockIdx.x / ACT_CHUNKS) % 6;
    const int s = blockIdx.x / (ACT_CHUNKS * 6);
    const int ax = f >> 1, side = f & 1;
    int sd[3];
    sd[2] = s % g.S[2]; sd[1] = (s / g.S[2]) % g.S[1]; sd[0] = s / (g.S[2] * g.S[1]);
    float acc = 0.f;
    bool live = a.flags[s] == 0 && g.a[ax] > 0;
    int nbd[3] = {sd[0], sd[1], sd[2]};
    if (live) {
        int nb = side ? sd[ax] + 1 : sd[ax] - 1;
        if (nb < 0 || nb >= g.S[ax]) {
            if (g.per[ax] && g.S[ax] > 1) nb = (nb + g.S[ax]) % g.S[ax];
            else live = false;
        }
        nbd[ax] = nb;
        if (live) live = a.flags[(nbd[0] * g.S[1] + nbd[1]) * g.S[2] + nbd[2]] != 0;
    }
    if (live) {
        const int d1 = ax == 0 ? 1 : 0, d2 = ax == 2 ? 1 : 2;   // the two transverse axes, d2 the faster one
        const long long stride[3] = {(long long)g.N[1] * g.N[2], (long long)g.N[2], 1LL};
        const int n1 = g.M[d1], n2 = g.M[d2];
        const int n_items = n1 * n2;
        const int per_chunk = (n_items + ACT_CHUNKS - 1) / ACT_CHUNKS;
        const int lo = ch * per_chunk, hi = min(n_items, lo + per_chunk);
        // first point read along the axis: the neighbour's LAST t points (side 0) or FIRST t points (side 1)
        const long long base = ((long long)nbd[ax] * g.M[ax] + (side ? 0 : g.M[ax] - t)) * stride[ax] +
                               (long long)sd[d1] * g.M[d1] * stride[d1] + (long long)sd[d2] * g.M[d2] * stride[d2];
        for (int item = lo + (int)threadIdx.x; item < hi; item += (int)blockDim.x) {
            const int j1 = item / n2, j2 = item - j1 * n2;
            const cf* src = x + base + j1 * stride[d1] + j2 * stride[d2];
            cf v[TT];
#pragma unroll
            for (int q = 0; q < TT; ++q) v[q] = src[q * stride[ax]];
#pragma unroll
            for (int e = 0; e < TT; ++e) {
                float sr = 0.f, si = 0.f;
#pragma unroll
                for (int q = 0; q < TT; ++q) {
                    const float k = side ? Ks[e * TT + q] : Ks[q * TT + e];
                    sr = fmaf(k, v[q].x, sr);
                    si = fmaf(k, v[q].y, si);
                }
                const cf cc = cmul(c, make_float2(sr, si));
                acc += cc.x * cc.x + cc.y * cc.y;
            }
        }
    }
    const double bs = block_sum((double)acc, red);
    if (threadIdx.x == 0) {
        a.partials[blockIdx.x] = bs;
        __threadfence();
        s_last = (atomicAdd(a.ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (int q = threadIdx.x; q < n_sub; q += blockDim.x) {
        if (a.flags[q]) continue;
        double T2 = 0.0;
        for (int i = 0; i < 6 * ACT_CHUNKS; ++i) T2 += __ldcg(&a.partials[q * 6 * ACT_CHUNKS + i]);
        if (T2 >= a.thr2 * state->nu2) {
            a.flags[q] = 1;
            a.act_iter[q] = state->iter;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        *a.ticket = 0;
        int n = 0;
        for (int q = 0; q < n_sub; ++q)
            if (a.flags[q]) a.list[n++] = q;
        *a.n_act = n;
        state->n_active = n;
    }
}

cudaError_t launch_activation_init(const GridDesc& g, const ActivationState& a, const cf* y, const cf* x, DevState* state,
                                   cudaStream_t st) {
    const int n_sub = g.S[0] * g.S[1] * g.S[2];
    cudaError_t e = cudaMemsetAsync(a.flags, 0, sizeof(int) * n_sub, st);
    if (e != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(a.ticket, 0, sizeof(unsigned int), st)) != cudaSuccess) return e;
    k_activation_mark<<<148 * 8, 256, 0, st>>>(g, y, x, a.flags);
    k_activation_list<<<1, 32, 0, st>>>(n_sub, a.flags, a.list, a.n_act, a.act_iter, state, 1);
    return cudaGetLastError();
}

cudaError_t launch_activation_step(const GridDesc& g, const ActivationState& a, const cf* x, const float* Kh, cf c,
                                   DevState* state, cudaStream_t st) {
    const int n_sub = g.S[0] * g.S[1] * g.S[2];
    const unsigned nb = (unsigned)(n_sub * 6 * ACT_CHUNKS);
    switch (g.t) {
        case 2: k_activation_step<2><<<nb, 256, 0, st>>>(g, a, x, Kh, c, state); break;
        case 4: k_activation_step<4><<<nb, 256, 0, st>>>(g, a, x, Kh, c, state); break;
        case 8: k_activation_step<8><<<nb, 256, 0, st>>>(g, a, x, Kh, c, state); break;
        case 16: k_activation_step<16><<<nb, 256, 0, st>>>(g, a, x, Kh, c, state); break;
        default: return cudaErrorNotSupported;
    }
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// setup (double precision): k^2 = kw2 * n^2 + i beta kw2 w(r)   (R3)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double ramp_weight(int i, int N, int W) {
    if (W <= 0) return 0.0;
    double w = 0.0;
    if (i < W) w = (double)(W - i) / (double)W;
    const int j = N - 1 - i;
    if (j < W) w = fmax(w, (double)(W - j) / (double)W);
    return w;
}

__device__ __forceinline__ double2 k2_at(const GridDesc& g, const SetupParams& p, long long idx, double* im_n) {
    const int i2 = (int)(idx % g.N[2]);
    const long long row = idx / g.N[2];
    const int i1 = (int)(row % g.N[1]);
    const int i0 = (int)(row / g.N[1]);
    const cf n = p.n_map[idx];
    const double nr = n.x, ni = n.y;
    *im_n = ni;
    double w = ramp_weight(i0, g.N[0], p.W[0]);
    w = fmax(w, ramp_weight(i1, g.N[1], p.W[1]));
    w = fmax(w, ramp_weight(i2, g.N[2], p.W[2]));
    return make_double2(p.kw2 * (nr * nr - ni * ni), p.kw2 * (2.0 * nr * ni) + p.beta * p.kw2 * w);
}

__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

__global__ void __launch_bounds__(256) k_setup(const GridDesc g, const SetupParams p, const int pass, double* out,
                                               cf* bdiag) {
    __shared__ double sm[5][8];
    double mn_re = CUDART_INF, mx_re = -CUDART_INF, mn_im = CUDART_INF, mx_im = -CUDART_INF, mn_n = CUDART_INF;
    double vmax2 = 0.0;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < g.voxels;
         idx += (long long)gridDim.x * blockDim.x) {
        double im_n;
        const double2 k2 = k2_at(g, p, idx, &im_n);
        if (pass == 0) {
            // fmin / fmax drop a NaN operand: a non-finite voxel of n is carried explicitly as +inf in the maximum of
            // Re k^2, which mbs_set_potential rejects (MBS_ERR_NUMERIC)
            if (!isfinite(k2.x) || !isfinite(k2.y)) mx_re = CUDART_INF;
            mn_re = fmin(mn_re, k2.x); mx_re = fmax(mx_re, k2.x);
            mn_im = fmin(mn_im, k2.y); mx_im = fmax(mx_im, k2.y);
            mn_n = fmin(mn_n, im_n);
        } else {
            const double dr = k2.x - p.k02_re, di = k2.y - p.k02_im;
            if (pass == 1) {
                vmax2 = fmax(vmax2, dr * dr + di * di);
            } else {
                // B_diag = 1 - c (k^2 - k0^2)
                const double br = 1.0 - (p.c_re * dr - p.c_im * di);
                const double bi = -(p.c_re * di + p.c_im * dr);
                bdiag[idx] = make_float2((float)br, (float)bi);
                if (p.bdiag64) { p.bdiag64[2 * idx] = br; p.bdiag64[2 * idx + 1] = bi; }
            }
        }
    }
    if (pass == 2) return;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (pass == 0) {
        mn_re = warp_min(mn_re); mx_re = warp_max(mx_re); mn_im = warp_min(mn_im); mx_im = warp_max(mx_im);
        mn_n = warp_min(mn_n);
        if (lane == 0) { sm[0][wid] = mn_re; sm[1][wid] = mx_re; sm[2][wid] = mn_im; sm[3][wid] = mx_im; sm[4][wid] = mn_n; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < 8; ++w) {
                sm[0][0] = fmin(sm[0][0], sm[0][w]); sm[1][0] = fmax(sm[1][0], sm[1][w]);
                sm[2][0] = fmin(sm[2][0], sm[2][w]); sm[3][0] = fmax(sm[3][0], sm[3][w]);
                sm[4][0] = fmin(sm[4][0], sm[4][w]);
            }
            for (int q = 0; q < 5; ++q) out[blockIdx.x * 5 + q] = sm[q][0];
        }
    } else {
        vmax2 = warp_max(vmax2);
        if (lane == 0) sm[0][wid] = vmax2;
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < 8; ++w) sm[0][0] = fmax(sm[0][0], sm[0][w]);
            out[blockIdx.x] = sm[0][0];
        }
    }
}

cudaError_t launch_setup(const GridDesc& g, const SetupParams& p, int pass, double* out, cf* bdiag, int nblocks,
                         cudaStream_t st) {
    k_setup<<<nblocks, 256, 0, st>>>(g, p, pass, out, bdiag);
    return cudaGetLastError();
}

}  // namespace mbs
