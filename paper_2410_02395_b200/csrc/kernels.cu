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

namespace mbs {

// ---------------------------------------------------------------------------------------------
// block reduction helpers (fixed order -> bitwise reproducible sums)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ double block_sum(double v, double* red /*[32]*/) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) red[wid] = v;
    __syncthreads();
    const int nw = (blockDim.x + 31) >> 5;
    double r = (threadIdx.x < nw) ? red[threadIdx.x] : 0.0;
    if (wid == 0) r = warp_sum(r);
    return r;  // valid in warp 0
}

// Called by every block with its partial sum; the last block to arrive adds all partials in index
// order and finishes the reduction (no extra launch, no host round trip).
__device__ void finish_reduction(double block_partial, const PointwiseParams& p, double* red) {
    __shared__ int s_last;
    if (threadIdx.x == 0) {
        p.partials[blockIdx.x] = block_partial;
        __threadfence();
        const unsigned int ticket = atomicAdd(&p.state->ticket, 1u);
        s_last = (ticket == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double acc = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += blockDim.x) acc += __ldcg(&p.partials[i]);
    const double total = block_sum(acc, red);
    if (threadIdx.x == 0) {
        DevState* s = p.state;
        s->ticket = 0;
        s->last_sum = total;
        if (p.reduce == RED_NU2) {
            s->nu2 = total;
        } else if (p.reduce == RED_RESIDUAL) {
            const double eps = sqrt(total / s->nu2);
            const int n = s->iter;
            if (p.hist) p.hist[n] = eps;
            s->iter = n + 1;
            if (!(eps == eps) || eps > 1.0e300) s->done = 3;      // NaN / Inf
            else if (eps < s->tol) s->done = 1;
            else if (n + 1 >= s->max_iter) s->done = 2;
        }
    }
}

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
        finish_reduction(bs, p, red);
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

template <int TT>
__global__ void __launch_bounds__(SLAB_THREADS) k_slab(const GridDesc g, const SlabParams p, const long long outer,
                                                       const long long inner, const long long n_items) {
    __shared__ float Ks[TT * TT];
    if (p.check_done && p.state->done) return;
    const int t = (TT > 0) ? TT : g.t;
    for (int i = threadIdx.x; i < TT * TT; i += SLAB_THREADS) Ks[i] = p.Kh[i];
    __syncthreads();
    const int ax = p.axis;
    const int S = g.S[ax], M = g.M[ax];
    const long long axis_stride = inner;
    for (long long item = (long long)blockIdx.x * SLAB_THREADS + threadIdx.x; item < n_items;
         item += (long long)gridDim.x * SLAB_THREADS) {
        const long long in_i = item % inner;
        long long rest = item / inner;
        const int side = (int)(rest % 2);
        rest /= 2;
        const int s = (int)(rest % S);
        const long long o = rest / S;
        // neighbour subdomain
        int nb = side ? s + 1 : s - 1;
        bool has_nb = true;
        if (nb < 0 || nb >= S) {
            if (g.per[ax]) nb = (nb + S) % S;
            else has_nb = false;
        }
        const long long base_o = o * (long long)g.N[ax] * inner + in_i;
        // side 1 reads the FIRST t points of own and neighbour; side 0 reads the LAST t points
        const long long off = side ? 0 : (long long)(M - t);
        const long long own0 = base_o + ((long long)s * M + off) * axis_stride;
        const long long nb0 = base_o + ((long long)nb * M + off) * axis_stride;
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
        const long long base_o = o * (long long)g.N[ax] * inner + in_i;
        const long long off = side ? 0 : (long long)(M - t);
        const long long own0 = base_o + ((long long)s * M + off) * inner;
        const long long nb0 = base_o + ((long long)nb * M + off) * inner;
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
        case 2: k_slab<2><<<(unsigned)nb, SLAB_THREADS, 0, st>>>(g, p, outer, inner, n_items); break;
        case 4: k_slab<4><<<(unsigned)nb, SLAB_THREADS, 0, st>>>(g, p, outer, inner, n_items); break;
        case 8: k_slab<8><<<(unsigned)nb, SLAB_THREADS, 0, st>>>(g, p, outer, inner, n_items); break;
        case 16: k_slab<16><<<(unsigned)nb, SLAB_THREADS, 0, st>>>(g, p, outer, inner, n_items); break;
        default: {
            long long nb2 = (n_items * g.t + SLAB_THREADS - 1) / SLAB_THREADS;
            if (nb2 > 65535LL * 16) nb2 = 65535LL * 16;
            k_slab_generic<<<(unsigned)nb2, SLAB_THREADS, 0, st>>>(g, p, outer, inner, n_items);
        }
    }
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
