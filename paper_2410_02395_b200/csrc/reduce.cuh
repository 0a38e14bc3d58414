// reduce.cuh -- fixed-order block / grid reductions of the residual partial sums (a8 of the scope table,
// P:130) and the device-side stop decision (a10).  Device only.
#pragma once
#include "mbs_internal.h"

namespace mbs {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the block in a fixed order; the result is valid in warp 0.  red: 32 doubles of shared memory.
__device__ __forceinline__ double block_sum(double v, double* red) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) red[wid] = v;
    __syncthreads();
    const int nw = (blockDim.x + 31) >> 5;
    double r = (threadIdx.x < nw) ? red[threadIdx.x] : 0.0;
    if (wid == 0) r = warp_sum(r);
    return r;
}

// Every block of the launch calls this with its partial sum (valid in thread 0).  The partial goes to
// partials[slot0 + blockIdx.x].  If `finish` is set, the last block to arrive adds partials[0 .. n_total)
// in index order (bitwise reproducible, no host round trip) and finishes according to `mode`:
//   RED_NU2       nu^2 = sum                                   (||Gamma^-1 y_vec||^2)
//   RED_RESIDUAL  eps_n = sqrt(sum / nu^2) -> hist[n], n + 1 -> iter, stop flag (R7, R8)
//   RED_PLAIN     last_sum = sum
//   RED_XNORM     xnorm2 = sum (last_sum untouched: the host derives eps from it)
// partials written by earlier launches on the same stream (slots below slot0) are included.
__device__ __forceinline__ void grid_reduce_finish(double block_partial, double* partials, int slot0, int n_total,
                                                   int finish, int mode, DevState* s, double* hist, double* red) {
    __shared__ int s_last;
    if (threadIdx.x == 0) {
        partials[slot0 + blockIdx.x] = block_partial;
        s_last = 0;
        if (finish) {
            __threadfence();
            const unsigned int ticket = atomicAdd(&s->ticket, 1u);
            s_last = (ticket == gridDim.x - 1);
        }
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double acc = 0.0;
    for (int i = threadIdx.x; i < n_total; i += blockDim.x) acc += __ldcg(&partials[i]);
    const double total = block_sum(acc, red);
    if (threadIdx.x == 0) {
        s->ticket = 0;
        if (mode != RED_XNORM) s->last_sum = total;
        if (mode == RED_XNORM) {
            s->xnorm2 = total;
        } else if (mode == RED_NU2) {
            s->nu2 = total;
        } else if (mode == RED_RESIDUAL) {
            const double eps = sqrt(total / s->nu2);
            const int n = s->iter;
            if (hist) hist[n] = eps;
            s->iter = n + 1;
            if (!(eps == eps) || eps > 1.0e300) s->done = 3;      // NaN / Inf
            else if (eps < s->tol) s->done = 1;
            else if (n + 1 >= s->max_iter) s->done = 2;
        }
    }
}

}  // namespace mbs
