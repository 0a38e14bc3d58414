// line_merged.cuh -- last sweep of iteration n merged with the first sweep of iteration n+1 (warp-line kernel).
//
// On a row that lies in no slab of axis 0 or 1, everything the next iteration's first sweep needs is on chip at
// the end of the last sweep: x_new of the line, B_diag of the line, and (through a small exchange between the
// warps that hold the segments of the same grid row) the edge values for the corrections along the line.  So
// the kernel goes on and forms u_next = B_diag x_new + y_vec - corr_2(x_new), runs the forward FFT of the line
// and stores it: the next iteration starts at its second sweep.  Saved per voxel and iteration: the re-read of
// x and B_diag (16 B of the 112 B ledger, "beyond the floor" row of SURVEY 8(d)).
//
//   inverse FFT -> u' ;  d = x - u' (a6) ;  r = B_diag d - corr_2(d) (a7; corr_2 from the exchanged edge values)
//   non-slab row:  |r|^2 (a8), x_new = x - alpha r (a9) -> x ;  u_next (a1, a2) -> forward FFT (a3) -> u
//   slab row:      d -> compact buffers of axes 0/1, r -> u in place; the slab passes (kernels.cu) finish the row
//                  and the slab-rows-only first sweep (line_kernels.cuh) produces its u_next afterwards.
//
// Row groups: the S2 segments of a grid row are S2 consecutive lines.  With LW = 32/T lines per warp either one
// warp holds whole rows (LW % S2 == 0: exchange + __syncwarp) or G = S2/LW consecutive warps of the CTA hold one
// row (exchange + named barrier over those G warps).  Both need no block-wide barrier.
#pragma once
#include "line_kernels.cuh"

namespace mbs {

template <class PL, int NWARP>
constexpr bool line_merge_shape_ok(int S2) {
    constexpr int LW = 32 / PL::T;
    return (LW % S2 == 0) || (S2 % LW == 0 && S2 / LW <= NWARP && NWARP % (S2 / LW) == 0);
}

template <class PL, int NWARP>
constexpr size_t line_merged_smem_bytes(int t) {
    // line scratch + twiddles + K_t (as line_body) + exchange buffers of 2t edge values per line: d and x_new, two rounds
    return line_smem_bytes<PL, NWARP>(t) + sizeof(cf) * (size_t)(4 * NWARP * (32 / PL::T) * 2 * t);
}

// corr_2 at edge slot e (first t: e < t, last t: e >= t) of line `li` (CTA-local line index, segment `seg` of its
// row) from the exchanged edge values ex[line][2t] of the lines of the same row.  Same formulas as fused_corr2.
__device__ __forceinline__ cf merged_corr2(const cf* ex, const float* Ks, const int t, const int S2, const int per2, const cf c,
                                           const int li, const int seg, const int e) {
    const int t2 = 2 * t;
    const bool last = e >= t;
    const int k = last ? e - t : e;
    int nb = last ? seg + 1 : seg - 1;
    bool has_nb = true;
    if (nb < 0 || nb >= S2) {
        if (per2) nb = (nb + S2) % S2;
        else has_nb = false;
    }
    const cf* own = ex + li * t2 + (last ? 0 : t);                 // last edge reads FIRST points
    const cf* nbp = ex + (li - seg + nb) * t2 + (last ? 0 : t);
    float sr = 0.f, si = 0.f;
    for (int q = 0; q < t; ++q) {
        const float kk = last ? Ks[k * t + q] : Ks[q * t + k];
        const cf ov = own[q];
        cf dv = make_float2(-ov.x, -ov.y);
        if (has_nb) {
            const cf nv = nbp[q];
            dv = make_float2(nv.x - ov.x, nv.y - ov.y);
        }
        sr = fmaf(kk, dv.x, sr);
        si = fmaf(kk, dv.y, si);
    }
    return cmul(c, make_float2(sr, si));
}

template <int G>
__device__ __forceinline__ void row_group_sync(const int group) {
    if constexpr (G <= 1) {
        __syncwarp();
    } else {
        asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "n"(32 * G) : "memory");
    }
}

template <class PL, int NWARP, int G>
__device__ __forceinline__ void line_merged_body(const FusedParams& p, const cf* __restrict__ tw_global, cf* smem, double* red) {
    constexpr int M = PL::M, P = PL::P, T = PL::T, NT = NWARP * 32;
    static_assert(T <= 32 && 32 % T == 0, "a line must fit in one warp");
    constexpr int LW = 32 / T;
    constexpr int LSE = line_scratch_elems<PL>();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int t = p.t, t2 = 2 * p.t;
    cf* tw = smem;
    cf* scratch = tw + M + (warp * LW + lane / T) * LSE;
    float* Ks = reinterpret_cast<float*>(tw + M + NWARP * LW * LSE);
    cf* ex0 = reinterpret_cast<cf*>(Ks + ((t * t + 3) / 4) * 4);   // exchange buffers [2][NWARP*LW][2t]
    fill_warp_twiddles<PL>(tw, tw_global, tid, NT);   // per-pass [r][k] layout: conflict-free for lanes along a line
    if (p.a2) for (int i = tid; i < t * t; i += NT) Ks[i] = p.Kh[i];
    __syncthreads();
    const int jt = lane % T, lsub = lane / T;
    const int li = warp * LW + lsub;                  // CTA-local line index
    const int group = warp / (G > 0 ? G : 1);
    const unsigned n_lines = (unsigned)p.n_lines;
    const unsigned n_units = (n_lines + LW - 1) / LW;
    // every warp of a row group runs the same number of rounds (n_lines is a multiple of S2 and units of a group
    // are consecutive), so the group barriers below match up
    const unsigned rounds = (n_units + gridDim.x * NWARP - 1) / (gridDim.x * NWARP);
    float acc = 0.f;
    for (unsigned k = 0; k < rounds; ++k) {
        const unsigned unit = (k * gridDim.x + blockIdx.x) * NWARP + warp;
        const unsigned line = unit * LW + lsub;
        const bool valid = unit < n_units && line < n_lines;
        const unsigned row = valid ? line / (unsigned)p.S2 : 0u;
        const int seg = valid ? (int)(line - row * (unsigned)p.S2) : 0;
        const int i0 = (int)(row / (unsigned)p.N1), i1 = (int)(row - (unsigned)i0 * (unsigned)p.N1);
        long long o0 = -1, o1 = -1;
        if (valid && p.e0) {
            const int q = line_edge_slot(i0, p.M0, t);
            if (q >= 0) o0 = ((long long)q * p.N1 + i1) * p.N2 + (long long)seg * M;
        }
        if (valid && p.e1) {
            const int q = line_edge_slot(i1, p.M1, t);
            if (q >= 0) o1 = ((long long)i0 * (p.S1 * t2) + q) * p.N2 + (long long)seg * M;
        }
        const bool slab_row = (o0 >= 0) || (o1 >= 0);
        const long long gl = (long long)line * M;
        cf* exd = ex0 + (size_t)(k & 1u) * 2 * (NWARP * LW * t2);        // edge values of d, then of x_new
        cf* exx = exd + NWARP * LW * t2;
        cf v[P], xr[P], br[P];
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            v[m] = valid ? cswap(p.u[gl + jt + m * T]) : make_float2(0.f, 0.f);
        });
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            xr[m] = valid ? p.x[gl + jt + m * T] : make_float2(0.f, 0.f);
            br[m] = valid ? p.bdiag[gl + jt + m * T] : make_float2(0.f, 0.f);
        });
        fft_line_forward_warp<PL>(v, scratch, jt, tw);
        // d = x - u'; publish its edge values to the row group
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            const int pidx = jt + m * T;
            v[m] = csub(xr[m], cswap(v[m]));
            if (p.a2 && (pidx < t || pidx >= M - t)) exd[li * t2 + (pidx < t ? pidx : pidx - (M - t2))] = v[m];
        });
        if (p.a2) row_group_sync<G>(group);
        // r = B_diag d - corr_2(d); finish the row or hand it to the slab passes
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            const int pidx = jt + m * T;
            cf r = cmul(br[m], v[m]);
            if (valid && p.a2 && (pidx < t || pidx >= M - t))
                r = csub(r, merged_corr2(exd, Ks, t, p.S2, p.per2, p.c, li, seg, pidx < t ? pidx : pidx - (M - t2)));
            if (valid && slab_row) {
                if (o0 >= 0) p.ds0[o0 + pidx] = v[m];
                if (o1 >= 0) p.ds1[o1 + pidx] = v[m];
                p.u[gl + pidx] = r;
            } else {
                acc += r.x * r.x + r.y * r.y;          // (an invalid line holds zeros)
                xr[m] = make_float2(xr[m].x - p.alpha * r.x, xr[m].y - p.alpha * r.y);
                if (valid) p.x[gl + pidx] = xr[m];
                if (p.a2 && (pidx < t || pidx >= M - t)) exx[li * t2 + (pidx < t ? pidx : pidx - (M - t2))] = xr[m];
            }
        });
        if (p.a2) row_group_sync<G>(group);
        // first sweep of the next iteration on the finished row: u_next = B_diag x_new + y_vec - corr_2(x_new)
        const bool has_y = valid && !slab_row && p.y != nullptr && (p.ymask == nullptr || p.ymask[row] != 0);
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            const int pidx = jt + m * T;
            cf un = cmul(br[m], xr[m]);
            if (valid && p.a2 && !slab_row && (pidx < t || pidx >= M - t))
                un = csub(un, merged_corr2(exx, Ks, t, p.S2, p.per2, p.c, li, seg, pidx < t ? pidx : pidx - (M - t2)));
            v[m] = un;
        });
        if (has_y) {
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = cadd(v[m], cmul(p.ysc, p.y[gl + jt + m * T]));
            });
        }
        fft_line_forward_warp<PL>(v, scratch, jt, tw);   // (every lane takes part; slab rows discard the result)
        if (valid && !slab_row) {
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                p.u[gl + jt + m * T] = v[m];
            });
        }
    }
    const double bs = block_sum((double)acc, red);
    grid_reduce_finish(bs, p.partials, p.slot0, p.n_total, p.finish, p.reduce_mode, p.state, p.hist, red);
}

}  // namespace mbs
