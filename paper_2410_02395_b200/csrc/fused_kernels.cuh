// fused_kernels.cuh -- the first and the last sweep of one iteration of Eq. (6), fused with the
// contiguous-axis FFT of the propagator (device only; instantiated per FFT size in fft_inst.cu).
//
//   FUSED_S1 : u = B x + y_vec  (a1, a2 of the scope table)  -> forward FFT along the last axis -> u
//   FUSED_S5 : inverse FFT along the last axis of u -> u' ;  d = x - u' (a6) ;  r = B d (a7) ;
//              residual partial sums (a8) ;  x <- x - alpha r (a9)
//   FUSED_1D : both around the whole propagator (forward FFT, Fourier kernel, inverse FFT: a3-a5) -- a
//              1-D problem is one kernel per iteration.
//
// A tile is C consecutive lines of M contiguous voxels = C / S2 complete grid rows (S2 subdomains along
// the last axis), so the edge-slab correction ALONG THE LAST AXIS (wrap-around C_ss and transfer
// A_{s,s+-1}) is computed inside the CTA from the 2t edge points of each line: no halo copy,
// no extra pass.  The corrections along the other axes couple different rows:
//   S1 subtracts corr_0(x), corr_1(x) read from the compact buffers the slab kernel wrote (rows whose
//      index along axis 0 / 1 is one of the 2t edge points of a subdomain; all other rows skip it);
//   S5 finishes every row that is in no slab of axes 0/1; for a slab row it leaves x untouched, writes
//      d to the compact buffers and r_part = B_diag d - corr_2(d) in place into u (free at that point);
//      the fix-up kernels (kernels.cu) then apply corr_0(d), corr_1(d) there.
#pragma once
#include "fft_kernels.cuh"
#include "reduce.cuh"

namespace mbs {

template <class PL, int C>
constexpr int fused_smem_elems(int t) { return PL::M + C * (PL::M + 1) + 2 * C * 2 * t + (t * t + 1) / 2 + 2 * C + (C + 1) / 2; }

struct cf2 { cf a, b; };   // two neighbouring voxels = one 128-bit access
__device__ __forceinline__ cf2 ld2(const cf* p) {
    const float4 r = *reinterpret_cast<const float4*>(p);
    cf2 o;
    o.a = make_float2(r.x, r.y);
    o.b = make_float2(r.z, r.w);
    return o;
}
__device__ __forceinline__ void st2(cf* p, const cf a, const cf b) { *reinterpret_cast<float4*>(p) = make_float4(a.x, a.y, b.x, b.y); }

// subdomain-local edge slot in [0, 2t) of index i, or -1; adds s*2t
__device__ __forceinline__ int fused_edge_slot(int i, int M, int t) {
    const int s = i / M, e = i - s * M;
    if (e < t) return s * 2 * t + e;
    if (e >= M - t) return s * 2 * t + t + (e - (M - t));
    return -1;
}

// corr_2 for every line of the tile from its edge values ed[line][2t] (first t, last t) into ce[line][2t]
// (P:124-128 read with P:106; same formulas as k_slab):
//   last  t points, index a:  c * sum_b Kh[a][b] (first_{s+1}[b] - first_s[b])
//   first t points, index b:  c * sum_a Kh[a][b] (last_{s-1}[a]  - last_s[a])
template <int C>
__device__ __forceinline__ void fused_corr2(const cf* ed, cf* ce, const float* Ks, const int t, const int S2, const int per2,
                                            const cf c, const int nvalid, const int tid, const int NT) {
    const int per_line = 2 * t;
    for (int o = tid; o < nvalid * per_line; o += NT) {
        const int line = o / per_line, e = o - line * per_line;
        const int s = line % S2;
        const bool last = e >= t;
        const int k = last ? e - t : e;
        int nb = last ? s + 1 : s - 1;
        bool has_nb = true;
        if (nb < 0 || nb >= S2) {
            if (per2) nb = (nb + S2) % S2;
            else has_nb = false;
        }
        const cf* own = ed + line * per_line + (last ? 0 : t);                  // last edge reads FIRST points
        const cf* nbp = ed + (line - s + nb) * per_line + (last ? 0 : t);
        float sr = 0.f, si = 0.f;
        for (int q = 0; q < t; ++q) {
            const float kk = last ? Ks[k * t + q] : Ks[q * t + k];
            cf dv = make_float2(-own[q].x, -own[q].y);
            if (has_nb) dv = make_float2(nbp[q].x - own[q].x, nbp[q].y - own[q].y);
            sr = fmaf(kk, dv.x, sr);
            si = fmaf(kk, dv.y, si);
        }
        ce[o] = cmul(c, make_float2(sr, si));
    }
}

// first sweep, one line: u = B_diag x + y_vec - corr_0(x) - corr_1(x) - corr_2(x) -> tile
template <int M, bool SLAB>
__device__ __forceinline__ void fused_pro_line(const FusedParams& p, const cf* xl, const cf* bl, const long long gl, cf* trow,
                                               const cf* cel, const int lane, const bool has_y, const long long o0,
                                               const long long o1) {
    // xl, bl: this line of x and B_diag
    constexpr int EP2 = (M + 63) / 64;
    const int t = p.t;
    const cf* yl = p.y + gl;
#pragma unroll
    for (int k = 0; k < EP2; ++k) {
        const int q = 2 * lane + 64 * k;
        if (M % 64 == 0 || q < M) {
            const cf2 xv = ld2(xl + q), bv = ld2(bl + q);
            cf v0 = cmul(bv.a, xv.a), v1 = cmul(bv.b, xv.b);
            if (has_y) {
                const cf2 yv = ld2(yl + q);
                v0 = cadd(v0, cmul(p.ysc, yv.a));
                v1 = cadd(v1, cmul(p.ysc, yv.b));
            }
            if constexpr (SLAB) {
                if (o0 >= 0) {
                    const cf2 cc = ld2(p.cx0 + o0 + q);
                    v0 = csub(v0, cc.a);
                    v1 = csub(v1, cc.b);
                }
                if (o1 >= 0) {
                    const cf2 cc = ld2(p.cx1 + o1 + q);
                    v0 = csub(v0, cc.a);
                    v1 = csub(v1, cc.b);
                }
            }
            if (p.a2 && (64 * k < t || 64 * k + 64 > M - t)) {       // only the first / last chunks touch the edges
                if (q < t) v0 = csub(v0, cel[q]);
                else if (q >= M - t) v0 = csub(v0, cel[q - (M - 2 * t)]);
                if (q + 1 < t) v1 = csub(v1, cel[q + 1]);
                else if (q + 1 >= M - t) v1 = csub(v1, cel[q + 1 - (M - 2 * t)]);
            }
            trow[q] = v0;
            trow[q + 1] = v1;
        }
    }
}

// last sweep, one line: d = x - u'; r = B_diag d - corr_2(d); finish the row or hand it to the fix-up
template <int M, bool SLAB>
__device__ __forceinline__ float fused_epi_line(const FusedParams& p, const cf* xl, const cf* bl, const long long gl,
                                                const cf* trow, const cf* cel, const int lane, const long long o0,
                                                const long long o1) {
    constexpr int EP2 = (M + 63) / 64;
    const int t = p.t;
    cf* xout = p.x + gl;
    float acc = 0.f;
#pragma unroll
    for (int k = 0; k < EP2; ++k) {
        const int q = 2 * lane + 64 * k;
        if (M % 64 == 0 || q < M) {
            const cf2 xv = ld2(xl + q), bv = ld2(bl + q);
            cf d0 = csub(xv.a, trow[q]), d1 = csub(xv.b, trow[q + 1]);
            if (p.dref) {                                     // split iterate: d = d_ref + (delta - u')
                const cf2 dv = ld2(p.dref + gl + q);
                d0 = cadd(d0, dv.a);
                d1 = cadd(d1, dv.b);
            }
            cf r0 = cmul(bv.a, d0), r1 = cmul(bv.b, d1);
            if (p.a2 && (64 * k < t || 64 * k + 64 > M - t)) {
                if (q < t) r0 = csub(r0, cel[q]);
                else if (q >= M - t) r0 = csub(r0, cel[q - (M - 2 * t)]);
                if (q + 1 < t) r1 = csub(r1, cel[q + 1]);
                else if (q + 1 >= M - t) r1 = csub(r1, cel[q + 1 - (M - 2 * t)]);
            }
            if (p.rref) {                                     // split iterate, complex128 residual: r = r_ref + B (delta - u')
                const cf2 rv = ld2(p.rref + gl + q);
                r0 = cadd(r0, rv.a);
                r1 = cadd(r1, rv.b);
            }
            if constexpr (!SLAB) {
                acc += r0.x * r0.x + r0.y * r0.y + r1.x * r1.x + r1.y * r1.y;
                st2(xout + q, make_float2(xv.a.x - p.alpha * r0.x, xv.a.y - p.alpha * r0.y),
                    make_float2(xv.b.x - p.alpha * r1.x, xv.b.y - p.alpha * r1.y));
            } else {
                if (o0 >= 0) st2(p.ds0 + o0 + q, d0, d1);
                if (o1 >= 0) st2(p.ds1 + o1 + q, d0, d1);
                st2(p.u + gl + q, r0, r1);
            }
        }
    }
    return acc;
}

// per-line slab information for axes 0 and 1 (compact row offsets, -1 = not a slab row) and the source-row flag
template <int M>
__device__ __forceinline__ void fused_line_info(const FusedParams& p, const unsigned gline, long long* loff2, int* lflag1) {
    const int t = p.t, t2 = 2 * p.t;
    const unsigned row = gline / (unsigned)p.S2;
    const int seg = (int)(gline - row * (unsigned)p.S2);
    const int i0 = (int)(row / (unsigned)p.N1), i1 = (int)(row - (unsigned)i0 * (unsigned)p.N1);
    long long o0 = -1, o1 = -1;
    if (p.e0) {
        const int q = fused_edge_slot(i0, p.M0, t);
        if (q >= 0) o0 = ((long long)q * p.N1 + i1) * p.N2 + (long long)seg * M;
    }
    if (p.e1) {
        const int q = fused_edge_slot(i1, p.M1, t);
        if (q >= 0) o1 = ((long long)i0 * (p.S1 * t2) + q) * p.N2 + (long long)seg * M;
    }
    loff2[0] = o0;
    loff2[1] = o1;
    *lflag1 = (p.y != nullptr) && (p.ymask == nullptr || p.ymask[row] != 0);
}

template <class PL, int C, int MODE>
__device__ __forceinline__ void fused_contig_body(const FusedParams& p, const cf* __restrict__ tw_global, cf* smem,
                                                  double* red) {
    constexpr int M = PL::M, P = PL::P, T = PL::T, NT = T * C, LS = M + 1;
    constexpr int NW = NT / 32;                       // warps
    constexpr int EP2 = (M + 63) / 64;                // 128-bit accesses per lane per line
    static_assert(M % 2 == 0, "lines are moved as pairs of voxels");
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int t = p.t, t2 = 2 * p.t;
    cf* tw = smem;
    cf* tile = tw + M;
    cf* ed = tile + C * LS;                           // edge values  [C][2t]
    cf* ce = ed + C * t2;                             // corr_2       [C][2t]
    float* Ks = reinterpret_cast<float*>(ce + C * t2);                   // [t*t]
    long long* loff = reinterpret_cast<long long*>(Ks + ((t * t + 1) / 2) * 2);   // per line: compact row offsets (axis 0, axis 1), -1 = none
    int* lflag = reinterpret_cast<int*>(loff + 2 * C);                   // per line: bit 0 = the source row is not all zero
    for (int i = tid; i < M; i += NT) tw[i] = tw_global[i];
    if (p.a2) for (int i = tid; i < t * t; i += NT) Ks[i] = p.Kh[i];
    const int c_ = tid % C, jt = tid / C;
    const unsigned n_lines = (unsigned)p.n_lines;     // < 2^31 (mbs_create)
    float acc = 0.f;
    for (unsigned tix = blockIdx.x; tix < (unsigned)p.n_tiles; tix += gridDim.x) {
        const unsigned line0 = tix * C;
        const int nvalid = (int)((n_lines - line0) < (unsigned)C ? (n_lines - line0) : (unsigned)C);
        __syncthreads();                              // previous tile fully consumed; tables loaded
        // per-line slab information for axes 0 and 1
        if (tid < nvalid) fused_line_info<M>(p, line0 + tid, loff + 2 * tid, lflag + tid);
        const long long g0 = (long long)line0 * M;    // global index of the tile's first voxel
        if constexpr (MODE != FUSED_S5) {
            // ---- prologue: u = B_diag x + y_vec - corr_0(x) - corr_1(x) - corr_2(x) ----
            if (p.a2) {
                for (int o = tid; o < nvalid * t2; o += NT) {
                    const int line = o / t2, e = o - line * t2;
                    ed[o] = p.x[g0 + (long long)line * M + (e < t ? e : M - t2 + e)];
                }
                __syncthreads();
                fused_corr2<C>(ed, ce, Ks, t, p.S2, p.per2, p.c, nvalid, tid, NT);
            }
            __syncthreads();
            for (int line = warp; line < nvalid; line += NW) {
                const long long gl = g0 + (long long)line * M;
                const long long o0 = loff[2 * line], o1 = loff[2 * line + 1];
                const bool has_y = lflag[line] != 0;
                if (o0 >= 0 || o1 >= 0)
                    fused_pro_line<M, true>(p, p.x + gl, p.bdiag + gl, gl, tile + line * LS, ce + line * t2, lane, has_y, o0, o1);
                else
                    fused_pro_line<M, false>(p, p.x + gl, p.bdiag + gl, gl, tile + line * LS, ce + line * t2, lane, has_y, o0, o1);
            }
        } else {
            for (int line = warp; line < nvalid; line += NW) {
                const cf* ul = p.u + g0 + (long long)line * M;
                cf* trow = tile + line * LS;
#pragma unroll
                for (int k = 0; k < EP2; ++k) {
                    const int q = 2 * lane + 64 * k;
                    if (M % 64 == 0 || q < M) {
                        const cf2 uv = ld2(ul + q);
                        trow[q] = uv.a;
                        trow[q + 1] = uv.b;
                    }
                }
            }
        }
        __syncthreads();
        // ---- FFT along the line (lanes across lines, as fft_contig_body) ----
        cf v[P];
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            v[m] = tile[c_ * LS + jt + m * T];
        });
        if constexpr (PL::NPASS > 1) __syncthreads();
        if constexpr (MODE == FUSED_S5) {
            static_for<0, P>([&](auto mc) { v[decltype(mc)::value] = cswap(v[decltype(mc)::value]); });
        }
        fft_line_forward<PL, 1, LS>(v, tile, c_, jt, tw);
        if constexpr (MODE == FUSED_1D) {
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = cswap(apply_symbol(v[m], p.sp.tab_axis[jt + m * T], p.sp));
            });
            fft_line_forward<PL, 1, LS>(v, tile, c_, jt, tw);
        }
        if constexpr (MODE != FUSED_S1) {
            static_for<0, P>([&](auto mc) { v[decltype(mc)::value] = cswap(v[decltype(mc)::value]); });
        }
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            tile[c_ * LS + jt + m * T] = v[m];
        });
        __syncthreads();
        if constexpr (MODE == FUSED_S1) {
            for (int line = warp; line < nvalid; line += NW) {
                cf* ul = p.u + g0 + (long long)line * M;
                const cf* trow = tile + line * LS;
#pragma unroll
                for (int k = 0; k < EP2; ++k) {
                    const int q = 2 * lane + 64 * k;
                    if (M % 64 == 0 || q < M) st2(ul + q, trow[q], trow[q + 1]);
                }
            }
        } else {
            // ---- epilogue: d = x - u'; r = B_diag d - corr(d); |r|^2; x -= alpha r ----
            if (p.a2) {
                for (int o = tid; o < nvalid * t2; o += NT) {
                    const int line = o / t2, e = o - line * t2;
                    const int q = (e < t ? e : M - t2 + e);
                    cf dv = csub(p.x[g0 + (long long)line * M + q], tile[line * LS + q]);
                    if (p.dref) dv = cadd(dv, p.dref[g0 + (long long)line * M + q]);
                    ed[o] = dv;
                }
                __syncthreads();
                fused_corr2<C>(ed, ce, Ks, t, p.S2, p.per2, p.c, nvalid, tid, NT);
                __syncthreads();
            }
            for (int line = warp; line < nvalid; line += NW) {
                const long long gl = g0 + (long long)line * M;
                const long long o0 = loff[2 * line], o1 = loff[2 * line + 1];
                if (o0 >= 0 || o1 >= 0)
                    fused_epi_line<M, true>(p, p.x + gl, p.bdiag + gl, gl, tile + line * LS, ce + line * t2, lane, o0, o1);
                else
                    acc += fused_epi_line<M, false>(p, p.x + gl, p.bdiag + gl, gl, tile + line * LS, ce + line * t2, lane, o0, o1);
            }
        }
    }
    if constexpr (MODE != FUSED_S1) {
        const double bs = block_sum((double)acc, red);
        grid_reduce_finish(bs, p.partials, p.slot0, p.n_total, p.finish, p.reduce_mode, p.state, p.hist, red);
    }
}

}  // namespace mbs
