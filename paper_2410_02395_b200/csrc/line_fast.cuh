// line_fast.cuh -- the warp-line first / last sweep (line_kernels.cuh) with the number of correction points known at
// compile time (TT = t = 8, the paper's default) and TT <= T.
//
// Same arithmetic, same order, same results as line_body; what changes is the instruction count.  In line_body every
// one of the P points of a thread asks "am I one of the 2t edge points of the line?" with a run-time t: P x (two
// compares, a predicate, a divergence region) at each of the places that treat edge points differently, about a third
// of the 75 thread-instructions per voxel ncu counts for those sweeps (profiles/r02_line_kernels.md).  With TT <= T the
// edge points of a line are exactly
//     point m = 0     of the lanes jt < TT        (the first TT points), and
//     point m = P - 1 of the lanes jt >= T - TT   (the last TT points),
// so the edge work is written once, outside the loops over m, and the loops themselves are branch-free.  A line past
// the end of the grid (ragged last unit) is clamped to the last line for its loads and masked at its stores, instead of
// predicating every access.
#pragma once
#include "line_kernels.cuh"

namespace mbs {

template <class PL, int TT>
constexpr bool line_fast_ok() { return PL::T >= TT && PL::T <= 32 && 32 % PL::T == 0; }

// corr_2(x) of the edge point this lane holds (P:124-128 with P:106), as line_corr2_x_t, for a lane that is known to
// hold one: `last` selects the last-TT / first-TT formulas, k is the index within the edge.
template <int M, int TT>
__device__ __forceinline__ cf fast_corr2_x(const FusedParams& p, const float* Ks, const long long grow, const int seg,
                                           const bool last, const int k) {
    int nb = last ? seg + 1 : seg - 1;
    bool has_nb = true;
    if (nb < 0 || nb >= p.S2) {
        if (p.per2) nb = (nb + p.S2) % p.S2;
        else has_nb = false;
    }
    const cf* own = p.x + grow + (long long)seg * M + (last ? 0 : M - TT);
    const cf* nbp = p.x + grow + (long long)nb * M + (last ? 0 : M - TT);
    // four points at a time: the 2 x 4 loads of a group are in flight together, and only 8 values are live at once
    // (the first sweep runs at 80 registers per thread with the 16 points of the line in registers)
    constexpr int G = TT >= 4 ? 4 : TT;
    float sr = 0.f, si = 0.f;
#pragma unroll
    for (int q0 = 0; q0 < TT; q0 += G) {
        cf ov[G], nv[G];
#pragma unroll
        for (int q = 0; q < G; ++q) {
            ov[q] = own[q0 + q];
            nv[q] = has_nb ? nbp[q0 + q] : make_float2(0.f, 0.f);
        }
#pragma unroll
        for (int q = 0; q < G; ++q) {
            const float kk = last ? Ks[k * TT + q0 + q] : Ks[(q0 + q) * TT + k];
            sr = fmaf(kk, nv[q].x - ov[q].x, sr);
            si = fmaf(kk, nv[q].y - ov[q].y, si);
        }
    }
    return cmul(p.c, make_float2(sr, si));
}

template <class PL, int NWARP, int MODE, bool ACT, int TT>
__device__ __forceinline__ void line_body_fast(const FusedParams& p, const cf* __restrict__ tw_global, cf* smem, double* red) {
    constexpr int M = PL::M, P = PL::P, T = PL::T, NT = NWARP * 32;
    static_assert(line_fast_ok<PL, TT>(), "fast warp-line sweep: TT <= T <= 32");
    static_assert(!line_stage_b<PL, MODE>(), "plans with more than 16 points per thread use line_body");
    constexpr int LW = 32 / T;
    constexpr int LSE = line_scratch_elems<PL>();
    constexpr int t2 = 2 * TT;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    cf* tw = smem;
    cf* scratch = tw + M + (warp * LW + lane / T) * LSE;
    float* Ks = reinterpret_cast<float*>(tw + M + NWARP * LW * LSE);
    fill_warp_twiddles<PL>(tw, tw_global, tid, NT);
    if (p.a2) for (int i = tid; i < TT * TT; i += NT) Ks[i] = p.Kh[i];
    __syncthreads();
    const int jt = lane % T, lsub = lane / T;
    const unsigned n_lines = (unsigned)p.n_lines;
    const unsigned n_units = (n_lines + LW - 1) / LW;
    const bool first_edge = p.a2 && jt < TT;          // this lane's point m = 0 is one of the first TT points
    const bool last_edge = p.a2 && jt >= T - TT;      // this lane's point m = P-1 is one of the last TT points
    const int k_last = jt - (T - TT);
    float acc = 0.f;
    for (unsigned unit = blockIdx.x * NWARP + warp; unit < n_units; unit += gridDim.x * NWARP) {
        unsigned line = unit * LW + lsub;
        const bool in_range = line < n_lines;
        if (!in_range) line = n_lines - 1;            // clamp: loads stay legal, stores are masked
        unsigned row = line / (unsigned)p.S2;
        const int seg = (int)(line - row * (unsigned)p.S2);
        const int i0 = (int)(row / (unsigned)p.N1), i1 = (int)(row - (unsigned)i0 * (unsigned)p.N1);
        bool valid = in_range;
        if constexpr (ACT) {
            if (p.active) {
                valid = valid && p.active[((i0 / p.M0) * p.S1 + i1 / p.M1) * p.S2 + seg] != 0;
                if (!__any_sync(0xffffffffu, valid)) continue;
            }
        }
        long long o0b = -1, o1b = -1;                 // compact row offsets of the axis-0 / axis-1 slabs
        if (p.e0) {
            const int q = line_edge_slot(i0, p.M0, TT);
            if (q >= 0) o0b = ((long long)q * p.N1 + i1) * p.N2 + (long long)seg * M;
        }
        if (p.e1) {
            const int q = line_edge_slot(i1, p.M1, TT);
            if (q >= 0) o1b = ((long long)i0 * (p.S1 * t2) + q) * p.N2 + (long long)seg * M;
        }
        const long long gl0 = (long long)line * M + jt;   // this lane's first point in B_diag (shared by the sources of a batch)
        // batched solves (R18; the ACT instantiations only): the sources one after the other on the same line
        const int n_batch = ACT ? (p.n_batch > 1 ? p.n_batch : 1) : 1;
        for (int bsrc = 0; bsrc < n_batch; ++bsrc) {
        const long long boff = ACT ? bsrc * p.batch_stride : 0;
        const long long gl = gl0 + boff;                  // ... and in x, y, u of this source
        const long long grow = (long long)row * p.N2 + boff;
        const long long o0 = (ACT && o0b >= 0) ? o0b + bsrc * p.cstride[0] : o0b;
        const long long o1 = (ACT && o1b >= 0) ? o1b + bsrc * p.cstride[1] : o1b;
        const long long mrow = (long long)row + (ACT ? bsrc * p.mask_stride : 0);
        cf v[P];
        if constexpr (MODE == LINE_S1) {
            const cf* xb = p.x + gl;
            const cf* bb = p.bdiag + gl0;
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = cmul(bb[m * T], xb[m * T]);
            });
            if (p.y != nullptr && (p.ymask == nullptr || p.ymask[mrow] != 0)) {
                const cf* yb = p.y + gl;
                static_for<0, P>([&](auto mc) {
                    constexpr int m = decltype(mc)::value;
                    v[m] = cadd(v[m], cmul(p.ysc, yb[m * T]));
                });
            }
            if (o0 >= 0) {
                const cf* cb = p.cx0 + o0 + jt;
                static_for<0, P>([&](auto mc) {
                    constexpr int m = decltype(mc)::value;
                    v[m] = csub(v[m], cb[m * T]);
                });
            }
            if (o1 >= 0) {
                const cf* cb = p.cx1 + o1 + jt;
                static_for<0, P>([&](auto mc) {
                    constexpr int m = decltype(mc)::value;
                    v[m] = csub(v[m], cb[m * T]);
                });
            }
            if constexpr (T >= 2 * TT) {
                // a lane holds at most one edge point: one pass for the first-edge and the last-edge lanes together
                if (first_edge || last_edge) {
                    const cf corr = fast_corr2_x<M, TT>(p, Ks, grow, seg, last_edge, last_edge ? k_last : jt);
                    if (last_edge) v[P - 1] = csub(v[P - 1], corr);
                    else v[0] = csub(v[0], corr);
                }
            } else {
                if (first_edge) v[0] = csub(v[0], fast_corr2_x<M, TT>(p, Ks, grow, seg, false, jt));
                if (last_edge) v[P - 1] = csub(v[P - 1], fast_corr2_x<M, TT>(p, Ks, grow, seg, true, k_last));
            }
#ifndef MBS_NO_L2_PREFETCH
            {
                const unsigned nline = (unit + gridDim.x * NWARP) * LW + lsub;
                bool want = nline < n_lines;
                if constexpr (ACT) {
                    if (want && p.active) {
                        const unsigned nrow = nline / (unsigned)p.S2;
                        const int ni0 = (int)(nrow / (unsigned)p.N1), ni1 = (int)(nrow - (unsigned)ni0 * (unsigned)p.N1);
                        want = p.active[((ni0 / p.M0) * p.S1 + ni1 / p.M1) * p.S2 + (int)(nline - nrow * (unsigned)p.S2)] != 0;
                    }
                }
                if (want) {
                    const char* nx = reinterpret_cast<const char*>(p.x + (long long)nline * M);
                    const char* nb = reinterpret_cast<const char*>(p.bdiag + (long long)nline * M);
                    for (int off = jt * 128; off < M * (int)sizeof(cf); off += T * 128) {
                        prefetch_l2(nx + off);
                        prefetch_l2(nb + off);
                    }
                }
            }
#endif
            fft_line_forward_warp<PL>(v, scratch, jt, tw);
            if (valid) {
                cf* ub = p.u + gl;
                static_for<0, P>([&](auto mc) {
                    constexpr int m = decltype(mc)::value;
                    ub[m * T] = v[m];
                });
            }
        } else {
            const cf* ub = p.u + gl;
            const cf* xb = p.x + gl;
            const cf* bb = p.bdiag + gl0;
            cf xr[P], br[P];
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = cswap(ub[m * T]);
            });
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                xr[m] = xb[m * T];
                br[m] = bb[m * T];
            });
            fft_line_forward_warp<PL>(v, scratch, jt, tw);
            // d = x - u' (+ d_ref of the split iterate); r = B_diag d
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = csub(xr[m], cswap(v[m]));
            });
            if (p.dref) {
                const cf* db = p.dref + gl;
                static_for<0, P>([&](auto mc) {
                    constexpr int m = decltype(mc)::value;
                    v[m] = cadd(v[m], db[m * T]);
                });
            }
            if (valid) {
                cf* xo = p.x + gl;
                cf* uo = p.u + gl;
                if ((o0 >= 0) || (o1 >= 0)) {
                    // a row in a slab of axis 0 / 1: d to the compact buffers, r_part in place in u; the slab passes finish it
                    static_for<0, P>([&](auto mc) {
                        constexpr int m = decltype(mc)::value;
                        cf r = cmul(br[m], v[m]);
                        if (p.rref) r = cadd(r, p.rref[gl + m * T]);   // split iterate, complex128 residual
                        uo[m * T] = r;
                    });
                    if (o0 >= 0) {
                        cf* db = p.ds0 + o0 + jt;
                        static_for<0, P>([&](auto mc) { db[decltype(mc)::value * T] = v[decltype(mc)::value]; });
                    }
                    if (o1 >= 0) {
                        cf* db = p.ds1 + o1 + jt;
                        static_for<0, P>([&](auto mc) { db[decltype(mc)::value * T] = v[decltype(mc)::value]; });
                    }
                } else {
                    // every point that is not one of the 2 TT edge points of the line is finished here (a7-a9)
                    static_for<0, P>([&](auto mc) {
                        constexpr int m = decltype(mc)::value;
                        cf r = cmul(br[m], v[m]);
                        if (p.rref) r = cadd(r, p.rref[gl + m * T]);   // split iterate, complex128 residual
                        bool edge = false;
                        if constexpr (m == 0) edge = first_edge;
                        if constexpr (m == P - 1) edge = edge || last_edge;
                        if (!edge) {
                            acc += r.x * r.x + r.y * r.y;
                            xo[m * T] = make_float2(xr[m].x - p.alpha * r.x, xr[m].y - p.alpha * r.y);
                        } else {
                            uo[m * T] = r;
                        }
                    });
                }
                // d at the edge points of the line, for corr_2(d) in the slab pass of the last axis
                if (first_edge || last_edge) {
                    cf* d2 = p.ds2 + (long long)row * (p.S2 * t2) + (long long)seg * t2 + (ACT ? bsrc * p.cstride[2] : 0);
                    if (first_edge) d2[jt] = v[0];
                    if (last_edge) d2[TT + k_last] = v[P - 1];
                }
            }
        }
        }   // sources of the batch
    }
    if constexpr (MODE == LINE_S5) {
        const double bs = block_sum((double)acc, red);
        grid_reduce_finish(bs, p.partials, p.slot0, p.n_total, p.finish, p.reduce_mode, p.state, p.hist, red);
    }
}

}  // namespace mbs
