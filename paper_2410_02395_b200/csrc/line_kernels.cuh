// line_kernels.cuh -- warp-line variant of the first and last sweep of one iteration of Eq. (6).
//
// The T <= 32 threads that own one line of the contiguous axis are lanes of a single warp.  Each warp loads its
// line(s) straight from global memory in the FFT's own register layout (thread jt holds points jt + m*T, so
// every load/store instruction of a warp is one contiguous run), applies the scattering operator on the fly,
// runs the FFT with warp-local exchanges through a private padded scratch line (__syncwarp only) and stores
// the result.  No block-level barrier exists inside the loop: the 16-24 resident warps of an SM drift apart and
// hide each other's HBM, shared-memory and pipeline latencies.
//
//   LINE_S1 : u = B_diag x + y_vec - corr_0(x) - corr_1(x) - corr_2(x), forward FFT         (a1, a2, a3)
//             corr_0, corr_1 come from the compact buffers of the slab kernel; corr_2 (wrap-around C_ss and
//             transfer A_{s,s+-1} along the line) is evaluated by the lanes that hold the 2t edge
//             points from the edge points of the own and the neighbouring line, read in place.
//   LINE_S5 : inverse FFT, d = x - u', r_part = B_diag d; every voxel outside all edge slabs is finished here
//             (|r|^2, x -= alpha r: a6-a9); at slab voxels (rows in a slab of axis 0/1, or one of the 2t edge
//             points of the line) it stores d to the compact buffers and r_part in place into u, and the
//             fix-up kernels (kernels.cu) complete them.
#pragma once
#include "fft_kernels.cuh"
#include "reduce.cuh"

namespace mbs {

// Plans with more than 16 points per thread (5 * 2^a and 3 * 2^a sizes) cannot hold u, x AND B_diag of a line in 128
// registers across the FFT of the last sweep: there B_diag of the line is requested with cp.async into a per-line stage
// in shared memory before the butterflies (no registers, no spills) and read back after them.
template <class PL, int MODE>
constexpr bool line_stage_b() { return MODE == LINE_S5 && PL::P > 16; }
template <class PL, int NWARP, int MODE = LINE_S1>
constexpr size_t line_smem_bytes(int t) {
    return sizeof(cf) * (size_t)(PL::M + NWARP * (32 / PL::T) * line_scratch_elems<PL>() +
                                 (line_stage_b<PL, MODE>() ? NWARP * 32 * PL::P + 2 : 0)) +
           sizeof(float) * (size_t)(t * t) + 16;
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void prefetch_l2(const void* gptr) { asm volatile("prefetch.global.L2 [%0];" ::"l"(gptr)); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ int line_edge_slot(int i, int M, int t) {   // as fused_edge_slot: s*2t + e, or -1
    const int s = i / M, e = i - s * M;
    if (e < t) return s * 2 * t + e;
    if (e >= M - t) return s * 2 * t + t + (e - (M - t));
    return -1;
}

// corr_2(x) at edge point `pidx` of line (row, seg): c * sum_q K (x_nb[q] - x_own[q])   (P:124-128 with P:106)
//   last  t points (a = pidx - (M-t)): K[a][q], own/nb = FIRST t points of this segment / of segment seg+1
//   first t points (b = pidx):         K[q][b], own/nb = LAST  t points of this segment / of segment seg-1
// TT > 0: t known at compile time (all 2t loads are issued before the first use); TT = 0: any t.
template <int M, int TT>
__device__ __forceinline__ cf line_corr2_x_t(const FusedParams& p, const float* Ks, const long long grow, const int seg,
                                             const int pidx) {
    const int t = TT > 0 ? TT : p.t;
    const bool last = pidx >= M - t;
    const int k = last ? pidx - (M - t) : pidx;
    int nb = last ? seg + 1 : seg - 1;
    bool has_nb = true;
    if (nb < 0 || nb >= p.S2) {
        if (p.per2) nb = (nb + p.S2) % p.S2;
        else has_nb = false;
    }
    const cf* own = p.x + grow + (long long)seg * M + (last ? 0 : M - t);
    const cf* nbp = p.x + grow + (long long)nb * M + (last ? 0 : M - t);
    float sr = 0.f, si = 0.f;
    if constexpr (TT > 0) {
        cf ov[TT], nv[TT];
#pragma unroll
        for (int q = 0; q < TT; ++q) {
            ov[q] = own[q];
            nv[q] = has_nb ? nbp[q] : make_float2(0.f, 0.f);
        }
#pragma unroll
        for (int q = 0; q < TT; ++q) {
            const float kk = last ? Ks[k * TT + q] : Ks[q * TT + k];
            sr = fmaf(kk, nv[q].x - ov[q].x, sr);
            si = fmaf(kk, nv[q].y - ov[q].y, si);
        }
    } else {
        for (int q = 0; q < t; ++q) {
            const float kk = last ? Ks[k * t + q] : Ks[q * t + k];
            cf dv = own[q];
            dv = make_float2(-dv.x, -dv.y);
            if (has_nb) {
                const cf nv = nbp[q];
                dv = make_float2(nv.x + dv.x, nv.y + dv.y);
            }
            sr = fmaf(kk, dv.x, sr);
            si = fmaf(kk, dv.y, si);
        }
    }
    return cmul(p.c, make_float2(sr, si));
}

template <int M>
__device__ __forceinline__ cf line_corr2_x(const FusedParams& p, const float* Ks, const long long grow, const int seg,
                                           const int pidx) {
    if (p.t == 8) return line_corr2_x_t<M, 8>(p, Ks, grow, seg, pidx);   // the paper's default
    if (p.t == 4) return line_corr2_x_t<M, 4>(p, Ks, grow, seg, pidx);
    return line_corr2_x_t<M, 0>(p, Ks, grow, seg, pidx);
}

__device__ __forceinline__ int line_edge_index(int q, int M, int t) {   // q in [0, S*2t) -> index along the axis
    const int s = q / (2 * t), e = q - s * 2 * t;
    return s * M + (e < t ? e : M - 2 * t + e);
}

// ACT: subdomain activation -- lines of inactive subdomains are skipped; a separate instantiation so that
// the plain kernels keep their code exactly
template <class PL, int NWARP, int MODE, bool ACT = false>
__device__ __forceinline__ void line_body(const FusedParams& p, const cf* __restrict__ tw_global, cf* smem, double* red) {
    constexpr int M = PL::M, P = PL::P, T = PL::T, NT = NWARP * 32;
    static_assert(T <= 32 && 32 % T == 0, "a line must fit in one warp");
    constexpr int LW = 32 / T;                        // lines per warp
    constexpr int LSE = line_scratch_elems<PL>();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int t = p.t, t2 = 2 * p.t;
    cf* tw = smem;
    cf* scratch = tw + M + (warp * LW + lane / T) * LSE;
    constexpr bool STAGE_B = line_stage_b<PL, MODE>();
    constexpr int BST0 = (M + NWARP * LW * LSE + 1) & ~1;              // 16-byte aligned start of the B_diag stages
    cf* bst = tw + BST0 + (warp * LW + lane / T) * M;                  // this line's stage (STAGE_B only)
    float* Ks = reinterpret_cast<float*>(tw + (STAGE_B ? BST0 + NWARP * LW * M : M + NWARP * LW * LSE));
    fill_warp_twiddles<PL>(tw, tw_global, tid, NT);   // per-pass [r][k] layout: conflict-free for lanes along a line
    if (p.a2) for (int i = tid; i < t * t; i += NT) Ks[i] = p.Kh[i];
    __syncthreads();
    const int jt = lane % T, lsub = lane / T;
    const unsigned n_lines = (unsigned)p.n_lines;
    const unsigned n_units = (n_lines + LW - 1) / LW;
    float acc = 0.f;
    for (unsigned unit = blockIdx.x * NWARP + warp; unit < n_units; unit += gridDim.x * NWARP) {
        unsigned line = unit * LW + lsub;
        const bool in_range = line < n_lines;
        unsigned row = line / (unsigned)p.S2;
        const int seg = (int)(line - row * (unsigned)p.S2);
        const int i0 = (int)(row / (unsigned)p.N1), i1 = (int)(row - (unsigned)i0 * (unsigned)p.N1);
        bool act_ok = true;
        if constexpr (ACT) {
            if (p.active) {
                // the lines of an inactive subdomain are not computed
                act_ok = in_range && p.active[((i0 / p.M0) * p.S1 + i1 / p.M1) * p.S2 + seg] != 0;
                if (!__any_sync(0xffffffffu, act_ok)) continue;
            }
        }
        const bool valid = in_range && act_ok;
        long long o0b = -1, o1b = -1;                 // compact row offsets of the axis-0 / axis-1 slabs
        if (valid && p.e0) {
            const int q = line_edge_slot(i0, p.M0, t);
            if (q >= 0) o0b = ((long long)q * p.N1 + i1) * p.N2 + (long long)seg * M;
        }
        if (valid && p.e1) {
            const int q = line_edge_slot(i1, p.M1, t);
            if (q >= 0) o1b = ((long long)i0 * (p.S1 * t2) + q) * p.N2 + (long long)seg * M;
        }
        const long long gl0 = (long long)line * M;    // offset of the line in B_diag (shared by the sources of a batch)
        // batched solves (R18; the ACT instantiations only): the sources of a batch one after the other on the same
        // line, so that B_diag of the line is read from DRAM once (the later reads hit L1 / L2)
        const int n_batch = ACT ? (p.n_batch > 1 ? p.n_batch : 1) : 1;
        for (int bsrc = 0; bsrc < n_batch; ++bsrc) {
        const long long boff = ACT ? bsrc * p.batch_stride : 0;
        const long long gl = gl0 + boff;              // offset of the line in x, y, u of this source
        const long long grow = (long long)row * p.N2 + boff;
        const long long o0 = (ACT && o0b >= 0) ? o0b + bsrc * p.cstride[0] : o0b;
        const long long o1 = (ACT && o1b >= 0) ? o1b + bsrc * p.cstride[1] : o1b;
        const long long mrow = (long long)row + (ACT ? bsrc * p.mask_stride : 0);
        cf v[P];
        if constexpr (MODE == LINE_S1) {
            const bool has_y = valid && p.y != nullptr && (p.ymask == nullptr || p.ymask[mrow] != 0);
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                const int pidx = jt + m * T;
                v[m] = valid ? cmul(p.bdiag[gl0 + pidx], p.x[gl + pidx]) : make_float2(0.f, 0.f);
            });
            if (has_y) {
                static_for<0, P>([&](auto mc) {
                    constexpr int m = decltype(mc)::value;
                    v[m] = cadd(v[m], cmul(p.ysc, p.y[gl + jt + m * T]));
                });
            }
            if (o0 >= 0) {
                static_for<0, P>([&](auto mc) {
                    constexpr int m = decltype(mc)::value;
                    v[m] = csub(v[m], p.cx0[o0 + jt + m * T]);
                });
            }
            if (o1 >= 0) {
                static_for<0, P>([&](auto mc) {
                    constexpr int m = decltype(mc)::value;
                    v[m] = csub(v[m], p.cx1[o1 + jt + m * T]);
                });
            }
            if (p.a2 && valid) {
                static_for<0, P>([&](auto mc) {
                    constexpr int m = decltype(mc)::value;
                    const int pidx = jt + m * T;
                    if (pidx < t || pidx >= M - t) v[m] = csub(v[m], line_corr2_x<M>(p, Ks, grow, seg, pidx));
                });
            }
#ifndef MBS_NO_L2_PREFETCH
            // x and B_diag of the line this warp takes next are requested into L2 now (one 128-byte line per lane and
            // request: no registers, no shared memory), so that their loads after this FFT are L2 hits
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
                static_for<0, P>([&](auto mc) {
                    constexpr int m = decltype(mc)::value;
                    p.u[gl + jt + m * T] = v[m];
                });
            }
        } else {
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = valid ? cswap(p.u[gl + jt + m * T]) : make_float2(0.f, 0.f);
            });
            // x and B_diag of the line are requested before the butterflies, so their HBM latency is covered
            constexpr bool PREFETCH_B = !STAGE_B;
            if constexpr (STAGE_B) {
                __syncwarp();                                          // the stage is no longer read by the unit before
                if (valid) {
                    const cf* src = p.bdiag + gl0;
#pragma unroll
                    for (int i = 0; i < P / 2; ++i) cp_async16(bst + 2 * (jt + i * T), src + 2 * (jt + i * T));
                }
                cp_async_commit();
            }
            cf xr[P], br[PREFETCH_B ? P : 1];
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                xr[m] = valid ? p.x[gl + jt + m * T] : make_float2(0.f, 0.f);
                if constexpr (PREFETCH_B) br[m] = valid ? p.bdiag[gl0 + jt + m * T] : make_float2(0.f, 0.f);
            });
            fft_line_forward_warp<PL>(v, scratch, jt, tw);
            if constexpr (STAGE_B) {
                cp_async_wait_all();
                __syncwarp();                                          // every lane's copies have landed
            }
            if (valid) {
                const bool slab_row = (o0 >= 0) || (o1 >= 0);
                const long long o2 = (long long)row * (p.S2 * t2) + (long long)seg * t2 + (ACT ? bsrc * p.cstride[2] : 0);
                static_for<0, P>([&](auto mc) {
                    constexpr int m = decltype(mc)::value;
                    const int pidx = jt + m * T;
                    const cf xv = xr[m];
                    cf d = csub(xv, cswap(v[m]));
                    if (p.dref) d = cadd(d, p.dref[gl + pidx]);        // split iterate: d = d_ref + (delta - u')
                    cf bv;
                    if constexpr (PREFETCH_B) bv = br[m];
                    else bv = bst[pidx];
                    cf r = cmul(bv, d);
                    if (p.rref) r = cadd(r, p.rref[gl + pidx]);        // split iterate, complex128 residual: r = r_ref + B (delta - u')
                    const bool edge2 = p.a2 && (pidx < t || pidx >= M - t);
                    if (!slab_row && !edge2) {
                        acc += r.x * r.x + r.y * r.y;
                        p.x[gl + pidx] = make_float2(xv.x - p.alpha * r.x, xv.y - p.alpha * r.y);
                    } else {
                        if (o0 >= 0) p.ds0[o0 + pidx] = d;
                        if (o1 >= 0) p.ds1[o1 + pidx] = d;
                        if (edge2) p.ds2[o2 + (pidx < t ? pidx : pidx - (M - t2))] = d;
                        p.u[gl + pidx] = r;
                    }
                });
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
