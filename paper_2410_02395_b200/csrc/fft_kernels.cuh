// fft_kernels.cuh -- tile kernels that run the per-subdomain FFTs of the propagator (L+I)^-1
// (forward FFT, multiply by 1/(c(k0^2-|p|^2)+1), inverse FFT, per subdomain).
//
// Two tile shapes, one register/shared-memory core (fft_core.cuh):
//   * strided axis (any axis but the last): tile = M points along the axis x C contiguous voxels.
//     Lanes run along the contiguous direction (128-byte segments for C = 16); the first pass
//     loads straight from global memory into registers and the last pass stores straight back.
//   * contiguous (last) axis: tile = C consecutive lines of M contiguous voxels, staged through a
//     padded transposed shared-memory tile so global accesses stay coalesced along the line while
//     the core still runs with lanes across lines (bank-conflict free: line stride M+1 is odd).
// MODE: forward, inverse (swap trick: ifft(z) = swap(fft(swap(z)))), or "mid" = forward, multiply
// by the Fourier-space kernel, inverse, all in one sweep (the axis transformed last/first).
#pragma once
#include "fft_core.cuh"

namespace mbs {

enum FftMode { FFT_FWD = 0, FFT_INV = 1, FFT_MID = 2 };

// Fourier-space symbol of L+I on one subdomain: D(p) = c (k0^2 - |p|^2) + 1 (Eq. (5)),
//   Re D = A0 - cr*|p|^2,  Im D = B0 - ci*|p|^2,  A0 = Re(c k0^2) + 1, B0 = Im(c k0^2).
// inverse != 0: multiply by scale / D (the propagator); else by scale * D (operator L+I).
struct SymbolParams {
    float A0, B0, cr, ci, scale;
    int inverse;
    const float* tab_axis;   // p_d^2 along the transformed axis, length M
    const float* tabA;       // p^2 table of the slower inner axis (period Ma), or nullptr
    const float* tabB;       // p^2 table of the faster inner axis (period Mb), or nullptr
    int Nb, Ma, Mb;          // inner index ii -> (ii / Nb) % Ma, (ii % Nb) % Mb
    const float* wtab;       // optional: tabA[..] + tabB[..] tabulated per inner index ii (replaces the two lookups)
};

MBS_HD cf apply_symbol(cf v, float p2, const SymbolParams& sp) {
    const float dre = sp.A0 - sp.cr * p2;
    const float dim = sp.B0 - sp.ci * p2;
    if (sp.inverse) {
#ifdef __CUDA_ARCH__
        const float inv = __fdividef(sp.scale, dre * dre + dim * dim);   // 2 ulp; the bar is 1e-5 per operator
#else
        const float inv = sp.scale / (dre * dre + dim * dim);
#endif
        const cf g = make_float2(dre * inv, -dim * inv);
        return cmul(v, g);
    } else {
        const cf g = make_float2(dre * sp.scale, dim * sp.scale);
        return cmul(v, g);
    }
}

struct StridedGeom {
    long long outer_stride;  // elements between consecutive outer indices
    long long stride;        // elements between consecutive points along the axis
    int n_outer;             // product of the axes before the transformed one
    int n_seg;               // S_d subdomains along the axis
    int inner;               // contiguous extent (product of the axes after)
    int tiles_inner;         // ceil(inner / C)
    long long n_tiles;       // n_outer * n_seg * tiles_inner
    // subdomain activation: when act_list != nullptr the sweep visits only the tiles of the *n_act
    // subdomains listed there (index (s0*S1 + s1)*S2 + s2); tile k of a listed subdomain, k in [0, tiles_per_sub):
    //   sweep along axis 1:  outer = s0*M0 + k / tps2,              segment = s1, inner tile = s2*tps2 + k % tps2
    //   sweep along axis 0:  segment = s0, i1 = s1*M1 + k / tps2,   inner tile = i1*(N2/C) + s2*tps2 + k % tps2
    // with tps2 = M2 / C tiles per subdomain row (the host enables this only when C divides M2).
    const int* act_list;
    const int* n_act;
    int axis;                // 0 or 1: the transformed axis in the internal 3-D description
    int tiles_per_sub, tps2;
    int S1, S2, M0, M1;      // subdomain counts of axes 1, 2; subdomain lengths of axes 0, 1
    int row_tiles;           // N2 / C
};

// tile index -> (outer index, segment along the axis, inner tile) of a strided sweep
MBS_HD void strided_tile_decode(const StridedGeom& g, const unsigned tix, unsigned& o, unsigned& seg, unsigned& ic) {
    if (g.act_list) {
        const unsigned u = tix / (unsigned)g.tiles_per_sub, k = tix - u * (unsigned)g.tiles_per_sub;
        const unsigned sub = (unsigned)g.act_list[u];
        const unsigned s2 = sub % (unsigned)g.S2, s01 = sub / (unsigned)g.S2;
        const unsigned s1 = s01 % (unsigned)g.S1, s0 = s01 / (unsigned)g.S1;
        const unsigned kr = k / (unsigned)g.tps2, kc = k - kr * (unsigned)g.tps2;
        if (g.axis == 1) {
            o = s0 * (unsigned)g.M0 + kr;
            seg = s1;
            ic = s2 * (unsigned)g.tps2 + kc;
        } else {
            o = 0;
            seg = s0;
            ic = (s1 * (unsigned)g.M1 + kr) * (unsigned)g.row_tiles + s2 * (unsigned)g.tps2 + kc;
        }
    } else {
        const unsigned os = tix / (unsigned)g.tiles_inner;
        ic = tix - os * (unsigned)g.tiles_inner;
        o = os / (unsigned)g.n_seg;
        seg = os - o * (unsigned)g.n_seg;
    }
}

template <class PL, int C, int MODE>
MBS_DEV void fft_strided_body(cf* MBS_RESTRICT data, const StridedGeom g, const SymbolParams sp,
                              const cf* MBS_RESTRICT tw_global, const int tid, const int bid,
                              const int nblocks, cf* smem) {
    constexpr int M = PL::M, P = PL::P, T = PL::T, NT = T * C;
    cf* tw = smem;
    cf* tile = smem + M;
    for (int i = tid; i < M; i += NT) tw[i] = tw_global[i];
    MBS_SYNC();
    const int c = tid % C;
    const int jt = tid / C;
    const long long n_tiles = g.act_list ? (long long)*g.n_act * g.tiles_per_sub : g.n_tiles;
    for (long long tix = bid; tix < n_tiles; tix += nblocks) {
        unsigned o_u, s_u, ic_u;
        strided_tile_decode(g, (unsigned)tix, o_u, s_u, ic_u);
        const int ic = (int)ic_u, s = (int)s_u;
        const long long o = (long long)o_u;
        const int ii = ic * C + c;
        const bool valid = ii < g.inner;
        cf* base = data + o * g.outer_stride + (long long)s * M * g.stride + ii;
        cf v[P];
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            v[m] = valid ? base[(long long)(jt + m * T) * g.stride] : make_float2(0.f, 0.f);
        });
        if constexpr (MODE == FFT_INV) {
            static_for<0, P>([&](auto mc) { v[decltype(mc)::value] = cswap(v[decltype(mc)::value]); });
        }
        fft_line_forward<PL, C, 1>(v, tile, c, jt, tw);
        if constexpr (MODE == FFT_MID) {
            float wline = 0.f;
            if (sp.tabA) wline += sp.tabA[(ii / sp.Nb) % sp.Ma];
            if (sp.tabB) wline += sp.tabB[(ii % sp.Nb) % sp.Mb];
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                const float p2 = sp.tab_axis[jt + m * T] + wline;
                v[m] = cswap(apply_symbol(v[m], p2, sp));
            });
            fft_line_forward<PL, C, 1>(v, tile, c, jt, tw);
        }
        if constexpr (MODE != FFT_FWD) {
            static_for<0, P>([&](auto mc) { v[decltype(mc)::value] = cswap(v[decltype(mc)::value]); });
        }
        if (valid) {
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                base[(long long)(jt + m * T) * g.stride] = v[m];
            });
        }
    }
}

struct ContigGeom {
    long long n_lines;   // voxels / M
    long long n_tiles;   // ceil(n_lines / C)
};

template <class PL, int C>
constexpr int contig_smem_elems() { return PL::M + C * (PL::M + 1); }
template <class PL, int C>
constexpr int strided_smem_elems() { return PL::M + (PL::NPASS > 1 ? C * PL::M : 0); }

template <class PL, int C, int MODE>
MBS_DEV void fft_contig_body(const cf* src, cf* dst, const ContigGeom g,
                             const SymbolParams sp, const cf* MBS_RESTRICT tw_global, const int tid,
                             const int bid, const int nblocks, cf* smem) {
    constexpr int M = PL::M, P = PL::P, T = PL::T, NT = T * C, LS = M + 1;
    cf* tw = smem;
    cf* tile = smem + M;
    for (int i = tid; i < M; i += NT) tw[i] = tw_global[i];
    const int c = tid % C;
    const int jt = tid / C;
    for (long long tix = bid; tix < g.n_tiles; tix += nblocks) {
        const long long line0 = tix * C;
        const int nvalid = (int)((g.n_lines - line0) < C ? (g.n_lines - line0) : C);
        const cf* in = src + line0 * M;
        MBS_SYNC();   // previous tile's store phase (and the twiddle load) is complete
        for (int idx = tid; idx < nvalid * M; idx += NT) {
            const int line = idx / M, p = idx - line * M;
            tile[line * LS + p] = in[idx];
        }
        MBS_SYNC();
        cf v[P];
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            v[m] = tile[c * LS + jt + m * T];
        });
        if constexpr (PL::NPASS > 1) MBS_SYNC();
        if constexpr (MODE == FFT_INV) {
            static_for<0, P>([&](auto mc) { v[decltype(mc)::value] = cswap(v[decltype(mc)::value]); });
        }
        fft_line_forward<PL, 1, LS>(v, tile, c, jt, tw);
        if constexpr (MODE == FFT_MID) {
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = cswap(apply_symbol(v[m], sp.tab_axis[jt + m * T], sp));
            });
            fft_line_forward<PL, 1, LS>(v, tile, c, jt, tw);
        }
        if constexpr (MODE != FFT_FWD) {
            static_for<0, P>([&](auto mc) { v[decltype(mc)::value] = cswap(v[decltype(mc)::value]); });
        }
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            tile[c * LS + jt + m * T] = v[m];
        });
        MBS_SYNC();
        cf* out = dst + line0 * M;
        for (int idx = tid; idx < nvalid * M; idx += NT) {
            const int line = idx / M, p = idx - line * M;
            out[idx] = tile[line * LS + p];
        }
    }
}

}  // namespace mbs
