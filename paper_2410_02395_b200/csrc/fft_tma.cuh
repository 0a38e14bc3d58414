// fft_tma.cuh -- strided-axis FFT sweep fed by TMA (sm_100a; device only).
//
// Same transform as fft_strided_body (fft_kernels.cuh): a tile is M points along the transformed axis x
// C contiguous voxels.  Here the tile is moved by the Tensor Memory Accelerator instead of by the
// threads: one `cp.async.bulk.tensor` box load per (at most 256-row) half of the tile lands it in a
// shared-memory stage and signals an mbarrier; after the in-place FFT passes the threads write the result
// back to the same stage and one elected thread issues the bulk tensor store.  A CTA is persistent and
// cycles through NSTAGE stages, so the load of tile i+1 and the store of tile i-1 overlap the butterflies of
// tile i without costing registers or issue slots for address arithmetic.
//
// The tensor map views the array as [outer][N_axis][inner] float32 pairs (dims {2*inner, N_axis, outer}),
// box {2*C, M / NBOX, 1}; a ragged inner tail is zero-filled on load and clipped on store by the hardware.
#pragma once
#include <cuda.h>

#include "fft_kernels.cuh"

namespace mbs {

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, unsigned long long* bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* map, const void* src, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(map),
                 "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void tma_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void tma_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// a tile is moved as NBOX boxes of M / NBOX <= 256 rows (TMA box dimensions are limited to 256)
constexpr int tma_nbox_of(int M) {
    int nb = 1;
    while (M % nb != 0 || M / nb > 256) ++nb;
    return nb;
}
template <class PL, int C>
constexpr int tma_nbox() { return tma_nbox_of(PL::M); }
template <class PL, int C, int NSTAGE>
constexpr size_t tma_smem_bytes() { return (size_t)NSTAGE * PL::M * C * sizeof(cf) + PL::M * sizeof(cf) + NSTAGE * 8 + 64; }

template <class PL, int C, int MODE, int NSTAGE>
__device__ __forceinline__ void fft_strided_tma_body(const CUtensorMap* map, const StridedGeom g, const SymbolParams sp,
                                                     const cf* __restrict__ tw_global, cf* smem_raw) {
    constexpr int M = PL::M, P = PL::P, T = PL::T, NT = T * C;
    constexpr int NBOX = tma_nbox<PL, C>(), MB = M / NBOX;
    static_assert(M % NBOX == 0 && MB <= 256 && 2 * C <= 256, "TMA box limits");
    constexpr unsigned TILE_BYTES = M * C * sizeof(cf);
    // stage buffers (128-byte aligned: the dynamic shared memory is declared __align__(128)), then the
    // twiddle table, then the mbarriers
    cf* stage0 = reinterpret_cast<cf*>(smem_raw);
    cf* tw = stage0 + (size_t)NSTAGE * M * C;
    unsigned long long* full = reinterpret_cast<unsigned long long*>(tw + M);
    const int tid = threadIdx.x;
    if (tid == 0 && (smem_u32(smem_raw) & 127u) != 0) __trap();
    for (int i = tid; i < M; i += NT) tw[i] = tw_global[i];
    if (tid == 0) {
        for (int s = 0; s < NSTAGE; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_async_smem();
    }
    __syncthreads();
    const int c = tid % C;
    const int jt = tid / C;
    // tile counters fit 32 bits (fewer than 2^31 voxels): keep the per-tile index arithmetic cheap
    const unsigned first = blockIdx.x, step = gridDim.x;
    // with subdomain activation the sweep covers the listed subdomains only (the count lives in device memory)
    const unsigned n_tiles = g.act_list ? (unsigned)*g.n_act * (unsigned)g.tiles_per_sub : (unsigned)g.n_tiles;
    const unsigned n_mine = first < n_tiles ? (n_tiles - first + step - 1) / step : 0;

    auto coords = [&](unsigned i, int& c0, int& c1, int& c2, int& ii0) {
        unsigned o, seg, ic;
        strided_tile_decode(g, first + i * step, o, seg, ic);
        c0 = (int)(2 * ic * C);
        c1 = (int)seg * M;
        c2 = (int)o;
        ii0 = (int)(ic * C);
    };
    auto issue_load = [&](unsigned i) {
        int c0, c1, c2, ii0;
        coords(i, c0, c1, c2, ii0);
        const int s = (int)(i % NSTAGE);
        mbar_expect_tx(&full[s], TILE_BYTES);
#pragma unroll
        for (int b = 0; b < NBOX; ++b)
            tma_load_3d(stage0 + (size_t)s * M * C + (size_t)b * MB * C, map, &full[s], c0, c1 + b * MB, c2);
    };
    if (tid == 0) {
        for (unsigned i = 0; i < NSTAGE - 1 && i < n_mine; ++i) issue_load(i);
    }
    // |p|^2 of the transformed axis at this thread's points (kernel-multiply sweep)
    float p2a[P];
    if constexpr (MODE == FFT_MID) {
        static_for<0, P>([&](auto mc) { p2a[decltype(mc)::value] = sp.tab_axis[jt + decltype(mc)::value * T]; });
    }
    for (unsigned i = 0; i < n_mine; ++i) {
        const int s = (int)(i % NSTAGE);
        cf* tile = stage0 + (size_t)s * M * C;
        int c0, c1, c2, ii0;
        coords(i, c0, c1, c2, ii0);
        // |p|^2 of the other axes for this thread's line: requested before the wait so its latency is covered
        float wline = 0.f;
        if constexpr (MODE == FFT_MID) {
            const int ii = ii0 + c;
            if (sp.wtab) {
                wline = ii < g.inner ? sp.wtab[ii] : 0.f;
            } else {
                if (sp.tabA) wline += sp.tabA[(ii / sp.Nb) % sp.Ma];
                if (sp.tabB) wline += sp.tabB[(ii % sp.Nb) % sp.Mb];
            }
        }
        mbar_wait(&full[s], (unsigned)((i / NSTAGE) & 1));
        cf v[P];
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            v[m] = tile[(jt + m * T) * C + c];
        });
        if constexpr (PL::NPASS > 1) __syncthreads();      // every thread holds its inputs before the first exchange
        if constexpr (MODE == FFT_INV) {
            static_for<0, P>([&](auto mc) { v[decltype(mc)::value] = cswap(v[decltype(mc)::value]); });
        }
        fft_line_forward<PL, C, 1>(v, tile, c, jt, tw);
        if constexpr (NSTAGE < 3 && MODE != FFT_MID) {
            // two stages: refill the other one after the butterflies of this tile (see the kernel-multiply case below)
            if (tid == 0 && i + NSTAGE - 1 < n_mine) {
                tma_wait_read<0>();
                issue_load(i + NSTAGE - 1);
            }
        }
        if constexpr (MODE == FFT_MID) {
            if constexpr (NSTAGE < 3) {
                // two stages: refill the other one between the two FFTs of this tile; by now the store of the tile
                // before has long finished reading it, so the elected thread does not hold the CTA back
                if (tid == 0 && i + NSTAGE - 1 < n_mine) {
                    tma_wait_read<0>();
                    issue_load(i + NSTAGE - 1);
                }
            }
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = cswap(apply_symbol(v[m], p2a[m] + wline, sp));
            });
            fft_line_forward<PL, C, 1>(v, tile, c, jt, tw);
        }
        if constexpr (MODE != FFT_FWD) {
            static_for<0, P>([&](auto mc) { v[decltype(mc)::value] = cswap(v[decltype(mc)::value]); });
        }
        static_for<0, P>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            tile[(jt + m * T) * C + c] = v[m];
        });
        fence_async_smem();                                 // generic-proxy writes -> visible to the TMA store
        __syncthreads();
        if (tid == 0) {
#pragma unroll
            for (int b = 0; b < NBOX; ++b) tma_store_3d(map, tile + (size_t)b * MB * C, c0, c1 + b * MB, c2);
            tma_commit();
            if constexpr (NSTAGE >= 3) {
                // refill the stage of tile i-1 with tile i+NSTAGE-1: only the store just committed may still be
                // reading shared memory, so this never waits on a store in flight
                if (i + NSTAGE - 1 < n_mine) {
                    tma_wait_read<1>();
                    issue_load(i + NSTAGE - 1);
                }
            }
        }
    }
    if (tid == 0) tma_wait_all();
}

}  // namespace mbs
