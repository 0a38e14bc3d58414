// fft_plans.h -- the subdomain lengths M this build has FFT plans for (2^a, 5*2^a, 3*2^a, 25*2^a and 3^2 5 7 sizes), with the
// points per thread P, the pass radices, the tile widths CS / CSM of the strided forward-inverse / kernel-multiply
// sweeps (voxels per tile row) and the lines per tile CC of the contiguous tile kernels.  An optional NSTAGE fixes
// the TMA stages of the forward/inverse strided sweeps (default: as many as fit, at most 3); 320 runs two 40 KiB
// stages so that two CTAs share an SM (measured on cfg 4: 0.77 ms against 0.86 ms with one CTA of 32-wide tiles).
// BASELINE.json configs need 128 (cfg 1, 3), 256 (cfg 3, 5), 320 (cfg 4) and 512 (cfg 2, 5).
#pragma once
#include "fft_core.cuh"

namespace mbs {

template <int M> struct FftPlan;
//                                          M     P   radices...
template <> struct FftPlan<8>    { using type = Plan<8,    8,  8>;            static constexpr int CS = 64, CSM = 64, CC = 64; };
template <> struct FftPlan<16>   { using type = Plan<16,   8,  8, 2>;         static constexpr int CS = 64, CSM = 64, CC = 64; };
template <> struct FftPlan<32>   { using type = Plan<32,   8,  8, 4>;         static constexpr int CS = 32, CSM = 32, CC = 32; };
template <> struct FftPlan<64>   { using type = Plan<64,   8,  8, 8>;         static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<128>  { using type = Plan<128,  16, 16, 8>;        static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<256>  { using type = Plan<256,  16, 16, 16>;       static constexpr int CS = 32, CSM = 16, CC = 16; };
template <> struct FftPlan<512>  { using type = Plan<512,  16, 16, 16, 2>;    static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<1024> { using type = Plan<1024, 16, 16, 16, 4>;    static constexpr int CS = 8, CSM = 8, CC = 8;  };
template <> struct FftPlan<40>   { using type = Plan<40,   20, 20, 2>;        static constexpr int CS = 64, CSM = 64, CC = 64; };
template <> struct FftPlan<80>   { using type = Plan<80,   20, 20, 4>;        static constexpr int CS = 32, CSM = 32, CC = 32; };
template <> struct FftPlan<160>  { using type = Plan<160,  20, 20, 4, 2>;     static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<320>  { using type = Plan<320,  20, 20, 4, 4>;     static constexpr int CS = 16, CSM = 32, CC = 16, NSTAGE = 2; };
template <> struct FftPlan<640>  { using type = Plan<640,  20, 20, 4, 4, 2>;  static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<48>   { using type = Plan<48,   12, 12, 4>;        static constexpr int CS = 64, CSM = 64, CC = 64; };
template <> struct FftPlan<96>   { using type = Plan<96,   24, 12, 8>;        static constexpr int CS = 32, CSM = 32, CC = 32; };
template <> struct FftPlan<192>  { using type = Plan<192,  12, 12, 4, 4>;     static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<384>  { using type = Plan<384,  24, 12, 8, 4>;     static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<768>  { using type = Plan<768,  24, 12, 8, 8>;     static constexpr int CS = 8, CSM = 8, CC = 8;  };

// 5^2 * 2^a (decimal grids such as the paper's 200^3 validation run)
template <> struct FftPlan<100>  { using type = Plan<100,  10, 10, 10>;       static constexpr int CS = 32, CSM = 32, CC = 32; };
template <> struct FftPlan<200>  { using type = Plan<200,  20, 20, 10>;       static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<400>  { using type = Plan<400,  20, 20, 20>;       static constexpr int CS = 16, CSM = 16, CC = 16; };
// sizes with the factors 3^2 and 7 (generic two-pass plans, fft_core.cuh GPlan): the paper's own grid is 1260 = 2^2 3^2 5 7
// voxels per axis, i.e. subdomains of 1260, 630, 420, 315 or 252 voxels for 1..5 subdomains per axis
template <> struct FftPlan<63>   { using type = GPlan<63,   7,  7, 9>;        static constexpr int CS = 32, CSM = 32, CC = 32; };
template <> struct FftPlan<90>   { using type = GPlan<90,   9,  9, 10>;       static constexpr int CS = 32, CSM = 32, CC = 32; };
template <> struct FftPlan<126>  { using type = GPlan<126,  9,  9, 14>;       static constexpr int CS = 32, CSM = 32, CC = 32; };
template <> struct FftPlan<180>  { using type = GPlan<180,  12, 12, 15>;      static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<252>  { using type = GPlan<252,  12, 12, 21>;      static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<315>  { using type = GPlan<315,  21, 21, 15>;      static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<360>  { using type = GPlan<360,  18, 18, 20>;      static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<420>  { using type = GPlan<420,  20, 20, 21>;      static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<630>  { using type = GPlan<630,  21, 21, 30>;      static constexpr int CS = 16, CSM = 16, CC = 16; };
template <> struct FftPlan<1260> { using type = GPlan<1260, 30, 30, 42>;      static constexpr int CS = 8, CSM = 8, CC = 8;  };

}  // namespace mbs

// MBS_DEV_SIZES (build.py --sizes, kernel development only) restricts the library to a few sizes for quick rebuilds.
#ifdef MBS_DEV_SIZES
#define MBS_FOR_EACH_FFT_SIZE(X) MBS_DEV_SIZES(X)
#else
#define MBS_FOR_EACH_FFT_SIZE(X) \
    X(8) X(16) X(32) X(64) X(128) X(256) X(512) X(1024) X(40) X(80) X(160) X(320) X(640) X(48) X(96) X(192) X(384) X(768) \
    X(100) X(200) X(400) X(63) X(90) X(126) X(180) X(252) X(315) X(360) X(420) X(630) X(1260)
#endif
