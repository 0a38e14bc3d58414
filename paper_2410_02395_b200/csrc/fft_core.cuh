// fft_core.cuh -- register/shared-memory complex64 FFT of one line, forward sign e^{-2 pi i jk/M}
// (R9: forward unnormalised; the 1/M of the inverse is folded into the Fourier kernel).
//
// Scheme (Stockham autosort, decimation in time).  A line of M points is owned by T = M/P threads;
// thread jt holds, at the start of EVERY pass and at the end of the last one, the P points
//     p = jt + m*T,  m = 0..P-1                                  (register v[m])
// in natural order.  A pass of radix R (R | P) performs P/R butterflies per thread on registers
// v[b + r*(P/R)] (= points j + r*M/R with j = jt + b*T), after multiplying by the twiddles
// W_{Ns R}^{r k}, k = j mod Ns (Ns = product of the earlier radices), and -- unless it is the
// last pass -- scatters the results through shared memory to positions (j-k)*R + k + r*Ns and
// reads back v[m] = tile[jt + m*T].  The last pass writes to positions j + r*M/R, i.e. back into
// the same registers, so a forward transform, the Fourier-kernel multiply and the (swap-trick)
// inverse chain without any exchange, and global loads/stores always use the same pattern.
//
// Composite radices (8, 10, 16, 20, ...) are computed entirely in registers by a compile-time
// Cooley-Tukey split with constant twiddles; all register indices are compile-time.
#pragma once
#include "compat.h"
#include <type_traits>
#include <utility>

namespace mbs {

// ---------------------------------------------------------------------------------------------
// compile-time helpers
// ---------------------------------------------------------------------------------------------
template <int I, int N, class F>
MBS_HD void static_for(F&& f) {
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

constexpr double kPi = 3.14159265358979323846264338327950288;

constexpr double cx_sin_small(double x) {  // |x| <= pi/4
    double term = x, sum = x, x2 = x * x;
    for (int n = 1; n < 14; ++n) {
        term *= -x2 / double((2 * n) * (2 * n + 1));
        sum += term;
    }
    return sum;
}
constexpr double cx_cos_small(double x) {
    double term = 1.0, sum = 1.0, x2 = x * x;
    for (int n = 1; n < 14; ++n) {
        term *= -x2 / double((2 * n - 1) * (2 * n));
        sum += term;
    }
    return sum;
}
// cos / sin of 2 pi num / den, octant-reduced so the series argument stays in [-pi/4, pi/4]
constexpr double cx_cos_2pi(long long num, long long den) {
    num %= den;
    if (num < 0) num += den;
    // angle = 2 pi num/den = (pi/4) * (8 num/den)
    long long oct = (8 * num) / den;             // 0..7
    double rem = 2.0 * kPi * (double(num) / double(den)) - double(oct) * (kPi / 4.0);  // in [0, pi/4)
    switch (oct) {
        case 0: return cx_cos_small(rem);
        case 1: return cx_sin_small(kPi / 4.0 - rem);
        case 2: return -cx_sin_small(rem);
        case 3: return -cx_cos_small(kPi / 4.0 - rem);
        case 4: return -cx_cos_small(rem);
        case 5: return -cx_sin_small(kPi / 4.0 - rem);
        case 6: return cx_sin_small(rem);
        default: return cx_cos_small(kPi / 4.0 - rem);
    }
}
constexpr double cx_sin_2pi(long long num, long long den) { return cx_cos_2pi(4 * num - den, 4 * den); }

// multiply by W_R^m = exp(-2 pi i m / R), m and R compile-time, with the trivial cases folded
template <int R, int m>
MBS_HD cf mul_const_twiddle(cf a) {
    constexpr int mm = ((m % R) + R) % R;
    if constexpr (mm == 0) {
        return a;
    } else if constexpr (4 * mm == R) {
        return cmul_mi(a);
    } else if constexpr (2 * mm == R) {
        return make_float2(-a.x, -a.y);
    } else if constexpr (4 * mm == 3 * R) {
        return cmul_pi(a);
    } else if constexpr (8 * mm == R) {          // (1 - i)/sqrt2
        constexpr float s = 0.70710678118654752440f;
        return make_float2((a.x + a.y) * s, (a.y - a.x) * s);
    } else if constexpr (8 * mm == 3 * R) {      // (-1 - i)/sqrt2
        constexpr float s = 0.70710678118654752440f;
        return make_float2((a.y - a.x) * s, -(a.x + a.y) * s);
    } else if constexpr (8 * mm == 5 * R) {      // (-1 + i)/sqrt2
        constexpr float s = 0.70710678118654752440f;
        return make_float2(-(a.x + a.y) * s, (a.x - a.y) * s);
    } else if constexpr (8 * mm == 7 * R) {      // (1 + i)/sqrt2
        constexpr float s = 0.70710678118654752440f;
        return make_float2((a.x - a.y) * s, (a.x + a.y) * s);
    } else {
        constexpr float wr = (float)cx_cos_2pi(mm, R);
        constexpr float wi = (float)(-cx_sin_2pi(mm, R));
        return make_float2(a.x * wr - a.y * wi, a.x * wi + a.y * wr);
    }
}

// ---------------------------------------------------------------------------------------------
// in-register DFTs on v[BASE + STRIDE*n], n = 0..R-1.  After run(), X[k] is in
// v[BASE + STRIDE*slot(k)].
// ---------------------------------------------------------------------------------------------
template <int R> struct Split { static constexpr int A = 0, B = 0; };   // prime / hand-coded
template <> struct Split<6>  { static constexpr int A = 2, B = 3; };
template <> struct Split<8>  { static constexpr int A = 2, B = 4; };
template <> struct Split<10> { static constexpr int A = 2, B = 5; };
template <> struct Split<12> { static constexpr int A = 3, B = 4; };
template <> struct Split<16> { static constexpr int A = 4, B = 4; };
template <> struct Split<20> { static constexpr int A = 4, B = 5; };
template <> struct Split<32> { static constexpr int A = 4, B = 8; };
template <> struct Split<40> { static constexpr int A = 5, B = 8; };
// radices of the 3^2 * 5 * 7 sizes (the paper's own 1260 = 2^2 3^2 5 7 voxels per axis)
template <> struct Split<9>  { static constexpr int A = 3, B = 3; };
template <> struct Split<14> { static constexpr int A = 2, B = 7; };
template <> struct Split<15> { static constexpr int A = 3, B = 5; };
template <> struct Split<18> { static constexpr int A = 2, B = 9; };
template <> struct Split<21> { static constexpr int A = 3, B = 7; };
template <> struct Split<30> { static constexpr int A = 5, B = 6; };
template <> struct Split<42> { static constexpr int A = 6, B = 7; };

template <int R, int BASE, int STRIDE, int P, class Enable = void>
struct Dft;

template <int BASE, int STRIDE, int P>
struct Dft<1, BASE, STRIDE, P> {
    static constexpr int slot(int k) { return k; }
    static MBS_HD void run(cf (&)[P]) {}
};

template <int BASE, int STRIDE, int P>
struct Dft<2, BASE, STRIDE, P> {
    static constexpr int slot(int k) { return k; }
    static MBS_HD void run(cf (&v)[P]) {
        cf a = v[BASE], b = v[BASE + STRIDE];
        v[BASE] = cadd(a, b);
        v[BASE + STRIDE] = csub(a, b);
    }
};

template <int BASE, int STRIDE, int P>
struct Dft<3, BASE, STRIDE, P> {
    static constexpr int slot(int k) { return k; }
    static MBS_HD void run(cf (&v)[P]) {
        constexpr float s = 0.86602540378443864676f;
        cf a = v[BASE], b = v[BASE + STRIDE], c = v[BASE + 2 * STRIDE];
        cf t1 = cadd(b, c);
        cf t2 = make_float2(a.x - 0.5f * t1.x, a.y - 0.5f * t1.y);
        cf t3 = cscale(csub(b, c), s);
        v[BASE] = cadd(a, t1);
        v[BASE + STRIDE] = make_float2(t2.x + t3.y, t2.y - t3.x);
        v[BASE + 2 * STRIDE] = make_float2(t2.x - t3.y, t2.y + t3.x);
    }
};

template <int BASE, int STRIDE, int P>
struct Dft<4, BASE, STRIDE, P> {
    static constexpr int slot(int k) { return k; }
    static MBS_HD void run(cf (&v)[P]) {
        cf x0 = v[BASE], x1 = v[BASE + STRIDE], x2 = v[BASE + 2 * STRIDE], x3 = v[BASE + 3 * STRIDE];
        cf t0 = cadd(x0, x2), t1 = csub(x0, x2), t2 = cadd(x1, x3), t3 = cmul_mi(csub(x1, x3));
        v[BASE] = cadd(t0, t2);
        v[BASE + STRIDE] = cadd(t1, t3);
        v[BASE + 2 * STRIDE] = csub(t0, t2);
        v[BASE + 3 * STRIDE] = csub(t1, t3);
    }
};

template <int BASE, int STRIDE, int P>
struct Dft<5, BASE, STRIDE, P> {
    static constexpr int slot(int k) { return k; }
    static MBS_HD void run(cf (&v)[P]) {
        constexpr float c1 = (float)cx_cos_2pi(1, 5), c2 = (float)cx_cos_2pi(2, 5);
        constexpr float s1 = (float)cx_sin_2pi(1, 5), s2 = (float)cx_sin_2pi(2, 5);
        cf x0 = v[BASE], x1 = v[BASE + STRIDE], x2 = v[BASE + 2 * STRIDE], x3 = v[BASE + 3 * STRIDE],
           x4 = v[BASE + 4 * STRIDE];
        cf t1 = cadd(x1, x4), t2 = cadd(x2, x3), t3 = csub(x1, x4), t4 = csub(x2, x3);
        cf a1 = make_float2(x0.x + c1 * t1.x + c2 * t2.x, x0.y + c1 * t1.y + c2 * t2.y);
        cf a2 = make_float2(x0.x + c2 * t1.x + c1 * t2.x, x0.y + c2 * t1.y + c1 * t2.y);
        cf b1 = make_float2(s1 * t3.x + s2 * t4.x, s1 * t3.y + s2 * t4.y);
        cf b2 = make_float2(s2 * t3.x - s1 * t4.x, s2 * t3.y - s1 * t4.y);
        v[BASE] = make_float2(x0.x + t1.x + t2.x, x0.y + t1.y + t2.y);
        v[BASE + STRIDE] = make_float2(a1.x + b1.y, a1.y - b1.x);       // a1 - i b1
        v[BASE + 4 * STRIDE] = make_float2(a1.x - b1.y, a1.y + b1.x);   // a1 + i b1
        v[BASE + 2 * STRIDE] = make_float2(a2.x + b2.y, a2.y - b2.x);   // a2 - i b2
        v[BASE + 3 * STRIDE] = make_float2(a2.x - b2.y, a2.y + b2.x);   // a2 + i b2
    }
};

// radix 7: x_j +- x_{7-j} pairs; X_k = x0 + sum_j cos(2 pi jk/7) s_j -+ i sum_j sin(2 pi jk/7) d_j
template <int BASE, int STRIDE, int P>
struct Dft<7, BASE, STRIDE, P> {
    static constexpr int slot(int k) { return k; }
    static MBS_HD void run(cf (&v)[P]) {
        constexpr float c1 = (float)cx_cos_2pi(1, 7), c2 = (float)cx_cos_2pi(2, 7), c3 = (float)cx_cos_2pi(3, 7);
        constexpr float s1 = (float)cx_sin_2pi(1, 7), s2 = (float)cx_sin_2pi(2, 7), s3 = (float)cx_sin_2pi(3, 7);
        const cf x0 = v[BASE];
        const cf p1 = cadd(v[BASE + STRIDE], v[BASE + 6 * STRIDE]), m1 = csub(v[BASE + STRIDE], v[BASE + 6 * STRIDE]);
        const cf p2 = cadd(v[BASE + 2 * STRIDE], v[BASE + 5 * STRIDE]), m2 = csub(v[BASE + 2 * STRIDE], v[BASE + 5 * STRIDE]);
        const cf p3 = cadd(v[BASE + 3 * STRIDE], v[BASE + 4 * STRIDE]), m3 = csub(v[BASE + 3 * STRIDE], v[BASE + 4 * STRIDE]);
        // k = 1: cos(1,2,3), sin(1,2,3);  k = 2: cos(2,4->3,6->1), sin(2, -3, -1);  k = 3: cos(3,6->1,9->2), sin(3, -1, 2)
        const cf a1 = make_float2(x0.x + c1 * p1.x + c2 * p2.x + c3 * p3.x, x0.y + c1 * p1.y + c2 * p2.y + c3 * p3.y);
        const cf a2 = make_float2(x0.x + c2 * p1.x + c3 * p2.x + c1 * p3.x, x0.y + c2 * p1.y + c3 * p2.y + c1 * p3.y);
        const cf a3 = make_float2(x0.x + c3 * p1.x + c1 * p2.x + c2 * p3.x, x0.y + c3 * p1.y + c1 * p2.y + c2 * p3.y);
        const cf b1 = make_float2(s1 * m1.x + s2 * m2.x + s3 * m3.x, s1 * m1.y + s2 * m2.y + s3 * m3.y);
        const cf b2 = make_float2(s2 * m1.x - s3 * m2.x - s1 * m3.x, s2 * m1.y - s3 * m2.y - s1 * m3.y);
        const cf b3 = make_float2(s3 * m1.x - s1 * m2.x + s2 * m3.x, s3 * m1.y - s1 * m2.y + s2 * m3.y);
        v[BASE] = make_float2(x0.x + p1.x + p2.x + p3.x, x0.y + p1.y + p2.y + p3.y);
        v[BASE + STRIDE] = make_float2(a1.x + b1.y, a1.y - b1.x);       // a - i b
        v[BASE + 6 * STRIDE] = make_float2(a1.x - b1.y, a1.y + b1.x);   // a + i b
        v[BASE + 2 * STRIDE] = make_float2(a2.x + b2.y, a2.y - b2.x);
        v[BASE + 5 * STRIDE] = make_float2(a2.x - b2.y, a2.y + b2.x);
        v[BASE + 3 * STRIDE] = make_float2(a3.x + b3.y, a3.y - b3.x);
        v[BASE + 4 * STRIDE] = make_float2(a3.x - b3.y, a3.y + b3.x);
    }
};

// composite R = A*B: n = B*n1 + n2, k = k1 + A*k2.
//  step 1: for each n2, A-point DFT over n1 on slots B*n1 + n2      -> k1 at slot B*slotA(k1) + n2
//  step 2: multiply (k1, n2) by W_R^{n2 k1}
//  step 3: for each k1, B-point DFT over n2 on slots B*slotA(k1)+n2 -> k2 at slot B*slotA(k1) + slotB(k2)
template <int R, int BASE, int STRIDE, int P>
struct Dft<R, BASE, STRIDE, P, std::enable_if_t<(Split<R>::A > 0)>> {
    static constexpr int A = Split<R>::A, B = Split<R>::B;
    using DA = Dft<A, 0, 1, A>;   // only for slot()
    using DB = Dft<B, 0, 1, B>;
    static constexpr int slot(int k) { return B * DA::slot(k % A) + DB::slot(k / A); }
    static MBS_HD void run(cf (&v)[P]) {
        static_for<0, B>([&](auto n2c) {
            constexpr int n2 = decltype(n2c)::value;
            Dft<A, BASE + STRIDE * n2, STRIDE * B, P>::run(v);
        });
        static_for<0, A>([&](auto k1c) {
            constexpr int k1 = decltype(k1c)::value;
            constexpr int sa = Dft<A, 0, 1, A>::slot(k1);
            static_for<1, B>([&](auto n2c) {
                constexpr int n2 = decltype(n2c)::value;
                constexpr int idx = BASE + STRIDE * (B * sa + n2);
                v[idx] = mul_const_twiddle<R, n2 * k1>(v[idx]);
            });
            Dft<B, BASE + STRIDE * B * sa, STRIDE, P>::run(v);
        });
    }
};

// ---------------------------------------------------------------------------------------------
// plans
// ---------------------------------------------------------------------------------------------
template <int M_, int P_, int... Rs>
struct Plan {
    static constexpr int M = M_;
    static constexpr int P = P_;
    static constexpr int T = M_ / P_;          // threads per line
    static constexpr int NPASS = sizeof...(Rs);
    static constexpr int radix(int i) {
        constexpr int r[sizeof...(Rs)] = {Rs...};
        return r[i];
    }
    static constexpr int ns(int i) {           // product of radices before pass i
        int n = 1;
        for (int q = 0; q < i; ++q) n *= radix(q);
        return n;
    }
    static constexpr bool valid() {
        int n = 1;
        for (int q = 0; q < NPASS; ++q) {
            if (P_ % radix(q) != 0) return false;
            n *= radix(q);
        }
        return n == M_ && M_ % P_ == 0;
    }
    static_assert(valid(), "bad FFT plan");
    static constexpr bool generic = false;
};

// Generic mixed-radix plan: the pass radices need not divide P (sizes with several odd prime factors, e.g.
// 630 = 21 * 30).  The interface to the kernels is unchanged -- thread jt holds points jt + m*T, m < P, before and
// after the transform -- but every pass goes through the shared-memory tile: pass i has M / R_i butterflies, thread jt
// takes butterflies jt, jt + T, ... (the last round may be partial).
template <int M_, int P_, int... Rs>
struct GPlan {
    static constexpr int M = M_;
    static constexpr int P = P_;
    static constexpr int T = M_ / P_;
    static constexpr int NPASS = sizeof...(Rs) + 1;     // +1: kernels size their tiles by "more than one pass"
    static constexpr int NR = sizeof...(Rs);
    static constexpr int radix(int i) {
        constexpr int r[sizeof...(Rs)] = {Rs...};
        return r[i];
    }
    static constexpr int ns(int i) {
        int n = 1;
        for (int q = 0; q < i; ++q) n *= radix(q);
        return n;
    }
    static constexpr bool valid() {
        int n = 1;
        for (int q = 0; q < NR; ++q) n *= radix(q);
        return n == M_ && M_ % P_ == 0;
    }
    static_assert(valid(), "bad generic FFT plan");
    static constexpr bool generic = true;
};

template <class PL, int SP, int SC>
MBS_DEV void fft_line_forward_generic(cf (&v)[PL::P], cf* tile, const int c, const int jt, const cf* MBS_RESTRICT tw) {
    constexpr int M = PL::M, P = PL::P, T = PL::T;
    // natural order into the tile (the caller's v may differ from what the tile holds)
    static_for<0, P>([&](auto mc) {
        constexpr int m = decltype(mc)::value;
        tile[(jt + m * T) * SP + c * SC] = v[m];
    });
    MBS_SYNC();
    static_for<0, PL::NR>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int R = PL::radix(i);
        constexpr int Ns = PL::ns(i);
        constexpr int NBF = M / R;                    // butterflies of this pass
        constexpr int ROUNDS = (NBF + T - 1) / T;
        cf w[ROUNDS][R];
        static_for<0, ROUNDS>([&](auto qc) {
            constexpr int q = decltype(qc)::value;
            const int j = jt + q * T;
            if (ROUNDS * T == NBF || j < NBF) {
                static_for<0, R>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    w[q][r] = tile[(j + r * NBF) * SP + c * SC];
                });
                if constexpr (i > 0) {
                    const int k = j % Ns;
                    const int step = k * (M / (Ns * R));
                    static_for<1, R>([&](auto rc) {
                        constexpr int r = decltype(rc)::value;
                        w[q][r] = cmul(w[q][r], tw[r * step]);
                    });
                }
                Dft<R, 0, 1, R>::run(w[q]);
            }
        });
        MBS_SYNC();                                   // every input of the pass has been read
        static_for<0, ROUNDS>([&](auto qc) {
            constexpr int q = decltype(qc)::value;
            const int j = jt + q * T;
            if (ROUNDS * T == NBF || j < NBF) {
                const int k = j % Ns;
                const int j0 = (j - k) * R + k;
                static_for<0, R>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    tile[(j0 + r * Ns) * SP + c * SC] = w[q][Dft<R, 0, 1, R>::slot(r)];
                });
            }
        });
        MBS_SYNC();
    });
    static_for<0, P>([&](auto mc) {
        constexpr int m = decltype(mc)::value;
        v[m] = tile[(jt + m * T) * SP + c * SC];
    });
    MBS_SYNC();                                       // the tile is free again when the call returns
}

// One forward FFT of the line owned by (c, jt).  tile: shared memory, element (p, c) at
// tile[p*SP + c*SC].  tw: table W_M^n = exp(-2 pi i n/M), n in [0, M) (shared or global).
template <class PL, int SP, int SC>
MBS_DEV void fft_line_forward(cf (&v)[PL::P], cf* tile, const int c, const int jt, const cf* MBS_RESTRICT tw) {
    constexpr int M = PL::M, P = PL::P, T = PL::T;
    if constexpr (PL::generic) {
        fft_line_forward_generic<PL, SP, SC>(v, tile, c, jt, tw);
        return;
    } else
    static_for<0, PL::NPASS>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int R = PL::radix(i);
        constexpr int Ns = PL::ns(i);
        constexpr int NB = P / R;
        constexpr bool last = (i == PL::NPASS - 1);
        // twiddles W_{Ns R}^{r k} = W_M^{r k M/(Ns R)}
        if constexpr (i > 0) {
            static_for<0, NB>([&](auto bc) {
                constexpr int b = decltype(bc)::value;
                const int j = jt + b * T;
                const int k = j % Ns;
                const int step = k * (M / (Ns * R));
                static_for<1, R>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    v[b + r * NB] = cmul(v[b + r * NB], tw[r * step]);
                });
            });
        }
        static_for<0, NB>([&](auto bc) {
            constexpr int b = decltype(bc)::value;
            Dft<R, b, NB, P>::run(v);
        });
        if constexpr (!last) {
            static_for<0, NB>([&](auto bc) {
                constexpr int b = decltype(bc)::value;
                const int j = jt + b * T;
                const int k = j % Ns;
                const int j0 = (j - k) * R + k;
                static_for<0, R>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    constexpr int src = b + NB * Dft<R, 0, 1, R>::slot(r);
                    tile[(j0 + r * Ns) * SP + c * SC] = v[src];
                });
            });
            MBS_SYNC();
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = tile[(jt + m * T) * SP + c * SC];
            });
            MBS_SYNC();
        } else {
            // bring X[r] of butterfly b from slot(r) to its natural register b + r*NB
            cf w[P];
            static_for<0, NB>([&](auto bc) {
                constexpr int b = decltype(bc)::value;
                static_for<0, R>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    w[b + r * NB] = v[b + NB * Dft<R, 0, 1, R>::slot(r)];
                });
            });
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = w[m];
            });
        }
    });
}

// ---------------------------------------------------------------------------------------------
// Warp-local variant: the T <= 32 threads of a line are lanes of ONE warp, so the exchanges need only
// __syncwarp and every warp runs its lines independently of the rest of the CTA.  `line` is the line's
// private scratch of line_scratch_elems<PL>() elements; point i lives at i + (i >> 4) (one pad element per
// 16), which makes both the scatter of a pass (stride R per lane) and the unit-stride read-back
// conflict-free.  Device only.
// ---------------------------------------------------------------------------------------------
#ifdef __CUDACC__
template <class PL>
constexpr int line_scratch_elems() { return PL::M + PL::M / 16 + 1; }

MBS_DEV int pad16(int i) { return i + (i >> 4); }

// Twiddles of the warp-local variant.  Lanes of a warp hold consecutive points of ONE line, so for a fixed butterfly
// input r they need W^{r k} for consecutive k: the table is laid out per pass as [r - 1][k] (k fastest), which makes
// those reads unit-stride (the natural table W_M^n would be read with stride 2 r ... 16 r: up to 16-way bank
// conflicts).  Pass i > 0 starts at Ns_i - Ns_1 (the sizes (R_i - 1) Ns_i telescope), total M - R_0 < M entries.
template <class PL>
MBS_DEV void fill_warp_twiddles(cf* twp, const cf* MBS_RESTRICT tw_global, const int tid, const int nthreads) {
    constexpr int M = PL::M;
    static_for<1, PL::NPASS>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int R = PL::radix(i), Ns = PL::ns(i), base = Ns - PL::ns(1);
        for (int idx = tid; idx < (R - 1) * Ns; idx += nthreads) {
            const int r = idx / Ns + 1, k = idx - (r - 1) * Ns;
            twp[base + idx] = tw_global[r * k * (M / (Ns * R))];
        }
    });
}

template <class PL>
MBS_DEV void fft_line_forward_warp(cf (&v)[PL::P], cf* line, const int jt, const cf* MBS_RESTRICT twp) {
    constexpr int M = PL::M, P = PL::P, T = PL::T;
    static_assert(T <= 32, "a line must fit in one warp");
    static_for<0, PL::NPASS>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int R = PL::radix(i);
        constexpr int Ns = PL::ns(i);
        constexpr int NB = P / R;
        constexpr bool last = (i == PL::NPASS - 1);
        if constexpr (i > 0) {
            static_for<0, NB>([&](auto bc) {
                constexpr int b = decltype(bc)::value;
                const int j = jt + b * T;
                const int k = j % Ns;
                constexpr int base = Ns - PL::ns(1);
                static_for<1, R>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    v[b + r * NB] = cmul(v[b + r * NB], twp[base + (r - 1) * Ns + k]);
                });
            });
        }
        static_for<0, NB>([&](auto bc) {
            constexpr int b = decltype(bc)::value;
            Dft<R, b, NB, P>::run(v);
        });
        if constexpr (!last) {
            static_for<0, NB>([&](auto bc) {
                constexpr int b = decltype(bc)::value;
                const int j = jt + b * T;
                const int k = j % Ns;
                const int j0 = (j - k) * R + k;
                static_for<0, R>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    constexpr int src = b + NB * Dft<R, 0, 1, R>::slot(r);
                    line[pad16(j0 + r * Ns)] = v[src];
                });
            });
            __syncwarp();
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = line[pad16(jt + m * T)];
            });
            __syncwarp();
        } else {
            cf w[P];
            static_for<0, NB>([&](auto bc) {
                constexpr int b = decltype(bc)::value;
                static_for<0, R>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    w[b + r * NB] = v[b + NB * Dft<R, 0, 1, R>::slot(r)];
                });
            });
            static_for<0, P>([&](auto mc) {
                constexpr int m = decltype(mc)::value;
                v[m] = w[m];
            });
        }
    });
}
#endif

}  // namespace mbs
