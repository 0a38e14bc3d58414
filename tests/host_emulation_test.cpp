// host_emulation_test.cpp -- runs the FFT tile kernel BODIES on the host, one std::thread per CUDA
// thread with a std::barrier for __syncthreads, and compares with a naive O(M^2) DFT in double.
// Purpose: check the Stockham / composite-radix index arithmetic on a machine without a GPU.
// Test-only (tests/test_host_emulation.py builds and runs it); never linked into the library.
//
//   g++ -std=c++20 -O1 -pthread host_emulation_test.cpp -o /tmp/mbs_host_emu && /tmp/mbs_host_emu
#include <barrier>
#include <complex>
#include <cstdio>
#include <cstdlib>
#include <functional>
#include <thread>
#include <vector>

static thread_local std::barrier<>* g_barrier = nullptr;
void mbs_host_barrier() { g_barrier->arrive_and_wait(); }

#include "fft_kernels.cuh"
#include "fft_plans.h"

using namespace mbs;
typedef std::complex<double> cd;

static std::vector<cf> make_twiddles(int M) {
    std::vector<cf> tw(M);
    for (int n = 0; n < M; ++n) {
        tw[n].x = (float)std::cos(2.0 * M_PI * n / M);
        tw[n].y = (float)(-std::sin(2.0 * M_PI * n / M));
    }
    return tw;
}

static void naive_dft(const std::vector<cd>& in, std::vector<cd>& out, int sign) {
    const int M = (int)in.size();
    out.assign(M, cd(0, 0));
    for (int k = 0; k < M; ++k) {
        cd acc(0, 0);
        for (int n = 0; n < M; ++n) acc += in[n] * std::polar(1.0, sign * 2.0 * M_PI * (double)((long long)k * n % M) / M);
        out[k] = acc;
    }
}

template <class F>
static void run_block(int nthreads, F&& body) {
    std::barrier<> bar(nthreads);
    std::vector<std::thread> th;
    for (int t = 0; t < nthreads; ++t)
        th.emplace_back([&, t]() {
            g_barrier = &bar;
            body(t);
        });
    for (auto& x : th) x.join();
}

static double frand() { return rand() / (double)RAND_MAX - 0.5; }

template <class PL, int C, int MODE>
static double test_strided(int n_outer, int n_seg, int inner) {
    constexpr int M = PL::M;
    const long long stride = inner;
    const long long outer_stride = (long long)n_seg * M * inner;
    const long long total = outer_stride * n_outer;
    std::vector<cf> data(total);
    for (auto& z : data) z = make_float2((float)frand(), (float)frand());
    std::vector<cf> ref = data;
    auto tw = make_twiddles(M);
    std::vector<float> tab(M), tabB(inner);
    for (int i = 0; i < M; ++i) tab[i] = (float)(0.37 * i);
    for (int i = 0; i < inner; ++i) tabB[i] = (float)(0.11 * i);
    SymbolParams sp{};
    sp.A0 = 1.1f; sp.B0 = 0.3f; sp.cr = 0.0f; sp.ci = -0.01f; sp.scale = 1.0f / M; sp.inverse = 1;
    sp.tab_axis = tab.data(); sp.tabA = nullptr; sp.tabB = tabB.data(); sp.Nb = inner; sp.Ma = 1; sp.Mb = inner;
    StridedGeom g{};
    g.outer_stride = outer_stride; g.stride = stride; g.n_outer = n_outer; g.n_seg = n_seg; g.inner = inner;
    g.tiles_inner = (inner + C - 1) / C; g.n_tiles = (long long)n_outer * n_seg * g.tiles_inner;
    const int nblocks = 2;
    std::vector<cf> smem(strided_smem_elems<PL, C>() + 8);
    for (int b = 0; b < nblocks; ++b)
        run_block(PL::T * C, [&](int tid) {
            fft_strided_body<PL, C, MODE>(data.data(), g, sp, tw.data(), tid, b, nblocks, smem.data());
        });
    double err = 0, nrm = 0;
    std::vector<cd> lin(M), lout(M), l2(M);
    for (int o = 0; o < n_outer; ++o)
        for (int s = 0; s < n_seg; ++s)
            for (int i = 0; i < inner; ++i) {
                long long base = o * outer_stride + (long long)s * M * stride + i;
                for (int p = 0; p < M; ++p) lin[p] = cd(ref[base + p * stride].x, ref[base + p * stride].y);
                if (MODE == FFT_FWD) naive_dft(lin, lout, -1);
                else if (MODE == FFT_INV) naive_dft(lin, lout, +1);
                else {
                    naive_dft(lin, l2, -1);
                    for (int p = 0; p < M; ++p) {
                        double p2 = (double)tab[p] + (double)tabB[i];
                        cd D(sp.A0 - sp.cr * p2, sp.B0 - sp.ci * p2);
                        l2[p] = l2[p] * (double)sp.scale / D;
                    }
                    naive_dft(l2, lout, +1);
                }
                for (int p = 0; p < M; ++p) {
                    cd got(data[base + p * stride].x, data[base + p * stride].y);
                    err += std::norm(got - lout[p]);
                    nrm += std::norm(lout[p]);
                }
            }
    return std::sqrt(err / nrm);
}

template <class PL, int C, int MODE>
static double test_contig(long long n_lines) {
    constexpr int M = PL::M;
    std::vector<cf> data(n_lines * M), out(n_lines * M);
    for (auto& z : data) z = make_float2((float)frand(), (float)frand());
    auto tw = make_twiddles(M);
    std::vector<float> tab(M);
    for (int i = 0; i < M; ++i) tab[i] = (float)(0.37 * i);
    SymbolParams sp{};
    sp.A0 = 1.1f; sp.B0 = 0.3f; sp.cr = 0.0f; sp.ci = -0.01f; sp.scale = 1.0f / M; sp.inverse = 1;
    sp.tab_axis = tab.data();
    ContigGeom g{};
    g.n_lines = n_lines; g.n_tiles = (n_lines + C - 1) / C;
    const int nblocks = 2;
    std::vector<cf> smem(contig_smem_elems<PL, C>() + 8);
    for (int b = 0; b < nblocks; ++b)
        run_block(PL::T * C, [&](int tid) {
            fft_contig_body<PL, C, MODE>(data.data(), out.data(), g, sp, tw.data(), tid, b, nblocks, smem.data());
        });
    double err = 0, nrm = 0;
    std::vector<cd> lin(M), lout(M), l2(M);
    for (long long l = 0; l < n_lines; ++l) {
        for (int p = 0; p < M; ++p) lin[p] = cd(data[l * M + p].x, data[l * M + p].y);
        if (MODE == FFT_FWD) naive_dft(lin, lout, -1);
        else if (MODE == FFT_INV) naive_dft(lin, lout, +1);
        else {
            naive_dft(lin, l2, -1);
            for (int p = 0; p < M; ++p) {
                double p2 = tab[p];
                cd D(sp.A0 - sp.cr * p2, sp.B0 - sp.ci * p2);
                l2[p] = l2[p] * (double)sp.scale / D;
            }
            naive_dft(l2, lout, +1);
        }
        for (int p = 0; p < M; ++p) {
            cd got(out[l * M + p].x, out[l * M + p].y);
            err += std::norm(got - lout[p]);
            nrm += std::norm(lout[p]);
        }
    }
    return std::sqrt(err / nrm);
}

static int g_fail = 0;
static void report(const char* what, int M, double err) {
    const bool ok = err < 2e-6;
    std::printf("%-18s M=%4d rel_l2=%.3e %s\n", what, M, err, ok ? "ok" : "FAIL");
    if (!ok) g_fail = 1;
}

template <int M>
static void test_size() {
    using PL = typename FftPlan<M>::type;
    constexpr int CS = FftPlan<M>::CSM, CC = FftPlan<M>::CC;
    report("strided fwd", M, test_strided<PL, CS, FFT_FWD>(2, 2, CS + 5));
    report("strided inv", M, test_strided<PL, CS, FFT_INV>(1, 2, CS + 5));
    report("strided mid", M, test_strided<PL, CS, FFT_MID>(1, 1, CS + 3));
    report("contig fwd", M, test_contig<PL, CC, FFT_FWD>(2 * CC + 3));
    report("contig inv", M, test_contig<PL, CC, FFT_INV>(CC + 1));
    report("contig mid", M, test_contig<PL, CC, FFT_MID>(CC + 2));
}

int main(int argc, char** argv) {
    srand(1234);
    int only = argc > 1 ? atoi(argv[1]) : 0;
#define MBS_PLAN_TEST(Mv) if (!only || only == Mv) test_size<Mv>();
    MBS_FOR_EACH_FFT_SIZE(MBS_PLAN_TEST)
    std::printf(g_fail ? "HOST EMULATION FAILED\n" : "HOST EMULATION PASSED\n");
    return g_fail;
}
