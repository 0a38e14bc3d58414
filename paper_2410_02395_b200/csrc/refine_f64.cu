// refine_f64.cu -- double-precision evaluation of  r_ref = B (x_ref - (L+I)^-1 (B x_ref + y_vec))  for the split iterate
// (api.cu recenter(); DESIGN.md section 6 "Split iterate").
//
// Mixed-precision iterative refinement: the iteration of Eq. (6) runs in complex64 on the small part delta of
// x = x_ref + delta, while the residual of the frozen part x_ref is computed here in complex128, a few times per solve, on
// small (L2-resident) grids.  The fixed point of the iteration is then the solution of the double-precision equations, not of
// their complex64 roundings (twiddles, B_diag, symbol), which on ill-conditioned problems differ by more than the parity bar
// (config 2: 1.6e-4 on the converged field).  Nothing here is on the per-iteration hot path; the kernels are plain:
//   k_bxy     u = B_diag x + ysc y - sum_d corr_d(x)         (Eq. (8); corrections evaluated per edge voxel)
//   k_dft     naive O(M) sum per output along one axis of a subdomain, twiddles from a double table
//   k_symbol  multiply by 1 / (c (k0^2 - |p|^2) + 1) / prod M_d
//   k_dref    d_ref = x_ref - u;  then k_bxy again: r_ref = B d_ref;  k_round: rounded once to complex64
// The complex64 last sweep then forms r = r_ref + B_diag (delta - u') - corr(delta - u'): its rounding (B_diag in complex64
// included) touches only the small part.
#include "mbs_internal.h"

namespace mbs {

typedef double2 cd2;
__device__ __forceinline__ cd2 zmul(cd2 a, cd2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ cd2 zadd(cd2 a, cd2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cd2 zsub(cd2 a, cd2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cd2 to_z(cf a) { return make_double2((double)a.x, (double)a.y); }
__device__ __forceinline__ cd2 to_z(cd2 a) { return a; }

// corr_ax(x) at the voxel with index i along axis `ax` (other indices fixed through base / stride), or 0 if it is no edge point
//   first t points of s (b = e):          c sum_a K[a][b] (x_{s-1}[M-t+a] - x_s[M-t+a])
//   last  t points of s (a = e - (M-t)):  c sum_b K[a][b] (x_{s+1}[b]     - x_s[b])         (P:124-128 read with P:106)
template <class T>
__device__ __forceinline__ cd2 corr_at(const GridDesc& g, const T* __restrict__ x, const double* __restrict__ K, const cd2 c,
                                       const int ax, const int i, const long long base, const long long stride) {
    cd2 out = make_double2(0.0, 0.0);
    if (g.a[ax] == 0 || g.t == 0) return out;
    const int t = g.t, M = g.M[ax], S = g.S[ax];
    const int s = i / M, e = i - s * M;
    const bool first = e < t, last = e >= M - t;
    if (!first && !last) return out;
    for (int pass = 0; pass < 2; ++pass) {                // a point may be in both edges only if 2t > M, which mbs_create refuses
        const bool is_last = pass == 1;
        if (is_last ? !last : !first) continue;
        int nb = is_last ? s + 1 : s - 1;
        bool has_nb = true;
        if (nb < 0 || nb >= S) {
            if (g.per[ax]) nb = (nb + S) % S;
            else has_nb = false;
        }
        const int k = is_last ? e - (M - t) : e;
        const int off = is_last ? 0 : M - t;              // last edge reads FIRST points, first edge reads LAST points
        double sr = 0.0, si = 0.0;
        for (int q = 0; q < t; ++q) {
            const double kk = is_last ? K[k * t + q] : K[q * t + k];
            const cd2 ov = to_z(x[base + (long long)(s * M + off + q) * stride]);
            double dx = -ov.x, dy = -ov.y;
            if (has_nb) {
                const cd2 nv = to_z(x[base + (long long)(nb * M + off + q) * stride]);
                dx += nv.x;
                dy += nv.y;
            }
            sr += kk * dx;
            si += kk * dy;
        }
        out = zadd(out, zmul(c, make_double2(sr, si)));
    }
    return out;
}

template <class T>
__global__ void __launch_bounds__(256) k_bxy_f64(const GridDesc g, const T* __restrict__ x, const cf* __restrict__ y, const cd2 ysc,
                                                 const cd2* __restrict__ bdiag, const double* __restrict__ K, const cd2 c,
                                                 cd2* __restrict__ out) {
    const long long s1 = g.N[2], s0 = (long long)g.N[1] * g.N[2];
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < g.voxels; idx += (long long)gridDim.x * blockDim.x) {
        const int i2 = (int)(idx % g.N[2]);
        const long long row = idx / g.N[2];
        const int i1 = (int)(row % g.N[1]), i0 = (int)(row / g.N[1]);
        cd2 v = zmul(bdiag[idx], to_z(x[idx]));
        if (y) v = zadd(v, zmul(ysc, to_z(y[idx])));
        v = zsub(v, corr_at(g, x, K, c, 0, i0, (long long)i1 * s1 + i2, s0));
        v = zsub(v, corr_at(g, x, K, c, 1, i1, (long long)i0 * s0 + i2, s1));
        v = zsub(v, corr_at(g, x, K, c, 2, i2, (long long)i0 * s0 + (long long)i1 * s1, 1));
        out[idx] = v;
    }
}

// out[k] = sum_n in[n] w^{sign n k} along axis `ax` within each subdomain; tw[j] = exp(-2 pi i j / M)
__global__ void __launch_bounds__(256) k_dft_f64(const GridDesc g, const cd2* __restrict__ in, cd2* __restrict__ out,
                                                 const cd2* __restrict__ tw, const int ax, const int inverse) {
    const long long stride = ax == 2 ? 1 : (ax == 1 ? (long long)g.N[2] : (long long)g.N[1] * g.N[2]);
    const int M = g.M[ax];
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < g.voxels; idx += (long long)gridDim.x * blockDim.x) {
        const int i2 = (int)(idx % g.N[2]);
        const long long row = idx / g.N[2];
        const int i1 = (int)(row % g.N[1]), i0 = (int)(row / g.N[1]);
        const int i = ax == 0 ? i0 : (ax == 1 ? i1 : i2);
        const int s = i / M, k = i - s * M;
        const long long base = idx - (long long)k * stride;       // first point of the subdomain line
        double sr = 0.0, si = 0.0;
        int j = 0;                                                 // (n k) mod M, updated incrementally
        for (int n = 0; n < M; ++n) {
            const cd2 a = in[base + (long long)n * stride];
            cd2 w = tw[j];
            if (inverse) w.y = -w.y;
            sr += a.x * w.x - a.y * w.y;
            si += a.x * w.y + a.y * w.x;
            j += k;
            if (j >= M) j -= M;
        }
        out[idx] = make_double2(sr, si);
    }
}

struct SymbolF64 {
    cd2 c, k02;
    double h, scale;
};

__device__ __forceinline__ double p2_of(int k, int M, double h) {
    const int f = (k < (M + 1) / 2) ? k : k - M;                  // fftfreq ordering (R9)
    const double p = 2.0 * 3.14159265358979323846 * (double)f / ((double)M * h);
    return p * p;
}

__global__ void __launch_bounds__(256) k_symbol_f64(const GridDesc g, cd2* __restrict__ u, const SymbolF64 sp, const int first_axis) {
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < g.voxels; idx += (long long)gridDim.x * blockDim.x) {
        const int i2 = (int)(idx % g.N[2]);
        const long long row = idx / g.N[2];
        const int i1 = (int)(row % g.N[1]), i0 = (int)(row / g.N[1]);
        double p2 = p2_of(i2 % g.M[2], g.M[2], sp.h);
        if (first_axis <= 1) p2 += p2_of(i1 % g.M[1], g.M[1], sp.h);
        if (first_axis <= 0) p2 += p2_of(i0 % g.M[0], g.M[0], sp.h);
        // D = c (k0^2 - p^2) + 1
        const cd2 D = zadd(zmul(sp.c, make_double2(sp.k02.x - p2, sp.k02.y)), make_double2(1.0, 0.0));
        const double inv = sp.scale / (D.x * D.x + D.y * D.y);
        u[idx] = zmul(u[idx], make_double2(D.x * inv, -D.y * inv));
    }
}

// d = x - u in complex128
__global__ void __launch_bounds__(256) k_dref_f64(const long long n, const cf* __restrict__ x, const cd2* __restrict__ u,
                                                  cd2* __restrict__ d) {
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (long long)gridDim.x * blockDim.x)
        d[idx] = make_double2((double)x[idx].x - u[idx].x, (double)x[idx].y - u[idx].y);
}

// complex128 -> complex64, rounded once
__global__ void __launch_bounds__(256) k_round_f64(const long long n, const cd2* __restrict__ in, cf* __restrict__ out) {
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n; idx += (long long)gridDim.x * blockDim.x)
        out[idx] = make_float2((float)in[idx].x, (float)in[idx].y);
}

static unsigned grid_for(long long n) {
    long long nb = (n + 255) / 256;
    if (nb > 148 * 32) nb = 148 * 32;
    return (unsigned)(nb < 1 ? 1 : nb);
}

// r_ref = B (x - (L+I)^-1 (B x + y_vec)), every step in complex128, rounded once to complex64 at the end (y may be nullptr)
cudaError_t launch_rref_f64(const GridDesc& g, const RefineF64& r, const cf* x, const cf* y, cf* rref, cudaStream_t st) {
    const unsigned nb = grid_for(g.voxels);
    const cd2 c = make_double2(r.c_re, r.c_im), ysc = make_double2(-r.c_re, -r.c_im);          // y_vec = -c y
    k_bxy_f64<cf><<<nb, 256, 0, st>>>(g, x, y, ysc, (const cd2*)r.bdiag, r.Kh, c, (cd2*)r.buf[0]);
    int cur = 0;
    for (int ax = 2; ax >= r.first_axis; --ax) {                                               // forward transforms
        k_dft_f64<<<nb, 256, 0, st>>>(g, (const cd2*)r.buf[cur], (cd2*)r.buf[cur ^ 1], (const cd2*)r.tw[ax], ax, 0);
        cur ^= 1;
    }
    SymbolF64 sp;
    sp.c = c; sp.k02 = make_double2(r.k02_re, r.k02_im); sp.h = r.h;
    sp.scale = 1.0 / ((double)g.M[0] * g.M[1] * g.M[2]);
    k_symbol_f64<<<nb, 256, 0, st>>>(g, (cd2*)r.buf[cur], sp, r.first_axis);
    for (int ax = r.first_axis; ax <= 2; ++ax) {                                               // inverse transforms
        k_dft_f64<<<nb, 256, 0, st>>>(g, (const cd2*)r.buf[cur], (cd2*)r.buf[cur ^ 1], (const cd2*)r.tw[ax], ax, 1);
        cur ^= 1;
    }
    k_dref_f64<<<nb, 256, 0, st>>>(g.voxels, x, (const cd2*)r.buf[cur], (cd2*)r.buf[cur ^ 1]);      // d_ref = x - u
    k_bxy_f64<cd2><<<nb, 256, 0, st>>>(g, (const cd2*)r.buf[cur ^ 1], nullptr, ysc, (const cd2*)r.bdiag, r.Kh, c, (cd2*)r.buf[cur]);   // B d_ref
    k_round_f64<<<nb, 256, 0, st>>>(g.voxels, (const cd2*)r.buf[cur], rref);
    return cudaGetLastError();
}

}  // namespace mbs
