"""Pins of oracle/mbs_oracle.py against what PAPER.md and the mathematics fix (no GPU).

Each test names the passage (P:NN = line of /root/reference/PAPER.md) or closed form it checks.
A plausible mistake in the oracle (dropped term, wrong sign or index, transposed operand) must
fail at least one of these.
"""
import os

import numpy as np
import pytest
from scipy import integrate

from oracle import mbs_oracle as orc
from paper_2410_02395_b200 import workloads
from tests import dense_reference as dr

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _small_oracle(shape, S, W, t, seed, periodic=None, h=0.25):
    n = workloads.random_medium(shape, seed, 1.0, 1.5, 0.02)
    return orc.MBSOracle(n, h, 1.0, W, S, periodic=periodic, n_correction=t)


# ------------------------------------------------------------------------------------------
# kernel K, K_t, ||A_12||
# ------------------------------------------------------------------------------------------
def test_kernel_is_bandlimited_second_derivative():
    """K[m] = (1/2pi) int_{-pi}^{pi} (-p^2) e^{i p m} dp (P:106 linear convolution with the angular
    spectrum kernel); checked by numerical quadrature, independent of the closed form."""
    for m in range(0, 9):
        val, _ = integrate.quad(lambda p: -p * p * np.cos(p * m) / (2 * np.pi), -np.pi, np.pi, limit=200)
        assert abs(orc.second_derivative_kernel(np.array([m]))[0] - val) < 1e-10
        assert abs(orc.second_derivative_kernel(np.array([-m]))[0] - val) < 1e-10


def test_alias_sum_equals_fft_circulant():
    """The circulant that a length-M FFT of -p^2 applies equals sum_q K[m + qM]."""
    M, h = 16, 1.0
    D2 = dr.block_second_derivative(M, h)
    assert np.abs(D2.imag).max() < 1e-12
    q = np.arange(-200000, 200001)
    for m in range(M):
        alias = orc.second_derivative_kernel(m + q * M).sum()
        assert abs(D2[m, 0].real - alias) < 2e-5


def test_Kt_golden_t4():
    """K_t for t = 4 (closed form -2(-1)^m/m^2 tabulated in SURVEY 8(c) step 5)."""
    gold = np.loadtxt(os.path.join(GOLD, "K_t4.txt"))
    assert np.allclose(orc.correction_matrix(4), gold, atol=6e-6)
    # exact rational entries
    K = orc.correction_matrix(4)
    assert K[3, 0] == pytest.approx(2.0)          # distance 1
    assert K[0, 0] == pytest.approx(-0.125)       # distance 4
    assert K[0, 3] == pytest.approx(-2.0 * -1 / 49.0)   # distance 7 -> +2/49


def test_sigma_max_values():
    """sigma_max(K_t) for t = 2, 4, 8, 16 and ||A_12|| = 34.866 at t = 8, h = 0.25."""
    gold = np.loadtxt(os.path.join(GOLD, "sigma_max.txt"))
    for t, s in gold:
        K = orc.correction_matrix(int(t))
        # power iteration on K^T K, independent of numpy's SVD
        v = np.ones(int(t))
        for _ in range(500):
            v = K.T @ (K @ v)
            v /= np.linalg.norm(v)
        sig = np.sqrt(v @ (K.T @ (K @ v)))
        assert sig == pytest.approx(s, abs=2e-5)
    o = _small_oracle((64,), (2,), (4,), 8, seed=1)
    assert o.norm_A12 == pytest.approx(34.866, abs=2e-3)


def test_corner_identity_P106():
    """bottom-left part of C_11 equals -A_12, top-right equals -A_12^T, where
    C_11 = (finite section of linear convolution) - (fast convolution on the subdomain) and
    A_12 is the off-diagonal block of the linear convolution.  Holds up to the |q| >= 2 aliases."""
    M, t, h = 32, 6, 1.0
    T = dr.toeplitz_second_derivative(2 * M, h)
    circ = dr.block_second_derivative(M, h).real
    C11 = T[:M, :M] - circ
    A12 = T[:M, M:]
    Kt = orc.correction_matrix(t)
    assert np.allclose(A12[M - t:, :t], Kt, atol=1e-14)               # truncated A_12 is K_t exactly
    bound = 2 * sum(2.0 / (q * M - M) ** 2 for q in range(2, 4000))   # dropped aliases
    assert np.abs(C11[M - t:, :t] + Kt).max() < bound
    assert np.abs(C11[:t, M - t:] + Kt.T).max() < bound
    assert np.abs(C11[M - t:, :t] + Kt).max() > 1e-6                  # and they are not zero: aliases exist


# ------------------------------------------------------------------------------------------
# scale factor
# ------------------------------------------------------------------------------------------
def test_eq9_reduces_to_eq4():
    """a_d = 0 (periodic, single domain) gives c = -0.95 i / ||k^2 - k0^2||_inf (Eq. (4))."""
    o = _small_oracle((32, 16), (1, 1), (0, 0), 0, seed=2, periodic=(1, 1))
    assert o.a == (0, 0)
    assert o.c == pytest.approx(-0.95j / o.v_max)
    assert abs(o.c.real) == 0.0


def test_eq9_a_d_values():
    """a_d = 1 for a single non-periodic domain, 2 when split; c shrinks accordingly."""
    o1 = _small_oracle((32, 32), (1, 1), (4, 4), 8, seed=3)
    o2 = _small_oracle((32, 32), (2, 1), (4, 4), 8, seed=3)
    o3 = _small_oracle((32, 32), (2, 2), (4, 4), 8, seed=3, periodic=(0, 1))
    assert o1.a == (1, 1) and o2.a == (2, 1) and o3.a == (2, 2)
    for o in (o1, o2, o3):
        # c is purely imaginary and |c| (v_max + sum_a ||A_12||) = 0.95; literal values of c are pinned in
        # test_scale_factor_literal_values
        assert o.c.real == 0.0 and o.c.imag < 0
        # convergence condition P:55: i c real and < 1 / ||k^2 - k0^2||_inf
        assert (1j * o.c).imag == pytest.approx(0.0)
        assert (1j * o.c).real < 1.0 / o.v_max
    assert abs(o2.c) < abs(o1.c)


def test_scale_factor_literal_values():
    """Eq. (4) and Eq. (9) on a medium whose numbers can be worked by hand, written out as literals
    (not the oracle's formula re-typed): lambda = 1, h = 1/4, n = 1 except one voxel with n = 2, no absorber.
      k^2 in {(2 pi)^2, 4 (2 pi)^2} = {39.4784176, 157.9136704};  k0^2 = 98.6960440 (R2: centre of the range);
      ||k^2 - k0^2||_inf = 59.2176264.
      periodic, one domain, t = 0:     c = -0.95 i / 59.2176264               = -0.0160425207 i       (Eq. (4))
      two subdomains, t = 8:           ||A_12|| = 2.17915 / h^2 = 34.8664 (sigma_max printed in SURVEY 8(c) step 6),
                                       c = -0.95 i / (59.2176264 + 2 * 34.8664) = -0.00736718 i       (Eq. (9), a = 2)
      one non-periodic domain, t = 8:  c = -0.95 i / (59.2176264 + 1 * 34.8664) = -0.0100974 i        (a = 1)"""
    n = np.ones(32, dtype=np.complex64)
    n[11] = 2.0
    o = orc.MBSOracle(n, 0.25, 1.0, (0,), (1,), periodic=(1,), n_correction=0)
    assert o.k02 == pytest.approx(98.6960440, rel=1e-8)
    assert o.v_max == pytest.approx(59.2176264, rel=1e-8)
    assert o.c.real == 0.0 and o.c.imag == pytest.approx(-0.0160425207, rel=1e-8)
    o2 = orc.MBSOracle(n, 0.25, 1.0, (0,), (2,), n_correction=8)
    assert o2.c.real == 0.0 and o2.c.imag == pytest.approx(-0.00736718, rel=2e-5)
    o1 = orc.MBSOracle(n, 0.25, 1.0, (0,), (1,), n_correction=8)
    assert o1.c.real == 0.0 and o1.c.imag == pytest.approx(-0.0100974, rel=2e-5)


def test_absorber_weight_is_max_over_axes_2d():
    """R3: w(r) = max_d w_d(r).  2-D, n = 1, W = (8, 4): at pixel (2, 3) the two ramps give 6/8 and 1/4, at (6, 0)
    they give 2/8 and 1; the layer adds i 0.5 (2 pi)^2 max(...) to k^2 (a sum would give 1.0 and 1.25, a product
    0.1875 and 0.25)."""
    o = orc.MBSOracle(np.ones((32, 24), dtype=np.complex64), 0.25, 1.0, (8, 4), (1, 1), n_correction=4)
    kw2 = 39.47841760435743
    assert o.k2[2, 3].imag == pytest.approx(0.5 * kw2 * 0.75, rel=1e-12)
    assert o.k2[6, 0].imag == pytest.approx(0.5 * kw2 * 1.0, rel=1e-12)
    assert o.k2[29, 20].imag == pytest.approx(0.5 * kw2 * 0.75, rel=1e-12)      # mirrored: (32-1-29, 24-1-20) = (2, 3)
    assert o.k2[16, 12].imag == 0.0


def test_first_update_is_alpha_times_preconditioned_source():
    """P:76 Eq. (6) with x^(0) = 0: x^(1) = alpha B (L+I)^-1 y_vec, alpha = 0.75 (Eq. (4)), y_vec = -c y.
    The right-hand side is assembled from the dense matrices of tests/dense_reference.py with the literal 0.75."""
    shape, S, t = (16, 12), (2, 1), 4
    o = _small_oracle(shape, S, (2, 2), t, seed=41)
    L, V = dr.assemble(o.k2, o.k02, o.c, shape, S, t, o.h, o.a, (0, 0))
    I = np.eye(L.shape[0])
    rng = np.random.default_rng(3)
    y = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    x1_dense = 0.75 * (I - V) @ np.linalg.solve(L + I, (-o.c * y).reshape(-1))
    x1, hist = o.solve(y, tol=0.0, max_iter=1)
    assert len(hist) == 1 and hist[0] == pytest.approx(1.0, abs=1e-13)
    assert np.linalg.norm(x1.reshape(-1) - x1_dense) / np.linalg.norm(x1_dense) < 1e-12
    # and the second update follows Eq. (6) from x^(1) with the same alpha
    x1v = x1_dense
    r = (I - V) @ (x1v - np.linalg.solve(L + I, (-o.c * y).reshape(-1) + (I - V) @ x1v))
    x2_dense = x1v - 0.75 * r
    x2, _ = o.solve(y, tol=0.0, max_iter=2)
    assert np.linalg.norm(x2.reshape(-1) - x2_dense) / np.linalg.norm(x2_dense) < 1e-12


def test_k0_minimises_vmax_box():
    """R2: k0^2 is the centre of the bounding box of k^2 (after the absorber)."""
    o = _small_oracle((40,), (1,), (6,), 4, seed=4)
    assert o.k02.real == pytest.approx(0.5 * (o.k2.real.min() + o.k2.real.max()))
    assert o.k02.imag == pytest.approx(0.5 * (o.k2.imag.min() + o.k2.imag.max()))
    # absorber: linear ramp, 1 at the outermost pixel, beta = 0.5 (R3)
    n = np.ones(40, dtype=np.complex64)
    oh = orc.MBSOracle(n, 0.25, 1.0, (8,), (1,), n_correction=4)
    kw2 = (2 * np.pi) ** 2
    assert oh.k2[0].imag == pytest.approx(0.5 * kw2)
    assert oh.k2[39].imag == pytest.approx(0.5 * kw2)
    assert oh.k2[7].imag == pytest.approx(0.5 * kw2 / 8)
    assert oh.k2[32].imag == pytest.approx(0.5 * kw2 / 8)
    assert oh.k2[8].imag == 0.0 and oh.k2[31].imag == 0.0
    assert np.allclose(oh.k2.real, kw2)


# ------------------------------------------------------------------------------------------
# matrix-free operators vs dense assembly from the definitions
# ------------------------------------------------------------------------------------------
DENSE_CASES = [
    ((16,), (1,), (2,), 4, None),
    ((16,), (2,), (2,), 3, None),
    ((24,), (3,), (2,), 4, (1,)),
    ((16, 12), (2, 1), (2, 2), 4, None),
    ((16, 12), (2, 2), (2, 2), 3, None),
    ((12, 16), (1, 2), (2, 0), 4, (0, 1)),
    ((8, 6, 6), (2, 1, 1), (1, 1, 1), 3, None),
    ((8, 6, 8), (2, 1, 2), (1, 1, 1), 2, (0, 1, 0)),
]


@pytest.mark.parametrize("shape,S,W,t,periodic", DENSE_CASES)
def test_operators_match_dense_assembly(shape, S, W, t, periodic):
    o = _small_oracle(shape, S, W, t, seed=10 + len(shape), periodic=periodic)
    per = periodic if periodic is not None else (0,) * len(shape)
    L, V = dr.assemble(o.k2, o.k02, o.c, shape, S, t, o.h, o.a, per)
    N = L.shape[0]
    I = np.eye(N)
    rng = np.random.default_rng(5)
    u = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    uf = u.reshape(-1)

    def rel(a, b):
        return np.linalg.norm(a.reshape(-1) - b) / np.linalg.norm(b)

    assert rel(o.apply_V(u), V @ uf) < 1e-12
    assert rel(o.apply_B(u), (I - V) @ uf) < 1e-12
    assert rel(o.apply_L_plus_1(u), (L + I) @ uf) < 1e-12
    assert rel(o.propagate(u), np.linalg.solve(L + I, uf)) < 1e-11
    assert rel(o.apply_A(u), (L + V) @ uf) < 1e-12
    G_inv_A = (I - V) @ np.linalg.solve(L + I, L + V)
    assert rel(o.apply_precond_A(u), G_inv_A @ uf) < 1e-11
    # ||V|| < 1 for the estimate of Eq. (9)
    assert np.linalg.norm(V, 2) < 1.0


@pytest.mark.parametrize("shape,S,W,t", [
    ((16, 12), (1, 1), (2, 2), 4),
    ((16, 12), (2, 1), (2, 2), 4),
    ((16, 12), (2, 2), (2, 2), 4),
    ((8, 6, 6), (2, 1, 1), (1, 1, 1), 3),
])
def test_fixed_point_is_dense_direct_solve(shape, S, W, t):
    """the limit of Eq. (6) solves A x = y_vec, y_vec = -c y."""
    o = _small_oracle(shape, S, W, t, seed=21)
    L, V = dr.assemble(o.k2, o.k02, o.c, shape, S, t, o.h, o.a, (0,) * len(shape))
    y = np.zeros(shape, dtype=np.complex128)
    y[tuple(s // 3 for s in shape)] = 1.0
    x_direct = np.linalg.solve(L + V, (-o.c * y).reshape(-1)).reshape(shape)
    x, hist = o.solve(y, tol=1e-11, max_iter=20000)
    assert hist[-1] < 1e-11
    assert np.linalg.norm(x - x_direct) / np.linalg.norm(x_direct) < 1e-9
    # eps_0 = 1 for a cold start (R8) and monotone non-increase
    assert hist[0] == pytest.approx(1.0, abs=1e-13)
    assert np.all(np.diff(hist) <= 1e-15)


def test_warm_start_converges_to_same_field():
    """the MBS converges to the correct solution from any starting point."""
    shape, S = (32,), (2,)
    o = _small_oracle(shape, S, (4,), 4, seed=22)
    y = np.zeros(shape, dtype=np.complex128)
    y[5] = 1.0
    x, _ = o.solve(y, tol=1e-11, max_iter=20000)
    rng = np.random.default_rng(0)
    x0 = x + 0.1 * (rng.standard_normal(shape) + 1j * rng.standard_normal(shape))
    x2, hist2 = o.solve(y, x0=x0, tol=1e-11, max_iter=20000)
    assert np.linalg.norm(x2 - x) / np.linalg.norm(x) < 1e-9
    assert np.all(np.diff(hist2) <= 1e-15)


# ------------------------------------------------------------------------------------------
# full (untruncated) correction reproduces the finite-section linear convolution
# ------------------------------------------------------------------------------------------
def test_full_correction_recovers_linear_convolution():
    """P:100 "the system being solved here is still the same": with t = M the decomposed A equals
    c [T/h^2 + diag k^2] (T = finite section of the linear convolution) up to the |q| >= 2 aliases."""
    N, S, h = 32, 2, 0.25
    M = N // S
    o = _small_oracle((N,), (S,), (2,), M, seed=30, h=h)
    T = dr.toeplitz_second_derivative(N, h)
    A_exact = o.c * (T + np.diag(o.k2))
    A_or = np.stack([o.apply_A(e) for e in np.eye(N, dtype=np.complex128)], axis=1)
    alias_bound = abs(o.c) / h ** 2 * 2 * sum(2.0 / (q * M - M) ** 2 for q in range(2, 4000))
    assert np.abs(A_or - A_exact).max() < alias_bound
    # a sign or placement error would be O(|c| K[1] / h^2), far above the alias bound
    assert alias_bound < 0.1 * abs(o.c) * 2.0 / h ** 2


# ------------------------------------------------------------------------------------------
# closed-form Green's function
# ------------------------------------------------------------------------------------------
def _green_error(S, t, periodic, N=1024, W=128, beta=0.3, n_val=1.0):
    h, lam = 0.25, 1.0
    n = np.full(N, n_val, dtype=np.complex64)
    o = orc.MBSOracle(n, h, lam, (W,), (S,), periodic=(periodic,), n_correction=t, beta=beta)
    y = np.zeros(N, dtype=np.complex128)
    src = N // 2 - 37
    y[src] = 1.0 / h
    x, hist = o.solve(y, tol=1e-9, max_iter=50000)
    k = 2 * np.pi * n_val / lam
    r = (np.arange(N) - src) * h
    exact = 1j / (2 * k) * np.exp(1j * k * np.abs(r))
    roi = np.zeros(N, dtype=bool)
    roi[W:N - W] = True
    roi[src - 8:src + 9] = False
    return np.linalg.norm(x[roi] - exact[roi]) / np.linalg.norm(exact[roi]), hist


def test_green_function_1d_undecomposed():
    """BASELINE.json north_star: 1D homogeneous medium, x(r) = (i/2k) e^{ik|r|} away from source and absorber
    for [d^2/dr^2 + k^2] x = -delta(r) (Eq. (1))."""
    err, hist = _green_error(S=1, t=0, periodic=1)
    assert err < 2e-3
    assert np.all(np.diff(hist) <= 1e-15)


def test_green_function_1d_in_a_medium_of_index_1p33():
    """the wavenumber is k = 2 pi n / lambda, i.e. k^2 = (2 pi / lambda)^2 n^2 (oracle step 1).  In a homogeneous
    medium of n = 1.33 the field of a point source is (i/2k) e^{ik|r|} with k = 2 pi 1.33 / lambda; k^2 proportional to
    n (or to anything but n^2) gives another wavelength and amplitude and fails by O(1)."""
    err, hist = _green_error(S=1, t=0, periodic=1, n_val=1.33)
    assert err < 3e-3
    assert np.all(np.diff(hist) <= 1e-15)
    # control: the closed form with the wavenumber of n = 1 does not fit this field (the pin can tell them apart)
    h, N, W = 0.25, 1024, 128
    o = orc.MBSOracle(np.full(N, 1.33, dtype=np.complex64), h, 1.0, (W,), (1,), periodic=(1,), n_correction=0, beta=0.3)
    assert o.k2[N // 2] == pytest.approx((2 * np.pi * 1.33) ** 2, rel=1e-6)


def test_green_function_1d_two_domains_full_correction():
    """Same closed form through the domain decomposition with untruncated corrections (t = M):
    pins signs and placement of C_ss and A_{s,s+-1}."""
    err, _ = _green_error(S=2, t=512, periodic=0)
    assert err < 2e-3


def test_truncation_error_decays_with_t():
    """P:173, Fig. 6a: error w.r.t. the exact field decays with the number of correction points."""
    e8, _ = _green_error(S=2, t=8, periodic=0)
    e32, _ = _green_error(S=2, t=32, periodic=0)
    assert e32 < e8 < 0.1
    assert e8 > 2e-3


# ------------------------------------------------------------------------------------------
# BASELINE.json config 1 end to end
# ------------------------------------------------------------------------------------------
def test_config1_iterations_and_split_ratio():
    """P:183 (1751/1160 = 1.51 when an axis is split), P:175 (iterations independent of t >= 4)."""
    w = workloads.config(1)
    n, y = w.make_medium(), w.make_source()
    o2 = orc.from_workload(w, n)
    x2, h2 = o2.solve(y, tol=w.tol, max_iter=w.max_iter)
    assert h2[-1] < w.tol and np.all(np.diff(h2) <= 1e-15)
    o1 = orc.MBSOracle(n, w.pixel_size, w.wavelength, w.boundary_width, (1,), n_correction=8)
    x1, h1 = o1.solve(y, tol=w.tol, max_iter=w.max_iter)
    ratio = len(h2) / len(h1)
    assert 1.35 < ratio < 1.75
    o2b = orc.MBSOracle(n, w.pixel_size, w.wavelength, w.boundary_width, (2,), n_correction=16)
    _, h2b = o2b.solve(y, tol=w.tol, max_iter=w.max_iter)
    assert abs(len(h2b) - len(h2)) < 0.05 * len(h2)
    # the two decompositions solve the same problem up to the truncation (1.7e-4 squared metric)
    err_sq = np.linalg.norm(x2 - x1) ** 2 / np.linalg.norm(x1) ** 2
    assert err_sq < 5e-3


# ------------------------------------------------------------------------------------------
# subdomain activation (reading R17 in DESIGN.md section 3)
# ------------------------------------------------------------------------------------------
def _activation_case():
    N = 512
    n = np.ones(N, dtype=np.complex64)
    n[200:260] = 1.3 + 0.01j
    o = orc.MBSOracle(n, 0.25, 1.0, (16,), (4,), n_correction=8)
    y = np.zeros(N, dtype=np.complex128)
    y[40] = 1.0
    return o, y


def test_activation_threshold_zero_is_the_plain_iteration():
    """R17: with threshold 0 every subdomain is active from n = 0, and the activated iteration IS Eq. (6)."""
    o, y = _activation_case()
    x0, h0 = o.solve(y, tol=1e-4, max_iter=20000)
    x1, h1, act = orc.solve_activated(o, y, tol=1e-4, max_iter=20000, threshold=0.0)
    assert act == [0, 0, 0, 0]
    assert np.array_equal(x1, x0) and np.array_equal(h1, h0)


def test_activation_converges_to_the_same_field():
    """"Although this initially causes a small error, the MBS converges to the correct solution from any
    starting point and thus nullifies these errors."  Only the source-holding subdomain starts active; the others
    follow in order of their distance from the source; the converged field agrees with the plain iteration far below
    the stopping threshold and the iteration count is unchanged within 1 %; work is saved (12 % in the paper)."""
    o, y = _activation_case()
    tol = 1e-4
    x0, h0 = o.solve(y, tol=tol, max_iter=20000)
    held = {}

    def cb(n, eps, x):
        # subdomains 2 and 3 hold exactly zero until they are activated
        held[n] = (bool(np.all(x[256:384] == 0)), bool(np.all(x[384:512] == 0)))

    x1, h1, act = orc.solve_activated(o, y, tol=tol, max_iter=20000, callback=cb)
    assert act[0] == 0 and all(a > 0 for a in act[1:])
    assert act[1] <= act[2] <= act[3]                      # the field reaches them in order of distance
    assert all(held[n][0] for n in range(act[2] - 1)) and not held[act[2]][0]
    assert all(held[n][1] for n in range(act[3] - 1)) and not held[act[3]][1]
    assert np.linalg.norm(x1 - x0) / np.linalg.norm(x0) < 0.1 * tol
    assert abs(len(h1) - len(h0)) <= 0.01 * len(h0)
    saved = 1.0 - sum(len(h1) - a for a in act) / (len(act) * len(h1))
    assert saved > 0.01
    # a larger threshold delays activation and saves more work; the field still agrees at the level of the threshold
    x2, h2, act2 = orc.solve_activated(o, y, tol=tol, max_iter=20000, threshold=10 * tol)
    assert all(b >= a for a, b in zip(act, act2)) and act2[3] > act[3]
    assert np.linalg.norm(x2 - x0) / np.linalg.norm(x0) < 30 * tol


def test_activation_rule_against_dense_transfer_norm():
    """R17 rule, checked against the dense correction matrices of tests/dense_reference.py: an inactive subdomain s is
    activated before the first update n at which sqrt(sum_d ||(c C_d x^(n))_s||^2) >= threshold * nu, where C_d holds the
    K_t entries placed by index and nu = ||B (L+I)^-1 y_vec||."""
    shape, S, t = (16, 12), (2, 2), 3
    o = _small_oracle(shape, S, (2, 2), t, seed=51)
    L, V = dr.assemble(o.k2, o.k02, o.c, shape, S, t, o.h, o.a, (0, 0))
    I = np.eye(L.shape[0])
    Cd = [o.c * dr.kron_axis(dr.axis_correction_matrix(shape[d], S[d], t, o.h, False), shape, d) for d in range(2)]
    y = np.zeros(shape, dtype=np.complex128)
    y[2, 2] = 1.0                                           # subdomain (0, 0)
    nu = np.linalg.norm((I - V) @ np.linalg.solve(L + I, (-o.c * y).reshape(-1)))
    thr = 3e-2
    xs = {}
    x, hist, act = orc.solve_activated(o, y, tol=1e-6, max_iter=400, threshold=thr,
                                       callback=lambda n, eps, xx: xs.__setitem__(n + 1, xx.copy()))
    xs[0] = np.zeros(shape, dtype=np.complex128)
    blocks = [(slice(0, 8), slice(0, 6)), (slice(0, 8), slice(6, 12)), (slice(8, 16), slice(0, 6)), (slice(8, 16), slice(6, 12))]
    assert act[0] == 0 and all(a > 0 for a in act[1:])
    for k in range(1, 4):
        def T(n):
            return np.sqrt(sum(np.linalg.norm((C @ xs[n].reshape(-1)).reshape(shape)[blocks[k]]) ** 2 for C in Cd))
        assert T(act[k]) >= thr * nu                        # activated when the transferred norm reaches the threshold
        assert all(T(n) < thr * nu for n in range(act[k]))  # ... and not before


# ------------------------------------------------------------------------------------------
# batched solves (reading R18 in DESIGN.md section 3)
# ------------------------------------------------------------------------------------------
def test_batch_is_independent_solves_with_a_stacked_residual():
    """R18: the sources do not couple (each x_b^(n) is the n-th iterate of its own Eq. (6)), and the one residual
    of the stacked block-diagonal system is eps_n^2 = sum_b eps_{b,n}^2 nu_b^2 / sum_b nu_b^2 (P:130 applied to it)."""
    shape, S, t = (16, 12), (2, 1), 4
    o = _small_oracle(shape, S, (2, 2), t, seed=61)
    rng = np.random.default_rng(7)
    ys = [rng.standard_normal(shape) + 1j * rng.standard_normal(shape) for _ in range(3)]
    ys[1] = np.zeros(shape, dtype=np.complex128)
    ys[1][3, 4] = 1.0                                   # one sparse source among dense ones
    n_it = 25
    xs, hist = orc.solve_batch(o, ys, tol=0.0, max_iter=n_it)
    singles = [o.solve(y, tol=0.0, max_iter=n_it) for y in ys]
    L, V = dr.assemble(o.k2, o.k02, o.c, shape, S, t, o.h, o.a, (0, 0))
    I = np.eye(L.shape[0])
    nus = [np.linalg.norm((I - V) @ np.linalg.solve(L + I, (-o.c * y).reshape(-1))) for y in ys]   # dense, independent
    for b in range(3):
        assert np.linalg.norm(xs[b] - singles[b][0]) <= 1e-13 * np.linalg.norm(singles[b][0])
    stacked = np.sqrt(sum((singles[b][1] * nus[b]) ** 2 for b in range(3)) / sum(nu ** 2 for nu in nus))
    assert np.allclose(hist, stacked, rtol=1e-11)
    assert hist[0] == pytest.approx(1.0, abs=1e-12)     # cold start: eps_0 = 1 for the stacked system too
    # the stop test acts on the stacked residual: every source gets the same number of updates
    xs2, hist2 = orc.solve_batch(o, ys, tol=1e-3, max_iter=5000)
    assert hist2[-1] < 1e-3 and np.all(hist2[:-1] >= 1e-3)
    for b in range(3):
        xb, _ = o.solve(ys[b], tol=0.0, max_iter=len(hist2))
        assert np.linalg.norm(xs2[b] - xb) <= 1e-13 * np.linalg.norm(xb)
