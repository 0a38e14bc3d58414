"""CPU oracle for the domain-decomposed modified Born series (TEST INFRASTRUCTURE, not product).

A plain, slow, double-precision (complex128) restatement of what the hot path computes, written
from /root/reference/PAPER.md (arxiv 2410.02395, Mache & Vellekoop).  `P:NN` below is a line of
that file.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl
reference` legs may import this module; the product (paper_2410_02395_b200/) never does, and this
module imports nothing from the product.  It shares no code, table or constant with the CUDA path.

The method is an iteration (Eq. (6)) that converges to the solution of A x = y (Eq. (2),
P:100), so the oracle provides (i) every operator as the closed-form linear map the paper defines
and (ii) the iteration step by step in the paper's order.  A library FFT (scipy.fft) serves as
the "fast Fourier transform" of P:66; nothing is blocked, fused or reordered.

Readings of points the paper leaves open (listed in DESIGN.md section 3, after SURVEY.md 8(c)):
  R1  iteration = Eq. (6) of PAPER.md, not the shorthand in BASELINE.json.
  R2  k0^2 = midpoint of the bounding box of k^2(r) in the complex plane, after the absorber.
  R3  absorbing layer = linear ramp in Im k^2, beta = 0.5 (stand-in for ref [3]).
  R4  A_12 from the closed-form band-limited second-derivative kernel, nearest alias, t x t corner.
  R5  ||A_12|| = sigma_max of that t x t matrix in physical units (1/h^2).
  R7  residual normalised by the global ||Gamma^-1 y||.
  R8  eps_n belongs to x^(n); the update is applied before the stop test.
  R9  p = 2 pi fftfreq(M, h); forward unnormalised, inverse 1/M.
  R17 subdomain activation (the paper gives neither the norm nor the threshold): see solve_activated.
  R18 batched solves ("solving each frequency separately"; several sources sharing one medium): see solve_batch.

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): printed K_t / sigma_max values, Eq. (9) -> Eq. (4),
dense assembly from explicit DFT matrices, dense direct solve, monotone residual, eps_0 = 1,
closed-form 1D Green's function (n = 1 and n = 1.33), full-correction identity, corner identity of P:106, literal values of c,
alpha through the first two updates, the 2-D absorber corner, the activation rule (R17) and the stacked batch residual (R18).
The converged fields of the five synthetic BASELINE.json media have no value printed in the paper:
for them "parity unpinned" beyond those invariants (last row).
"""
from __future__ import annotations

import os

import numpy as np
import scipy.fft as sfft

ALPHA = 0.75          # P:59 Eq. (4)
SCALE_095 = 0.95      # P:59 Eq. (4), Eq. (9)
BETA_ABSORB = 0.5     # reading R3


def _workers():
    return max(1, os.cpu_count() or 1)


def second_derivative_kernel(m):
    """Band-limited second derivative on the infinite grid, in units of 1/h^2 ("the angular
    spectrum kernel applied ... using a linear convolution", for -p^2 on |p| <= pi/h):
    K[0] = -pi^2/3, K[m] = -2 (-1)^m / m^2."""
    m = np.asarray(m, dtype=np.int64)
    out = np.empty(m.shape, dtype=np.float64)
    zero = (m == 0)
    out[zero] = -np.pi ** 2 / 3.0
    mm = m[~zero].astype(np.float64)
    out[~zero] = -2.0 * np.where(m[~zero] % 2 == 0, 1.0, -1.0) / (mm * mm)
    return out


def correction_matrix(t):
    """K_t[a, b] = K[t + b - a]  (reading R4; "bottom-left part of A_12", "square blocks
    of size t").  Row a = a-th of the LAST t points of a block, column b = b-th of the FIRST t
    points of the next block; their distance is (M + b) - (M - t + a) = t + b - a."""
    a = np.arange(t)[:, None]
    b = np.arange(t)[None, :]
    return second_derivative_kernel(t + b - a)


class MBSOracle:
    """Setup (steps 1-9 of SURVEY.md 8(c)) and operators (steps 10-13) for one medium."""

    def __init__(self, n_map, pixel_size, wavelength, boundary_width, n_subdomains,
                 periodic=None, n_correction=8, beta=BETA_ABSORB):
        n_map = np.asarray(n_map).astype(np.complex128)
        self.shape = n_map.shape
        self.ndim = D = n_map.ndim
        self.h = float(pixel_size)
        self.wavelength = float(wavelength)
        self.W = tuple(int(w) for w in boundary_width)
        self.S = tuple(int(s) for s in n_subdomains)
        self.periodic = tuple(int(p) for p in (periodic if periodic is not None else (0,) * D))
        self.t = int(n_correction)
        assert len(self.W) == D and len(self.S) == D and len(self.periodic) == D
        for d in range(D):
            assert self.shape[d] % self.S[d] == 0
        self.M = tuple(self.shape[d] // self.S[d] for d in range(D))

        kw = 2.0 * np.pi / self.wavelength
        # 1. k^2(r) = (2 pi / lambda)^2 n(r)^2   (P:41 wavenumber, P:147 refractive index)
        k2 = (kw ** 2) * n_map * n_map
        # 2. absorbing layer (R3): k^2 += i beta (2 pi/lambda)^2 w(r), linear ramp, 1 at the outermost pixel
        w = np.zeros(self.shape, dtype=np.float64)
        for d in range(D):
            Wd, Nd = self.W[d], self.shape[d]
            if Wd <= 0:
                continue
            prof = np.zeros(Nd, dtype=np.float64)
            i = np.arange(Wd)
            ramp = (Wd - i) / float(Wd)
            prof[:Wd] = ramp
            prof[Nd - Wd:] = np.maximum(prof[Nd - Wd:], ramp[::-1])
            sh = [1] * D
            sh[d] = Nd
            w = np.maximum(w, prof.reshape(sh))
        k2 = k2 + 1j * beta * (kw ** 2) * w
        self.k2 = k2
        # 3. k0^2 (R2) and v_max = ||k^2 - k0^2||_inf
        self.k02 = 0.5 * (k2.real.min() + k2.real.max()) + 0.5j * (k2.imag.min() + k2.imag.max())
        self.v_max = float(np.abs(k2 - self.k02).max())
        # 4-6. K_t and ||A_12|| = sigma_max(K_t) / h^2
        if self.t > 0:
            self.K_t = correction_matrix(self.t)
            self.norm_A12 = float(np.linalg.svd(self.K_t, compute_uv=False)[0]) / self.h ** 2
        else:
            self.K_t = np.zeros((0, 0))
            self.norm_A12 = 0.0
        # 7. a_d
        a = []
        for d in range(D):
            if self.S[d] >= 2:
                a.append(2)
            elif self.periodic[d]:
                a.append(0)
            else:
                a.append(1)
        if self.t == 0:
            assert all(ad == 0 for ad in a), "t = 0 is legal only for periodic single-domain axes"
        self.a = tuple(a)
        # 8. c (Eq. (9); Eq. (4) when all a_d = 0)
        self.c = -1j * SCALE_095 / (self.v_max + sum(self.a) * self.norm_A12)
        # 9. A_12 = c K_t / h^2; B_diag = 1 - c (k^2 - k0^2); g(p) = 1 / (c (k0^2 - |p|^2) + 1)
        self.A12 = self.c * self.K_t / self.h ** 2
        self.B_diag = 1.0 - self.c * (k2 - self.k02)
        p2 = np.zeros(self.M, dtype=np.float64)
        for d in range(D):
            pd = 2.0 * np.pi * np.fft.fftfreq(self.M[d], self.h)
            sh = [1] * D
            sh[d] = self.M[d]
            p2 = p2 + (pd ** 2).reshape(sh)
        self.L_plus_1_hat = self.c * (self.k02 - p2) + 1.0     # symbol of L + I on one subdomain
        self.g = 1.0 / self.L_plus_1_hat

    # ---- step 10: edge corrections along one axis -------------------------------------------
    def corr_axis(self, u, d):
        """corr_d(u) (P:124-128 steps 1, 2, 4, 5 read with P:106).  For subdomain s along axis d:
        l_s = A12 u_s[0:t], rho_s = A12^T u_s[M-t:M];
        corr_s[M-t:M] = -l_s + l_{s+1};  corr_s[0:t] = -rho_s + rho_{s-1};
        a neighbour outside a non-periodic grid contributes 0; periodic axes wrap."""
        out = np.zeros_like(u)
        if self.a[d] == 0 or self.t == 0:
            return out
        t, M, S = self.t, self.M[d], self.S[d]
        um = np.moveaxis(u, d, 0)
        om = np.moveaxis(out, d, 0)
        ell, rho = [], []
        for s in range(S):
            first = um[s * M: s * M + t]
            last = um[(s + 1) * M - t: (s + 1) * M]
            ell.append(np.tensordot(self.A12, first, axes=(1, 0)))
            rho.append(np.tensordot(self.A12.T, last, axes=(1, 0)))
        for s in range(S):
            hi = -ell[s]
            if s + 1 < S:
                hi = hi + ell[s + 1]
            elif self.periodic[d]:
                hi = hi + ell[0]
            lo = -rho[s]
            if s - 1 >= 0:
                lo = lo + rho[s - 1]
            elif self.periodic[d]:
                lo = lo + rho[S - 1]
            om[(s + 1) * M - t: (s + 1) * M] += hi
            om[s * M: s * M + t] += lo
        return out

    # ---- step 11 -------------------------------------------------------------------------------
    def apply_V(self, u):
        """V u = c (k^2 - k0^2) u + sum_d corr_d(u)  (Eq. (8))."""
        out = (1.0 - self.B_diag) * u
        for d in range(self.ndim):
            out = out + self.corr_axis(u, d)
        return out

    def apply_B(self, u):
        """B u = (I - V) u."""
        return u - self.apply_V(u)

    # ---- step 12 -------------------------------------------------------------------------------
    def _blockwise(self, u, symbol):
        out = np.empty_like(u)
        axes = tuple(range(self.ndim))
        for idx in np.ndindex(*self.S):
            sl = tuple(slice(i * m, (i + 1) * m) for i, m in zip(idx, self.M))
            blk = sfft.fftn(u[sl], axes=axes, workers=_workers())
            blk *= symbol
            out[sl] = sfft.ifftn(blk, axes=axes, workers=_workers())
        return out

    def propagate(self, u):
        """(L + I)^-1 u: per subdomain FFT, multiply by g, inverse FFT."""
        return self._blockwise(u, self.g)

    def apply_L_plus_1(self, u):
        """(L + I) u: same with 1/g (Eq. (5))."""
        return self._blockwise(u, self.L_plus_1_hat)

    # ---- step 13 -------------------------------------------------------------------------------
    def apply_A(self, u):
        """A u = (L + I) u - B u."""
        return self.apply_L_plus_1(u) - self.apply_B(u)

    def apply_precond_A(self, u):
        """Gamma^-1 A u = B u - B (L+I)^-1 B u  (from Gamma^-1 = B (L+I)^-1 and A = (L+I) - B)."""
        return self.apply_B(u - self.propagate(self.apply_B(u)))

    # ---- steps 14-15: the iteration ------------------------------------------------------------
    def solve(self, y, x0=None, tol=1e-6, max_iter=1000, callback=None):
        """Eq. (6) with the stop test of P:130.  Returns (x, residual_history).
        y is the physical source of Eq. (1); y_vec = -c y.  history[n] = eps_n of x^(n)."""
        y_vec = -self.c * np.asarray(y).astype(np.complex128)
        x = np.zeros(self.shape, dtype=np.complex128) if x0 is None else np.asarray(x0).astype(np.complex128).copy()
        nu = np.linalg.norm(self.apply_B(self.propagate(y_vec)))
        history = []
        for n in range(max_iter):
            u = self.propagate(self.apply_B(x) + y_vec)
            r = self.apply_B(x - u)
            eps = float(np.linalg.norm(r) / nu)
            history.append(eps)
            x = x - ALPHA * r
            if callback is not None:
                callback(n, eps, x)
            if eps < tol:
                break
        return x, np.asarray(history)


# ---- subdomain activation, reading R17 --------------------------------------------------
def _subdomain_slices(o):
    return [tuple(slice(i * m, (i + 1) * m) for i, m in zip(idx, o.M)) for idx in np.ndindex(*o.S)]


def solve_activated(o, y, x0=None, tol=1e-6, max_iter=1000, threshold=None, callback=None):
    """Eq. (6) with the activation strategy of P:139-141: "initially activating only those subdomains that hold
    a source term.  Neighbouring subdomains are activated only after the norm of the transferred field exceeds a
    certain threshold."  The paper fixes neither the norm nor the threshold; reading R17:

      * a subdomain is active from the start if y or x^(0) is non-zero anywhere in it;
      * before update n, an inactive subdomain s becomes active (and stays so) if
            T_s := sqrt( sum_d || (corr_d x^(n)) restricted to s ||_2^2 )  >=  threshold * nu,
        corr_d = the edge corrections of step 10 (an inactive subdomain holds x_s = 0, so what lands in it is exactly
        the field its neighbours transfer, P:126 step 2), nu = ||Gamma^-1 y_vec|| the normalisation of the residual
        (P:130).  Default threshold = tol / 10: what an inactive subdomain would add to the relative residual stays an
        order of magnitude below the stopping threshold;
      * an inactive subdomain is not computed: it contributes d_s = 0, receives no update and no residual.
    threshold = 0 activates every subdomain at n = 0 and reproduces `solve` exactly.
    Returns (x, residual_history, activation_iteration per subdomain in np.ndindex(S) order; -1 = never)."""
    if threshold is None:
        threshold = 0.1 * tol
    y_vec = -o.c * np.asarray(y).astype(np.complex128)
    x = np.zeros(o.shape, dtype=np.complex128) if x0 is None else np.asarray(x0).astype(np.complex128).copy()
    nu = np.linalg.norm(o.apply_B(o.propagate(y_vec)))
    blocks = _subdomain_slices(o)
    active = [bool(np.any(y_vec[sl] != 0) or np.any(x[sl] != 0)) for sl in blocks]
    activated_at = [0 if a else -1 for a in active]
    history = []
    for n in range(max_iter):
        if not all(active):
            corr = [o.corr_axis(x, d) for d in range(o.ndim)]
            for k, sl in enumerate(blocks):
                if not active[k]:
                    T = np.sqrt(sum(np.linalg.norm(cd[sl]) ** 2 for cd in corr))
                    if T >= threshold * nu:
                        active[k] = True
                        activated_at[k] = n
        mask = np.zeros(o.shape, dtype=np.float64)
        for k, sl in enumerate(blocks):
            if active[k]:
                mask[sl] = 1.0
        u = o.propagate(o.apply_B(x) + y_vec)
        d = (x - u) * mask
        r = o.apply_B(d) * mask
        eps = float(np.linalg.norm(r) / nu)
        history.append(eps)
        x = x - ALPHA * r
        if callback is not None:
            callback(n, eps, x)
        if eps < tol:
            break
    return x, np.asarray(history), activated_at


# ---- batched solves: several sources, one medium, reading R18 -----------------------------------
def solve_batch(o, ys, x0s=None, tol=1e-6, max_iter=1000):
    """Several right-hand sides y_b for one medium and wavelength (time- or source-dependent problems are solved
    "separately", one system per source; they share A).  Reading R18: the sources are iterated in
    lock step with Eq. (6), each exactly as `solve` would, and ONE stop test is applied to the stacked system
    diag(A, ..., A) [x_1 ... x_B] = [y_1 ... y_B], whose relative residual is
        eps_n = sqrt( sum_b ||r_b^(n)||^2 ) / sqrt( sum_b ||Gamma^-1 y_vec,b||^2 ).
    Nothing couples the sources: x_b^(n) equals the n-th iterate of `solve(y_b)`.
    Returns (list of fields, residual_history of the stacked system)."""
    ys = [np.asarray(y).astype(np.complex128) for y in ys]
    y_vecs = [-o.c * y for y in ys]
    xs = [np.zeros(o.shape, dtype=np.complex128) if x0s is None else np.asarray(x0).astype(np.complex128).copy()
          for x0 in (x0s if x0s is not None else ys)]
    nu2 = sum(np.linalg.norm(o.apply_B(o.propagate(yv))) ** 2 for yv in y_vecs)
    history = []
    for n in range(max_iter):
        total = 0.0
        for b in range(len(ys)):
            u = o.propagate(o.apply_B(xs[b]) + y_vecs[b])
            r = o.apply_B(xs[b] - u)
            total += np.linalg.norm(r) ** 2
            xs[b] = xs[b] - ALPHA * r
        eps = float(np.sqrt(total / nu2))
        history.append(eps)
        if eps < tol:
            break
    return xs, np.asarray(history)


def from_workload(w, n_map=None):
    """Oracle for a workload descriptor (any object with shape/pixel_size/... attributes)."""
    if n_map is None:
        n_map = w.make_medium()
    return MBSOracle(n_map, w.pixel_size, w.wavelength, w.boundary_width, w.n_subdomains,
                     periodic=w.periodic_flags(), n_correction=w.n_correction)
