"""Dense matrices assembled FROM THE DEFINITIONS in PAPER.md, independently of oracle/mbs_oracle.py's
matrix-free code (used only by the `-m "not gpu"` pins).  Nothing here calls the oracle's operators.

A = L + V with
  L   = c [ sum_d  I (x) blockdiag_s( F^-1 diag(-p^2) F ) (x) I  + k0^2 ]     (Eq. (5))
  V   = c diag(k^2 - k0^2) + c/h^2 * (K_t entries placed by index)            (Eq. (8))
"""
import numpy as np


def K_closed(m):
    """-2 (-1)^m / m^2, -pi^2/3 at 0 (band-limited second derivative, units 1/h^2)."""
    m = int(m)
    if m == 0:
        return -np.pi ** 2 / 3.0
    return -2.0 * (1.0 if m % 2 == 0 else -1.0) / float(m * m)


def dft_matrix(M):
    j = np.arange(M)
    return np.exp(-2j * np.pi * np.outer(j, j) / M)


def block_second_derivative(M, h):
    """F^-1 diag(-p^2) F for one subdomain of M points, p = 2 pi fftfreq(M, h)."""
    F = dft_matrix(M)
    p = 2.0 * np.pi * np.fft.fftfreq(M, h)
    return (F.conj().T / M) @ np.diag(-p ** 2) @ F


def axis_L_matrix(N, S, h):
    """block-diagonal second derivative along one axis (N = S*M points)."""
    M = N // S
    D2 = block_second_derivative(M, h)
    out = np.zeros((N, N), dtype=np.complex128)
    for s in range(S):
        out[s * M:(s + 1) * M, s * M:(s + 1) * M] = D2
    return out


def axis_correction_matrix(N, S, t, h, periodic):
    """Wrap corrections C_ss (corners -A12, -A12^T) and transfer blocks A_{s,s+-1} (+A12, +A12^T),
    truncated to t x t, in physical units (1/h^2), without the factor c."""
    M = N // S
    Cm = np.zeros((N, N), dtype=np.float64)
    for s in range(S):
        for a in range(t):
            for b in range(t):
                kab = K_closed(t + b - a) / h ** 2
                row_last = s * M + (M - t) + a      # a-th of the last t points of block s
                col_first = s * M + b               # b-th of the first t points of block s
                # C_ss bottom-left corner = -A12 ; top-right corner = -A12^T
                Cm[row_last, col_first] += -kab
                Cm[col_first, row_last] += -kab
                # transfer to / from the next block
                nxt = s + 1
                if nxt == S:
                    if not periodic:
                        continue
                    nxt = 0
                col_next_first = nxt * M + b
                Cm[row_last, col_next_first] += kab          # A_{s,s+1}
                Cm[col_next_first, row_last] += kab          # A_{s+1,s} = A_{s,s+1}^T
    return Cm


def kron_axis(mats_1d, shape, d):
    """I (x) ... (x) mat (x) ... (x) I acting on axis d of a C-ordered array."""
    out = np.array([[1.0]])
    for ax, n in enumerate(shape):
        out = np.kron(out, mats_1d if ax == d else np.eye(n))
    return out


def assemble(k2, k02, c, shape, S, t, h, a, periodic):
    """Returns dense (L, V) for the decomposed operator; A = L + V."""
    Nall = int(np.prod(shape))
    L = np.zeros((Nall, Nall), dtype=np.complex128)
    Vc = np.zeros((Nall, Nall), dtype=np.complex128)
    for d, Nd in enumerate(shape):
        L += kron_axis(axis_L_matrix(Nd, S[d], h), shape, d)
        if a[d] > 0 and t > 0:
            Vc += kron_axis(axis_correction_matrix(Nd, S[d], t, h, bool(periodic[d])), shape, d)
    L = c * (L + k02 * np.eye(Nall))
    V = c * (np.diag(k2.reshape(-1) - k02) + Vc)
    return L, V


def toeplitz_second_derivative(N, h):
    """Finite section of the linear convolution with K (P:106 situation 1)."""
    T = np.empty((N, N))
    for i in range(N):
        for j in range(N):
            T[i, j] = K_closed(i - j) / h ** 2
    return T
