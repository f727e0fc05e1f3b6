"""CPU oracle of the overlap pre-computation (eq. 8a-c).
TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/ may import it; it shares no code with paper_1902_04934_b200.

Discrete setting: N samples at rate f_s, two-sided FFT grid f_n = n' f_s / N with the
signed index n' of FFT order, whitened spectra, inner product <a|b> = sum_n conj(a[n]) b[n]:

    Q_{k,lm}[i] = <h_lm(. - tau_i) | d_k> = sum_n conj(x_{k,lm}[n]) d_k[n] exp(+2 pi i f_n tau_i),   tau_i = t0_Q + i / f_s
    U_k[a][b]   = <h_a | h_b>            = sum_n conj(x_a[n]) x_b[n]
    V_k[a][b]   = <h_a^* | h_b>          = sum_n x_a[(-n) mod N] x_b[n]

`overlaps` evaluates Q with one inverse FFT per series (numpy's FFT as the library step; the phase exp(2 pi i f_n t0_Q) is
applied to the spectrum first) and U, V by the sums as written.  `overlaps_direct` is the O(N^2) definition, loop by loop,
for pinning `overlaps` on tiny inputs.
"""
from __future__ import annotations

import numpy as np


def signed_index(n_q: int):
    """n' of FFT order: 0, 1, ..., N/2 - 1, -N/2, ..., -1."""
    n = np.arange(n_q)
    return np.where(n < (n_q + 1) // 2, n, n - n_q)


def overlaps(x, d, fs_hz: float, t0_q_s: float):
    """x: complex128 [K][M][N], d: complex128 [K][N]  ->  Q [K][M][N], U [K][M][M], V [K][M][M]."""
    x = np.asarray(x, dtype=np.complex128)
    d = np.asarray(d, dtype=np.complex128)
    K, M, N = x.shape
    f = signed_index(N) * (fs_hz / N)
    neg = (-np.arange(N)) % N
    Q = np.empty((K, M, N), dtype=np.complex128)
    U = np.empty((K, M, M), dtype=np.complex128)
    V = np.empty((K, M, M), dtype=np.complex128)
    for k in range(K):
        shifted = d[k] * np.exp(2j * np.pi * f * t0_q_s)
        for a in range(M):
            # sum_n c[n] exp(+2 pi i n i / N) = N * ifft(c)[i]
            Q[k, a] = np.fft.ifft(np.conj(x[k, a]) * shifted) * N
            for b in range(M):
                U[k, a, b] = np.sum(np.conj(x[k, a]) * x[k, b])
                V[k, a, b] = np.sum(x[k, a][neg] * x[k, b])
    return Q, U, V


def overlaps_direct(x, d, fs_hz: float, t0_q_s: float):
    """The definition, term by term (pure Python loops: tiny inputs only)."""
    x = np.asarray(x, dtype=np.complex128)
    d = np.asarray(d, dtype=np.complex128)
    K, M, N = x.shape
    npr = signed_index(N)
    Q = np.zeros((K, M, N), dtype=np.complex128)
    U = np.zeros((K, M, M), dtype=np.complex128)
    V = np.zeros((K, M, M), dtype=np.complex128)
    for k in range(K):
        for a in range(M):
            for i in range(N):
                tau = t0_q_s + i / fs_hz
                acc = 0j
                for n in range(N):
                    fn = npr[n] * fs_hz / N
                    acc += np.conj(x[k, a, n]) * d[k, n] * np.exp(2j * np.pi * fn * tau)
                Q[k, a, i] = acc
            for b in range(M):
                u = 0j
                v = 0j
                for n in range(N):
                    u += np.conj(x[k, a, n]) * x[k, b, n]
                    v += x[k, a, (-n) % N] * x[k, b, n]
                U[k, a, b] = u
                V[k, a, b] = v
    return Q, U, V
