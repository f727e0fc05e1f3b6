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


def psd_weights(n_q: int, S_k, fs_hz: float, f_min_hz: float, f_max_hz: float, scale: float):
    """Weight of frequency n in eq. 2 (<a|b>_k = 2 int_{f_min < |f| < f_max} a~*(f) b~(f) / S_k(|f|) df,
    two-sided): scale / S_k(|f_n|) inside the band f_min < |f_n| < f_max, 0 outside.  S_k is the one-sided PSD sampled at
    |f_n| on the FFT grid (FFT order); `scale` carries the measure (2 df for the integral as printed, times whatever the
    caller's Fourier convention asks for)."""
    af = np.abs(signed_index(n_q) * (fs_hz / n_q))
    return np.where((af > f_min_hz) & (af < f_max_hz), scale / np.asarray(S_k, dtype=np.float64), 0.0)


def overlaps_psd(h, d, S, fs_hz: float, t0_q_s: float, f_min_hz: float, f_max_hz: float, scale: float):
    """eq. 8a-c with eq. 2's weighting on UN-whitened spectra: h [K][M][N], d [K][N], S [K][N] (real, > 0 in the band).
        Q[k][a][i] = sum_n g_k[n] conj(h[k][a][n]) d[k][n] exp(+2 pi i f_n (t0_Q + i / f_s))
        U[k][a][b] = sum_n g_k[n] conj(h[k][a][n]) h[k][b][n],   V[k][a][b] = sum_n g_k[n] h[k][a][(-n) mod N] h[k][b][n]
    Q by one inverse FFT per series, U and V by the sums as written."""
    h = np.asarray(h, dtype=np.complex128)
    d = np.asarray(d, dtype=np.complex128)
    K, M, N = h.shape
    f = signed_index(N) * (fs_hz / N)
    neg = (-np.arange(N)) % N
    Q = np.empty((K, M, N), dtype=np.complex128)
    U = np.empty((K, M, M), dtype=np.complex128)
    V = np.empty((K, M, M), dtype=np.complex128)
    for k in range(K):
        g = psd_weights(N, S[k], fs_hz, f_min_hz, f_max_hz, scale)
        shifted = d[k] * np.exp(2j * np.pi * f * t0_q_s) * g
        for a in range(M):
            Q[k, a] = np.fft.ifft(np.conj(h[k, a]) * shifted) * N
            for b in range(M):
                U[k, a, b] = np.sum(g * np.conj(h[k, a]) * h[k, b])
                V[k, a, b] = np.sum(g * h[k, a][neg] * h[k, b])
    return Q, U, V


def overlaps_direct_psd(h, d, S, fs_hz: float, t0_q_s: float, f_min_hz: float, f_max_hz: float, scale: float):
    """overlaps_psd term by term (pure Python loops: tiny inputs only)."""
    h = np.asarray(h, dtype=np.complex128)
    d = np.asarray(d, dtype=np.complex128)
    K, M, N = h.shape
    npr = signed_index(N)
    Q = np.zeros((K, M, N), dtype=np.complex128)
    U = np.zeros((K, M, M), dtype=np.complex128)
    V = np.zeros((K, M, M), dtype=np.complex128)
    for k in range(K):
        for n in range(N):
            fn = npr[n] * fs_hz / N
            if not (f_min_hz < abs(fn) < f_max_hz):
                continue
            g = scale / S[k][n]
            for a in range(M):
                for i in range(N):
                    Q[k, a, i] += g * np.conj(h[k, a, n]) * d[k, n] * np.exp(2j * np.pi * fn * (t0_q_s + i / fs_hz))
                for b in range(M):
                    U[k, a, b] += g * np.conj(h[k, a, n]) * h[k, b, n]
                    V[k, a, b] += g * h[k, a, (-n) % N] * h[k, b, n]
    return Q, U, V
