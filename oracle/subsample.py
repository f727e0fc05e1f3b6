"""CPU oracle of the sub-sample (interpolated) time shifts.  TEST INFRASTRUCTURE, NOT THE PRODUCT:
only tests/ may import it; it shares no code with paper_1902_04934_b200.

PAPER.md L88: the likelihood needs Q_k(t + n.x_k) "for each detector k ... on a uniformly-sampled grid"; it says nothing about
arrival times that fall between samples.  The hot path's reading R8 takes the nearest sample.  This variant (DESIGN.md "NEXT-4",
reading R8') interpolates LINEARLY between the two neighbouring samples, per detector:

    x_k   = ((t_ref + dt_k) - t0_Q) f_s                      (the same individually rounded expression as O2)
    i0_k  = floor(x_k) - floor(N_t / 2),   phi_k = x_k - floor(x_k)  in [0, 1)
    lnL_j = a Re sum_k sum_lm conj(F_k Y_lm) [ (1 - phi_k) Q_k,lm[i0_k + j] + phi_k Q_k,lm[i0_k + j + 1] ] - quad

followed by the same time marginalisation (O6).  A window needs one sample more than the nearest-sample one: 0 <= i0_k and
i0_k + N_t + 1 <= N_Q, else -inf (R9).  Everything but the interpolation line comes from the pinned primitives of
ile_oracle.c (O1-O4, O6)."""
from __future__ import annotations

import math

import numpy as np

from . import antenna, delay, margT, quad, sYlm


def sample_series_lin(cfg, sample, point: int = 0):
    """(lnL_j [n_t], lnL_margT, i0 [K] int32, phi [K], out_of_range)."""
    K, M, n_q, n_t = int(cfg["n_det"]), int(cfg["n_modes"]), int(cfg["n_q"]), int(cfg["n_t"])
    fs, t0, gmst = float(cfg["fs_hz"]), float(cfg["t0_q_s"]), float(cfg["gmst_rad"])
    Q, U, V = cfg["Q"][point], cfg["U"][point], cfg["V"][point]
    F = np.zeros(K, dtype=np.complex128)
    i0 = np.zeros(K, dtype=np.int32)
    phi = np.zeros(K)
    bad = False
    for k in range(K):
        F[k] = antenna(cfg["arm_x"][k], cfg["arm_y"][k], gmst, sample["ra"], sample["dec"], sample["psi"])
        dtk = delay(cfg["vertex_m"][k], gmst, sample["ra"], sample["dec"])
        x = ((float(sample["t_ref"]) + dtk) - t0) * fs
        fl = math.floor(x)
        i0[k] = int(fl) - n_t // 2
        phi[k] = x - fl
        if i0[k] < 0 or int(i0[k]) + n_t + 1 > n_q:
            bad = True
    if bad:
        return np.full(n_t, -np.inf), -np.inf, i0, phi, True
    Y = np.array([sYlm(int(cfg["l"][j]), int(cfg["m"][j]), float(sample["incl"]), -float(sample["phi_ref"])) for j in range(M)])
    a = float(cfg["d_ref_mpc"]) / float(sample["dist_mpc"])
    qd = quad(F, Y, U, V, a)
    acc = np.zeros(n_t, dtype=np.complex128)
    for k in range(K):
        for m in range(M):
            w0 = Q[k, m, i0[k]:i0[k] + n_t]
            w1 = Q[k, m, i0[k] + 1:i0[k] + n_t + 1]
            acc += np.conj(F[k] * Y[m]) * ((1.0 - phi[k]) * w0 + phi[k] * w1)
    series = a * acc.real - qd
    return series, margT(series), i0, phi, False


def eval_batch_lin(cfg, samples, point: int = 0):
    """(lnL_margT [n], i0 [n][K], n_out_of_range)."""
    n = len(samples["ra"])
    out = np.zeros(n)
    idx = np.zeros((n, int(cfg["n_det"])), dtype=np.int32)
    bad = 0
    for a in range(n):
        _, out[a], idx[a], _, oob = sample_series_lin(cfg, {k: samples[k][a] for k in samples}, point)
        bad += int(oob)
    return out, idx, bad
