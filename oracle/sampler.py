"""CPU oracle of the on-device Monte Carlo sampler.  TEST INFRASTRUCTURE, NOT THE PRODUCT:
only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import it; it shares no code with
paper_1902_04934_b200 and imports nothing from it.

What the paper fixes (line numbers are /root/reference/PAPER.md):
  * eq. 4: L_marg = int L p(theta) dtheta "via direct Monte Carlo integration over almost all parameters theta,
    where p(theta) is uniform in 4-volume and source orientation ... to evaluate the likelihood in regions of high
    importance, we use an adaptive Monte Carlo as described in [9]";
  * L97: blocks of 1e4 random extrinsic parameters per likelihood call;
  * L119: "the sampling prior used in adaptive Monte Carlo is regenerated from the most recent n_chunk data points ...
    every n_chunk iterations ..., regenerating a sampling prior in two sky location parameters and distance";
  * L125: "we only adapt in two parameters, corresponding to sky location; and only adapt until a marginalized likelihood
    evaluation returns significant ln L_marg";
  * L101: "relative uncertainty of order 1/sqrt(n_eff) ... We adopt a fixed threshold on n_eff";
  * L251: "converting the Monte Carlo random number generation ... to GPU-based operations".
The sampler itself lives in ref. [9], which is not in /root/reference: the algorithm below is this build's reading
(readings S1-S9), followed here step by step in plain numpy.

S1  Random numbers: Philox4x32-10 (Salmon et al. 2011), counter-based.  Sample alpha (a 64-bit index counted from the
    start of the run) uses the four counters (alpha_lo, alpha_hi, j, 0), j = 0..3, under the key (seed_lo, seed_hi): 16
    words w[0..15].  Uniform i (i = 0..6) = ((w[2i] >> 5) * 2^26 + (w[2i+1] >> 6) + 0.5) * 2^-53, in (0, 1).
S2  Coordinates in which the prior is uniform on the unit cube (L47: uniform in volume and orientation):
    u0 = RA / 2pi, u1 = (sin dec + 1)/2, u2 = (t_ref - t_lo)/(t_hi - t_lo), u3 = phi_ref / 2pi, u4 = psi / pi,
    u5 = (cos iota + 1)/2, u6 = (D^3 - Dmin^3)/(Dmax^3 - Dmin^3).
S3  Sampling prior: product over the adaptive dimensions d in {0: RA, 1: dec, 6: distance} (those enabled) of piecewise-
    constant densities h_d on n_bins equal bins of u_d (sum_b h_d[b] / n_bins = 1); every other dimension is drawn from
    the prior.  So ln w = ln p - ln p_s = - sum_d ln h_d[bin_d].
S4  Draw: for an adaptive dimension, v = uniform i; cumulative C_d[0] = 0, C_d[b+1] = C_d[b] + h_d[b] / n_bins (one
    division and one addition per bin, in this order); b = the largest bin with C_d[b] <= v (clamped to n_bins - 1);
    u_d = (b + (v - C_d[b]) / (h_d[b] / n_bins)) / n_bins, clamped below 1.
S5  Physical parameters: RA = 2 pi u0, dec = asin(2 u1 - 1), t_ref = t_lo + (t_hi - t_lo) u2, phi_ref = 2 pi u3,
    psi = pi u4, iota = acos(2 u5 - 1), D = cbrt(Dmin^3 + u6 (Dmax^3 - Dmin^3)) with X^3 = (X X) X.
S6  Refit from the most recent chunk (L119): e_a = lnL_margT,a + ln w_a, M = max_a e_a, W_a = exp(temper * (e_a - M));
    per adaptive dimension the integer histogram H_d[b] = sum over the chunk's samples in bin b of rint(W_a * 2^40)
    (integers: the sum does not depend on the order); if sum_b H_d[b] = 0 (no finite sample) the density is kept;
    otherwise h_d[b] = (1 - floor) * n_bins * H_d[b] / sum_b H_d[b] + floor.
S7  Loop (L97, L119): chunk c draws samples c*n_chunk .. (c+1)*n_chunk - 1 from the current densities, evaluates
    lnL_margT, accumulates the evidence (eq. 4: lnZ = ln((1/N) sum w L), n_eff = sum wL / max wL over ALL samples so
    far), then refits while c < n_adapt_chunks (L125: adapt only early on).
S8  Stop (L101): after the first chunk at which n_eff >= n_eff_min, or after max_chunks.
S9  The densities start uniform (h = 1: the first chunk is drawn from the prior).
"""
from __future__ import annotations

import math

import numpy as np

M32 = np.uint64(0xFFFFFFFF)
PHILOX_M0, PHILOX_M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
PHILOX_W0, PHILOX_W1 = np.uint64(0x9E3779B9), np.uint64(0xBB67AE85)
ADAPTIVE_DIMS = (0, 1, 6)          # RA, dec, distance (L119)
FIXED_POINT = float(2 ** 40)       # S6


def philox4x32_10(counter, key):
    """Philox4x32 with 10 rounds.  counter: uint32 [..., 4], key: uint32 [..., 2] -> uint32 [..., 4].
    One round: (c0, c1, c2, c3) <- (hi(M1*c2) ^ c1 ^ k0, lo(M1*c2), hi(M0*c0) ^ c3 ^ k1, lo(M0*c0)); the key is bumped
    by (W0, W1) between rounds."""
    c = [np.asarray(counter[..., i], dtype=np.uint64) for i in range(4)]
    k0 = np.asarray(key[..., 0], dtype=np.uint64)
    k1 = np.asarray(key[..., 1], dtype=np.uint64)
    for r in range(10):
        p0 = PHILOX_M0 * c[0]
        p1 = PHILOX_M1 * c[2]
        hi0, lo0 = p0 >> np.uint64(32), p0 & M32
        hi1, lo1 = p1 >> np.uint64(32), p1 & M32
        c = [(hi1 ^ c[1] ^ k0) & M32, lo1, (hi0 ^ c[3] ^ k1) & M32, lo0]
        k0 = (k0 + PHILOX_W0) & M32
        k1 = (k1 + PHILOX_W1) & M32
    return np.stack(c, axis=-1).astype(np.uint32)


def uniforms(seed: int, first_index: int, n: int):
    """S1: float64 [n][7], the seven uniforms of samples first_index .. first_index + n - 1."""
    idx = np.arange(first_index, first_index + n, dtype=np.uint64)
    ctr = np.zeros((n, 4, 4), dtype=np.uint32)
    ctr[:, :, 0] = (idx & M32).astype(np.uint32)[:, None]
    ctr[:, :, 1] = (idx >> np.uint64(32)).astype(np.uint32)[:, None]
    ctr[:, :, 2] = np.arange(4, dtype=np.uint32)[None, :]
    key = np.zeros((n, 4, 2), dtype=np.uint32)
    key[..., 0] = np.uint32(seed & 0xFFFFFFFF)
    key[..., 1] = np.uint32((seed >> 32) & 0xFFFFFFFF)
    w = philox4x32_10(ctr, key).reshape(n, 16).astype(np.uint64)
    out = np.empty((n, 7))
    for i in range(7):
        hi, lo = w[:, 2 * i] >> np.uint64(5), w[:, 2 * i + 1] >> np.uint64(6)
        out[:, i] = (hi.astype(np.float64) * 67108864.0 + lo.astype(np.float64) + 0.5) * (2.0 ** -53)
    return out


def uniform_tables(n_bins: int):
    """S9: h [3][n_bins] = 1."""
    return np.ones((3, n_bins))


def cumulative(h_d):
    """S4: C[0] = 0, C[b+1] = C[b] + h[b]/n_bins, sequentially."""
    nb = len(h_d)
    C = np.zeros(nb + 1)
    for b in range(nb):
        C[b + 1] = C[b] + h_d[b] / nb
    return C


def draw(cfg, h, first_index: int, n: int):
    """S1-S5.  cfg: dict(seed, n_bins, adapt (3 bools for RA, dec, distance), dist_min_mpc, dist_max_mpc, t_ref_lo_s,
    t_ref_hi_s); h: densities [3][n_bins].  Returns (samples dict of float64 [n], log_w [n], bins int32 [n][3] (-1 for a
    dimension that is not adaptive), u [n][7])."""
    nb = int(cfg["n_bins"])
    v = uniforms(int(cfg["seed"]), first_index, n)
    u = v.copy()
    bins = np.full((n, 3), -1, dtype=np.int32)
    log_w = np.zeros(n)
    for j, d in enumerate(ADAPTIVE_DIMS):
        if not cfg["adapt"][j]:
            continue
        C = cumulative(h[j])
        b = np.searchsorted(C, v[:, d], side="right") - 1            # largest b with C[b] <= v
        b = np.clip(b, 0, nb - 1)
        width = h[j][b] / nb
        ud = (b + (v[:, d] - C[b]) / width) / nb
        u[:, d] = np.minimum(ud, 1.0 - 2.0 ** -53)
        bins[:, j] = b
        log_w -= np.log(h[j][b])
    two_pi = 2.0 * math.pi
    dmin, dmax = float(cfg["dist_min_mpc"]), float(cfg["dist_max_mpc"])
    dmin3, dmax3 = dmin * dmin * dmin, dmax * dmax * dmax           # two multiplications each (S5)
    s = {
        "ra": two_pi * u[:, 0],
        "dec": np.arcsin(2.0 * u[:, 1] - 1.0),
        "t_ref": cfg["t_ref_lo_s"] + (cfg["t_ref_hi_s"] - cfg["t_ref_lo_s"]) * u[:, 2],
        "phi_ref": two_pi * u[:, 3],
        "psi": math.pi * u[:, 4],
        "incl": np.arccos(2.0 * u[:, 5] - 1.0),
        "dist_mpc": np.cbrt(dmin3 + u[:, 6] * (dmax3 - dmin3)),
    }
    return {k: np.ascontiguousarray(x) for k, x in s.items()}, log_w, bins, u


def refit(cfg, h, bins, lnL, log_w):
    """S6: new densities [3][n_bins] from one chunk (bins [n][3], lnL [n], log_w [n])."""
    nb = int(cfg["n_bins"])
    e = np.asarray(lnL) + np.asarray(log_w)
    M = np.max(e) if len(e) else -np.inf
    out = np.array(h, dtype=np.float64, copy=True)
    if not np.isfinite(M):
        return out
    W = np.exp(float(cfg["temper"]) * (e - M))                       # exp(-inf) = 0 for out-of-range samples
    q = np.rint(W * FIXED_POINT).astype(np.int64)
    f = float(cfg["floor_frac"])
    for j in range(3):
        if not cfg["adapt"][j]:
            continue
        H = np.zeros(nb, dtype=np.int64)
        np.add.at(H, bins[:, j], q)
        tot = int(H.sum())
        if tot == 0:
            continue
        out[j] = (1.0 - f) * nb * (H.astype(np.float64) / float(tot)) + f
    return out


def integrate(cfg, eval_lnL, n_chunk: int, max_chunks: int, n_adapt_chunks: int, n_eff_min: float):
    """S7-S8.  eval_lnL(samples dict) -> lnL_margT [n] (the hot-path oracle).  Returns dict(lnZ, n_eff, n_samples,
    n_chunks, h (final densities), history [(lnZ, n_eff)] per chunk)."""
    h = uniform_tables(int(cfg["n_bins"]))
    m, ssum, count = -np.inf, 0.0, 0
    hist = []
    for c in range(max_chunks):
        s, log_w, bins, _ = draw(cfg, h, c * n_chunk, n_chunk)
        lnL = eval_lnL(s)
        e = lnL + log_w
        mc = float(np.max(e))
        if np.isfinite(mc):
            mx = max(m, mc)
            ssum = (ssum * math.exp(m - mx) if np.isfinite(m) else 0.0) + float(np.sum(np.exp(e - mx)))
            m = mx
        count += n_chunk
        lnZ = m + math.log(ssum) - math.log(count) if np.isfinite(m) else -np.inf
        n_eff = ssum if np.isfinite(m) else 0.0
        hist.append((lnZ, n_eff))
        if c < n_adapt_chunks:
            h = refit(cfg, h, bins, lnL, log_w)
        if n_eff >= n_eff_min:
            break
    return dict(lnZ=hist[-1][0], n_eff=hist[-1][1], n_samples=count, n_chunks=len(hist), h=h, history=hist)
