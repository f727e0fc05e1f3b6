"""CPU oracle of the extrinsic posterior harvesting.  TEST INFRASTRUCTURE, NOT THE PRODUCT: only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import it; it shares no code with
paper_1902_04934_b200.

PAPER.md L265: "The code also produces reliable extrinsic parameter distributions [9] ... we harvest joint intrinsic and
extrinsic information with a single final iteration."  The paper says no more; what a posterior over ALL extrinsic parameters
needs from this path follows from its own structure -- eq. 4 (L42-L47) integrates the other extrinsic parameters by Monte
Carlo with weights w = p/p_s and eq. 9 (L81-L86) integrates time by quadrature -- and is this build's reading (DESIGN.md
"NEXT-3", H1-H3):

H1  Posterior samples of the Monte Carlo parameters: the draws theta_a carry posterior weight W_a = w_a L_margT,a (eq. 4's
    integrand).  Equal-weight samples by SYSTEMATIC resampling: with one uniform v0 in [0, 1) and n_out points
    p_i = (i + v0) / n_out, output i is the smallest a whose inclusive cumulative weight c_a = sum_{b <= a} W_b / sum_b W_b
    exceeds p_i.  W_a = exp(e_a - max e), e_a = lnL_margT,a + ln w_a; c_a accumulated in sample order.
H2  The time of a harvested sample: eq. 9 marginalised it over the window, so its posterior given theta_a is the normalised
    integrand exp(lnL_j) over the N_t bins.  Draw with one uniform v in (0, 1): the smallest bin j whose inclusive
    cumulative sum_{i <= j} exp(lnL_i - max) reaches v * sum_i exp(lnL_i - max).
H3  The best-fit time: the first bin j* at which lnL_j is largest, and lnL_{j*} itself (the maximised-over-time lnL that
    eq. 9 replaces by an average).
A bin j of sample a means the geocentric time t_ref,a + (j - floor(N_t/2)) / f_s (reading R10: the window is centred on t_ref).

The series lnL_j itself is the hot-path oracle's (oracle.sample_series: O1-O5 of ile_oracle.c); this module adds the three
steps above in plain numpy, in the order written.
"""
from __future__ import annotations

import numpy as np


def argmax_bin(series):
    """H3: (first bin of the maximum, the maximum)."""
    series = np.asarray(series, dtype=np.float64)
    j = int(np.argmax(series))       # numpy returns the first occurrence
    return j, float(series[j])


def draw_time_bin(series, v: float):
    """H2: smallest j with cumsum_j(exp(lnL - max)) >= v * total; sequential accumulation."""
    series = np.asarray(series, dtype=np.float64)
    m = np.max(series)
    p = np.exp(series - m)
    c = np.cumsum(p)                 # sequential, in bin order
    target = v * c[-1]
    j = int(np.searchsorted(c, target, side="left"))
    return min(j, len(series) - 1)


def time_cdf(series):
    """Normalised inclusive cumulative of H2 (for tests that need the margin of a draw)."""
    series = np.asarray(series, dtype=np.float64)
    c = np.cumsum(np.exp(series - np.max(series)))
    return c / c[-1]


def systematic_resample(lnL_margT, log_w, n_out: int, v0: float):
    """H1: int64 [n_out] sample indices (non-decreasing).  A set without a finite weight returns an empty array."""
    e = np.asarray(lnL_margT, dtype=np.float64) + (0.0 if log_w is None else np.asarray(log_w, dtype=np.float64))
    m = np.max(e) if len(e) else -np.inf
    if not np.isfinite(m):
        return np.zeros(0, dtype=np.int64)
    W = np.exp(e - m)
    c = np.cumsum(W)                 # sequential, in sample order
    p = (np.arange(n_out) + v0) / n_out * c[-1]
    ids = np.searchsorted(c, p, side="right")      # smallest a with c_a > p_i
    return np.minimum(ids, len(e) - 1).astype(np.int64)


def resample_cdf(lnL_margT, log_w):
    e = np.asarray(lnL_margT, dtype=np.float64) + (0.0 if log_w is None else np.asarray(log_w, dtype=np.float64))
    c = np.cumsum(np.exp(e - np.max(e)))
    return c / c[-1]
