"""Pins for the harvesting oracle (oracle/harvest.py): hand-worked cases, brute-force loops, exact
expected counts, frequency tests and the noise-free injection whose true time bin is known.  All CPU, -m "not gpu"."""
import math

import numpy as np
from scipy import stats

import ile_inputs as gi
import oracle
from oracle import harvest as oh
from test_oracle_pins import C_SI, Y2m_closed, antenna_vec, source_dir


def test_argmax_by_brute_scan_first_of_ties_and_known_truth():
    rng = np.random.default_rng(0)
    for _ in range(200):
        x = rng.normal(0, 3, rng.integers(1, 60))
        best, jb = -math.inf, -1
        for j, v in enumerate(x):            # brute scan, strict > keeps the first of equal maxima
            if v > best:
                best, jb = v, j
        assert oh.argmax_bin(x) == (jb, best)
    assert oh.argmax_bin([1.0, 5.0, 5.0, 2.0]) == (1, 5.0)
    # the true arrival time of a noise-free injection: the harvested bin is the one the signal was put in (bin n_t // 2 when
    # t_ref = t_true), and lnL there is rho^2 / 2
    base = gi.make_config(1, n=1)
    th = dict(ra=1.3, dec=-0.4, psi=0.7, phi_ref=2.1, incl=0.9, dist_mpc=gi.D_TRUE_MPC, t_ref=0.0)
    resp, tau = [], []
    for k in range(base["n_det"]):
        fp, fc = antenna_vec(base["arm_x"][k], base["arm_y"][k], th["ra"], th["dec"], th["psi"], base["gmst_rad"])
        resp.append(complex(fp, fc))
        tau.append(int(np.rint(-float(np.dot(base["vertex_m"][k], source_dir(th["ra"], th["dec"], base["gmst_rad"]))) / C_SI * base["fs_hz"])))
    y = np.array([Y2m_closed(m, th["incl"], -th["phi_ref"]) for (_, m) in base["modes"]])
    Q, U, V, _ = gi.make_point(5, base["dets"], base["modes"], base["n_q"], 12.0, noise=False,
                               truth_response=dict(y=y, resp=np.array(resp), tau_samples=np.array(tau)))
    cfg = dict(base)
    cfg.update(Q=Q[None], U=U[None], V=V[None])
    for shift in (0, 7, -30):                # sample whose t_ref is `shift` bins early: the peak moves to n_t // 2 + shift
        s = dict(th, t_ref=-shift / base["fs_hz"])
        series = oracle.sample_series(cfg, s)[0]
        j, v = oh.argmax_bin(series)
        assert j == cfg["n_t"] // 2 + shift and abs(v - 72.0) < 1e-7


def test_time_draw_by_hand_and_frequencies():
    series = np.log(np.array([0.1, 0.2, 0.3, 0.4]))          # CDF 0.1, 0.3, 0.6, 1.0
    for v, want in ((0.05, 0), (0.0999, 0), (0.1001, 1), (0.25, 1), (0.3001, 2), (0.59, 2), (0.61, 3), (0.999, 3)):
        assert oh.draw_time_bin(series, v) == want
    assert oh.draw_time_bin(series + 700.0, 0.25) == 1 and oh.draw_time_bin(series - 700.0, 0.61) == 3   # max-subtracted
    assert oh.draw_time_bin([3.0], 0.7) == 0
    assert oh.draw_time_bin([-np.inf, 0.0, -np.inf], 0.5) == 1
    # brute force with exact rational arithmetic on dyadic probabilities
    rng = np.random.default_rng(1)
    p = rng.integers(1, 64, 40).astype(float)
    p /= 2.0 ** 12
    cdf = np.cumsum(p) / p.sum()
    for v in rng.random(500):
        want = next(j for j in range(40) if cdf[j] >= v)
        assert oh.draw_time_bin(np.log(p), v) == want
    # frequencies follow exp(lnL)
    n = 200_000
    x = rng.normal(0, 1.5, 30)
    cnt = np.bincount([oh.draw_time_bin(x, v) for v in rng.random(n)], minlength=30)
    pr = np.exp(x - x.max())
    pr /= pr.sum()
    assert stats.chi2.sf(np.sum((cnt - n * pr) ** 2 / (n * pr)), 29) > 1e-4
    assert np.allclose(oh.time_cdf(x), np.cumsum(pr), atol=1e-15)


def test_systematic_resampling_exact_counts_and_properties():
    # weights 1 : 2 : 3 : 4 and ten outputs: counts 1, 2, 3, 4 for EVERY offset v0
    e = np.log(np.array([1.0, 2.0, 3.0, 4.0]))
    for v0 in (0.0, 0.3, 0.77, 0.999):
        ids = oh.systematic_resample(e, None, 10, v0)
        assert np.array_equal(np.bincount(ids, minlength=4), [1, 2, 3, 4]) and np.all(np.diff(ids) >= 0)
    # ln w enters additively: the same weights split between lnL and ln w
    assert np.array_equal(oh.systematic_resample(np.zeros(4), e, 10, 0.3), oh.systematic_resample(e, None, 10, 0.3))
    # general weights: every count is floor or ceil of its expectation, -inf samples are never chosen, brute force agrees
    rng = np.random.default_rng(2)
    n, n_out = 5_000, 1_777
    lnL = rng.normal(0, 4, n)
    lw = rng.normal(0, 1, n)
    lnL[::41] = -np.inf
    for v0 in (0.0, 0.5, 0.123456):
        ids = oh.systematic_resample(lnL, lw, n_out, v0)
        assert len(ids) == n_out and np.all(np.diff(ids) >= 0)
        W = np.exp(lnL + lw - np.max(lnL + lw))
        expect = n_out * W / W.sum()
        cnt = np.bincount(ids, minlength=n)
        assert np.all(cnt >= np.floor(expect - 1e-9)) and np.all(cnt <= np.ceil(expect + 1e-9))
        assert np.all(cnt[::41] == 0)
        cdf, brute, a = np.cumsum(W) / W.sum(), [], 0
        for i in range(n_out):
            p = (i + v0) / n_out
            while cdf[a] <= p and a < n - 1:
                a += 1
            brute.append(a)
        assert np.array_equal(ids, brute)
    # unbiased over the offset: mean count = expectation
    tot = np.zeros(n)
    offs = (np.arange(400) + 0.5) / 400
    for v0 in offs:
        tot += np.bincount(oh.systematic_resample(lnL, lw, 50, v0), minlength=n)
    W = np.exp(lnL + lw - np.max(lnL + lw))
    assert np.max(np.abs(tot / len(offs) - 50 * W / W.sum())) < 0.01
    assert len(oh.systematic_resample(np.full(5, -np.inf), None, 10, 0.5)) == 0
