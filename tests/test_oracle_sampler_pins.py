"""Pins for the sampler oracle (oracle/sampler.py): every function is checked against something
other than itself -- the published Philox known-answer vectors, brute-force loops, exact expected values, distribution
tests against the seeded prior generator, unbiasedness of the importance weights (E[w] = 1) and agreement of the
evidence with the plain prior-sampled estimate of the existing path within Monte Carlo error.  All CPU, -m "not gpu"."""
import math

import numpy as np
import pytest
from scipy import stats

import ile_inputs as gi
import oracle
from oracle import sampler as osm

CFG = dict(seed=0x1234ABCD5678EF01, n_bins=64, adapt=(True, True, True), dist_min_mpc=1.0, dist_max_mpc=1000.0,
           t_ref_lo_s=-0.05, t_ref_hi_s=0.05, floor_frac=0.1, temper=1.0)


# ----------------------------------------------------------------------------------------------------------
# S1: Philox4x32-10
# ----------------------------------------------------------------------------------------------------------
def test_philox_known_answer_vectors():
    """Known-answer tests of Philox4x32-10 as published with the generator (Salmon, Moraes, Dror, Shaw, SC'11; the
    Random123 distribution's kat_vectors): counter / key -> output."""
    kat = [
        ((0x00000000, 0x00000000, 0x00000000, 0x00000000), (0x00000000, 0x00000000), (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
        ((0xffffffff, 0xffffffff, 0xffffffff, 0xffffffff), (0xffffffff, 0xffffffff), (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
        ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0), (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1)),
    ]
    for ctr, key, want in kat:
        got = osm.philox4x32_10(np.array(ctr, dtype=np.uint32), np.array(key, dtype=np.uint32))
        assert tuple(int(x) for x in got) == want


def test_philox_round_function_by_hand():
    """One application with python integers (arbitrary precision: no overflow subtleties) against the vectorised code."""
    def ref(ctr, key):
        c = list(ctr)
        k = list(key)
        for _ in range(10):
            p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
            c = [((p1 >> 32) ^ c[1] ^ k[0]) & 0xFFFFFFFF, p1 & 0xFFFFFFFF, ((p0 >> 32) ^ c[3] ^ k[1]) & 0xFFFFFFFF, p0 & 0xFFFFFFFF]
            k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
        return c
    rng = np.random.default_rng(1)
    for _ in range(50):
        ctr = [int(x) for x in rng.integers(0, 2 ** 32, 4)]
        key = [int(x) for x in rng.integers(0, 2 ** 32, 2)]
        got = osm.philox4x32_10(np.array(ctr, dtype=np.uint32), np.array(key, dtype=np.uint32))
        assert [int(x) for x in got] == ref(ctr, key)


def test_uniforms_layout_range_and_statistics():
    n = 200_000
    u = osm.uniforms(CFG["seed"], 0, n)
    assert u.shape == (n, 7) and u.min() > 0.0 and u.max() < 1.0
    # counter layout (S1): sample alpha, word pair (2i, 2i+1) of the 16 words of counters (alpha_lo, alpha_hi, j, 0)
    a = 123_456
    words = []
    for j in range(4):
        words += [int(x) for x in osm.philox4x32_10(np.array([a, 0, j, 0], dtype=np.uint32),
                                                     np.array([CFG["seed"] & 0xFFFFFFFF, CFG["seed"] >> 32], dtype=np.uint32))]
    for i in range(7):
        want = ((words[2 * i] >> 5) * 2 ** 26 + (words[2 * i + 1] >> 6) + 0.5) * 2.0 ** -53
        assert u[a, i] == want
    # a window of the same stream is the same numbers; indices beyond 2^32 use the high counter word
    assert np.array_equal(osm.uniforms(CFG["seed"], 1000, 50), u[1000:1050])
    hi = osm.uniforms(CFG["seed"], 2 ** 32 + 5, 3)
    assert not np.array_equal(hi, u[5:8])
    # statistics: every column uniform (KS), columns and neighbouring samples uncorrelated
    for i in range(7):
        assert stats.kstest(u[:, i], "uniform").pvalue > 1e-4
    cc = np.corrcoef(u.T)
    assert np.max(np.abs(cc - np.eye(7))) < 5.0 / math.sqrt(n)
    assert abs(np.corrcoef(u[:-1, 0], u[1:, 0])[0, 1]) < 5.0 / math.sqrt(n)
    assert len(np.unique(u[:, 0])) == n


# ----------------------------------------------------------------------------------------------------------
# S2-S5: draw
# ----------------------------------------------------------------------------------------------------------
def test_draw_from_uniform_tables_is_the_prior():
    """S9 + S5: with h = 1 the samples follow the prior of SURVEY.md §8(d) item 7 (the seeded generator's), ln w = 0."""
    n = 100_000
    s, lw, bins, u = osm.draw(CFG, osm.uniform_tables(CFG["n_bins"]), 0, n)
    assert np.all(lw == 0.0)
    ref = gi.make_samples(42, n)
    for k in gi.SAMPLE_FIELDS:
        assert stats.ks_2samp(s[k], ref[k]).pvalue > 1e-4, k
    # closed forms of the prior: sin dec and cos iota uniform on [-1, 1], D^3 uniform (uniform in volume, L47)
    assert stats.kstest((np.sin(s["dec"]) + 1) / 2, "uniform").pvalue > 1e-4
    assert stats.kstest((np.cos(s["incl"]) + 1) / 2, "uniform").pvalue > 1e-4
    assert stats.kstest((s["dist_mpc"] ** 3 - 1.0) / (1000.0 ** 3 - 1.0), "uniform").pvalue > 1e-4
    assert s["ra"].min() >= 0 and s["ra"].max() < 2 * np.pi and s["psi"].max() < np.pi
    assert abs(s["t_ref"]).max() <= 0.05
    # the uniform-table draw leaves the Philox uniforms untouched (up to the inverse-CDF arithmetic) and bins = floor(u nb)
    v = osm.uniforms(CFG["seed"], 0, n)
    assert np.max(np.abs(u - v)) < 1e-15
    for j, d in enumerate(osm.ADAPTIVE_DIMS):
        assert np.array_equal(bins[:, j], np.floor(v[:, d] * CFG["n_bins"]).astype(np.int32))


def test_inverse_cdf_by_hand():
    """S4 on a 4-bin density worked out by hand: h = (0.4, 2.0, 1.2, 0.4), C = (0, 0.1, 0.6, 0.9, 1)."""
    cfg = dict(CFG, n_bins=4, adapt=(True, False, False))
    h = np.array([[0.4, 2.0, 1.2, 0.4], [1, 1, 1, 1], [1, 1, 1, 1]], dtype=float)
    assert np.allclose(osm.cumulative(h[0]), [0, 0.1, 0.6, 0.9, 1.0], atol=1e-16)
    s, lw, bins, u = osm.draw(cfg, h, 0, 2000)
    v = osm.uniforms(cfg["seed"], 0, 2000)[:, 0]
    for vi, ui, bi, li in zip(v, u[:, 0], bins[:, 0], lw):
        if vi < 0.1:
            b, want = 0, (vi / 0.1) / 4
        elif vi < 0.6:
            b, want = 1, (1 + (vi - 0.1) / 0.5) / 4
        elif vi < 0.9:
            b, want = 2, (2 + (vi - 0.6) / 0.3) / 4
        else:
            b, want = 3, (3 + (vi - 0.9) / 0.1) / 4
        assert bi == b and abs(ui - want) < 1e-14 and abs(li + math.log(h[0][b])) < 1e-15
    assert np.all(bins[:, 1:] == -1)


def test_draw_follows_the_tables_and_weights_are_unbiased():
    """Empirical bin frequencies match h_d / n_bins (chi-square), E[w] = 1, and E[w g(theta)] = E_prior[g] (importance
    sampling identity) for a test function g."""
    rng = np.random.default_rng(5)
    nb = CFG["n_bins"]
    h = rng.uniform(0.2, 3.0, size=(3, nb))
    h /= h.mean(axis=1, keepdims=True)                        # sum h / nb = 1
    n = 400_000
    s, lw, bins, u = osm.draw(CFG, h, 0, n)
    for j in range(3):
        obs = np.bincount(bins[:, j], minlength=nb)
        chi2 = np.sum((obs - n * h[j] / nb) ** 2 / (n * h[j] / nb))
        assert stats.chi2.sf(chi2, nb - 1) > 1e-4
        # inside a bin the draw is uniform: fractional position
        frac = u[:, osm.ADAPTIVE_DIMS[j]] * nb - bins[:, j]
        assert frac.min() >= 0 and frac.max() <= 1 and stats.kstest(frac, "uniform").pvalue > 1e-4
    w = np.exp(lw)
    assert abs(w.mean() - 1.0) < 5 * w.std() / math.sqrt(n)
    g = np.sin(s["dec"]) ** 2 + np.cos(s["ra"]) + (s["dist_mpc"] / 1000.0) ** 3
    exact = 1.0 / 3.0 + 0.0 + (1000.0 ** 6 - 1.0) / (2.0 * (1000.0 ** 3 - 1.0)) / 1000.0 ** 3   # E[sin^2 dec], E[cos ra], E[D^3]/1e9
    assert abs((w * g).mean() - exact) < 5 * (w * g).std() / math.sqrt(n)


# ----------------------------------------------------------------------------------------------------------
# S6: refit
# ----------------------------------------------------------------------------------------------------------
def test_refit_against_a_plain_loop_and_exact_cases():
    rng = np.random.default_rng(9)
    nb, n = CFG["n_bins"], 5000
    bins = rng.integers(0, nb, size=(n, 3)).astype(np.int32)
    lnL = rng.normal(0, 3, n)
    lw = rng.normal(0, 0.5, n)
    lnL[::97] = -np.inf                                          # out-of-range samples carry no weight
    for temper in (1.0, 0.5):
        cfg = dict(CFG, temper=temper)
        h = osm.refit(cfg, osm.uniform_tables(nb), bins, lnL, lw)
        e = lnL + lw
        M = max(e)
        for j in range(3):
            H = [0] * nb
            for a in range(n):
                H[bins[a, j]] += int(round(math.exp(temper * (e[a] - M)) * 2 ** 40)) if np.isfinite(e[a]) else 0
            tot = sum(H)
            want = np.array([(1 - cfg["floor_frac"]) * nb * (x / tot) + cfg["floor_frac"] for x in H])
            assert np.max(np.abs(h[j] - want)) < 1e-12
            assert abs(h[j].sum() / nb - 1.0) < 1e-13               # normalised: sum h / n_bins = 1
            assert h[j].min() >= cfg["floor_frac"] - 1e-15           # the floor keeps every bin reachable
            assert abs(osm.cumulative(h[j])[-1] - 1.0) < 1e-13
    # exact: two samples, lnL differing by ln 2, in bins 3 and 7 -> H ratio 2 : 1 (temper 1), sqrt(2) : 1 (temper 1/2)
    b2 = np.array([[3, 3, 3], [7, 7, 7]], dtype=np.int32)
    for temper, ratio in ((1.0, 2.0), (0.5, math.sqrt(2.0))):
        cfg = dict(CFG, temper=temper, floor_frac=0.0)
        h = osm.refit(cfg, osm.uniform_tables(nb), b2, np.array([math.log(2.0), 0.0]), np.zeros(2))
        assert abs(h[0][3] / h[0][7] - ratio) < 1e-11 and h[0][0] == 0.0
    # no finite sample: densities unchanged; a non-adaptive dimension is never touched
    h0 = np.full((3, nb), 1.0)
    assert np.array_equal(osm.refit(CFG, h0, bins, np.full(n, -np.inf), lw), h0)
    cfg = dict(CFG, adapt=(True, True, False))
    assert np.array_equal(osm.refit(cfg, h0, bins, lnL, lw)[2], h0[2])


# ----------------------------------------------------------------------------------------------------------
# S7-S8: the loop
# ----------------------------------------------------------------------------------------------------------
def _eval(cfg_ile):
    return lambda s: oracle.eval_batch(cfg_ile, s, n_threads=8)[0]


def _quiet_config(snr):
    """Config 0's shapes with a weaker injection: at SNR 15 a prior-sampled evidence has n_eff ~ 1 and no usable error
    bar; at SNR 5-6 plain Monte Carlo converges (n_eff of tens to hundreds per 2e5 draws), so estimates can be compared."""
    base = gi.make_config(0)
    c = gi.CONFIGS[0]
    Q, U, V, _ = gi.make_point(4321, c["dets"], c["modes"], c["n_q"], snr)
    cfg = dict(base)
    cfg.update(Q=Q[None], U=U[None], V=V[None])
    return cfg


def test_prior_run_reproduces_the_evidence_of_the_existing_path():
    """adapt off: the loop is plain Monte Carlo from the prior, so lnZ agrees with the evidence of an INDEPENDENT prior
    batch from the seeded generator (the existing path's inputs) within Monte Carlo error (relative error of Z about
    1/sqrt(n_eff), L101)."""
    ile_cfg = _quiet_config(5.0)
    cfg = dict(CFG, adapt=(False, False, False))
    r = osm.integrate(cfg, _eval(ile_cfg), n_chunk=20_000, max_chunks=10, n_adapt_chunks=0, n_eff_min=1e30)
    assert r["n_samples"] == 200_000 and r["n_chunks"] == 10
    ref = oracle.eval_batch(ile_cfg, gi.make_samples(777, 200_000), n_threads=8)[0]
    rZ, rN = oracle.evidence(ref)
    sigma = math.sqrt(1.0 / r["n_eff"] + 1.0 / rN)
    assert abs(r["lnZ"] - rZ) < 4.0 * sigma, (r["lnZ"], rZ, sigma)
    # the history is the running evidence: its last entry is the evidence of everything drawn so far
    s_all = [osm.draw(cfg, osm.uniform_tables(cfg["n_bins"]), c * 20_000, 20_000)[0] for c in range(10)]
    every = np.concatenate([_eval(ile_cfg)(s) for s in s_all])
    z, ne = oracle.evidence(every)
    assert abs(z - r["lnZ"]) < 1e-10 * max(abs(z), 1) and abs(ne - r["n_eff"]) < 1e-9 * ne


def _gauss_lnL(sig=0.03, c=(0.3, 0.6, 0.2)):
    """A synthetic likelihood that depends on the three adaptive coordinates only: a Gaussian of width sig in (u0, u1, u6)
    well inside the unit cube, so that Z = int L p = (2 pi sig^2)^(3/2) in closed form."""
    def f(s):
        u0 = s["ra"] / (2 * np.pi)
        u1 = (np.sin(s["dec"]) + 1) / 2
        u6 = (s["dist_mpc"] ** 3 - 1.0) / (1000.0 ** 3 - 1.0)
        return -((u0 - c[0]) ** 2 + (u1 - c[1]) ** 2 + (u6 - c[2]) ** 2) / (2 * sig * sig)
    return f, 1.5 * math.log(2 * math.pi * sig * sig)


def test_adaptive_run_closed_form_evidence_and_efficiency():
    """On a likelihood with a closed-form evidence the adaptive loop (S3-S8) stays unbiased -- lnZ within Monte Carlo error
    of ln (2 pi sig^2)^(3/2) -- and, because this likelihood lives in exactly the dimensions the sampler adapts in (L119),
    collects effective samples far faster than the prior run."""
    f, lnZ_exact = _gauss_lnL()
    r0 = osm.integrate(dict(CFG, adapt=(False, False, False)), f, 10_000, 10, 0, 1e30)
    r1 = osm.integrate(CFG, f, 10_000, 10, 10, 1e30)
    for r in (r0, r1):
        assert abs(r["lnZ"] - lnZ_exact) < 5.0 / math.sqrt(r["n_eff"]), (r["lnZ"], lnZ_exact, r["n_eff"])
    # n_eff = sum / max over ALL samples is capped by the first (prior-drawn) chunk's best sample, so efficiency is
    # measured on a fresh batch: drawn from the adapted densities it is worth >= 20x as many effective samples as one
    # drawn from the prior
    def batch_neff(h):
        sb, lwb, _, _ = osm.draw(dict(CFG, seed=4242), h, 0, 50_000)
        e = f(sb) + lwb
        return float(np.sum(np.exp(e - e.max())))
    assert batch_neff(r1["h"]) > 20.0 * batch_neff(osm.uniform_tables(CFG["n_bins"]))
    assert r1["n_eff"] > r0["n_eff"]
    assert all(abs(h.sum() / CFG["n_bins"] - 1.0) < 1e-12 for h in r1["h"])
    # the adapted densities peak in the bins that hold the likelihood's centre
    for j, c in enumerate((0.3, 0.6, 0.2)):
        assert abs(int(np.argmax(r1["h"][j])) - int(c * CFG["n_bins"])) <= 1
    # S8: the stopping rule ends the loop at the first chunk whose n_eff reaches the threshold
    thr = r1["history"][4][1]
    r2 = osm.integrate(CFG, f, 10_000, 10, 10, thr)
    first = next(i for i, (_, ne) in enumerate(r1["history"]) if ne >= thr)
    assert r2["n_chunks"] == first + 1 and r2["lnZ"] == r1["history"][first][0] and r2["n_samples"] == 10_000 * (first + 1)
    # S7: n_adapt_chunks = 2 freezes the densities after the second refit
    r3 = osm.integrate(CFG, f, 10_000, 6, 2, 1e30)
    r4 = osm.integrate(CFG, f, 10_000, 2, 2, 1e30)
    assert np.array_equal(r3["h"], r4["h"])


def test_adaptive_run_on_the_ile_likelihood_is_unbiased():
    """The same loop on the hot path's likelihood (a quiet injection so that both estimates have an error bar)."""
    ile_cfg = _quiet_config(6.0)
    r0 = osm.integrate(dict(CFG, adapt=(False, False, False)), _eval(ile_cfg), 10_000, 20, 0, 1e30)
    r1 = osm.integrate(dict(CFG, temper=0.2), _eval(ile_cfg), 10_000, 20, 20, 1e30)
    sigma = math.sqrt(1.0 / r0["n_eff"] + 1.0 / r1["n_eff"])
    assert abs(r1["lnZ"] - r0["lnZ"]) < 4.0 * sigma, (r0["lnZ"], r1["lnZ"], sigma)
