"""GPU-vs-oracle parity of the on-device sampler (NEXT-2) through the C ABI: ile_sampler_* and ile_integrate against
oracle/sampler.py on the same seeds and the same density tables.

Bar: the Philox stream and the histogram bin indices are integers / exact binary64 values -> bit-exact; unit-cube
coordinates come from individually rounded operations in a fixed order -> bit-exact; physical parameters pass through
asin / acos / cbrt and ln w through log, whose last bit differs between libm and CUDA -> 1e-14 relative (parameters), 1e-10
(ln w, densities).  Through the adaptive loop the GPU's own lnL (equal to the oracle's within 1e-10, not bit for bit) feeds
the refit, so densities are compared at 1e-9 and the evidence at the hot path's 1e-10 scaled by the run length."""
import numpy as np
import pytest

import ile_inputs as gi
import oracle
from oracle import sampler as osm
from parity_util import ORACLE_THREADS, TOL, rel_err

pytestmark = pytest.mark.gpu

CFG = dict(seed=0xC0FFEE1234567, n_bins=64, adapt=(True, True, True), dist_min_mpc=1.0, dist_max_mpc=1000.0,
           t_ref_lo_s=-0.05, t_ref_hi_s=0.05, floor_frac=0.1, temper=1.0)


def random_tables(seed, nb):
    rng = np.random.default_rng(seed)
    h = rng.uniform(0.05, 4.0, size=(3, nb))
    return h / h.mean(axis=1, keepdims=True)


def test_uniforms_bit_exact(gpu_lib):
    smp = gpu_lib.Sampler(CFG)
    for first, n in ((0, 100_003), (2 ** 32 - 7, 4_000), (2 ** 40 + 1, 1_000)):   # across and beyond the 32-bit counter word
        got = smp.uniforms(first, n).cpu().numpy()
        assert np.array_equal(got, osm.uniforms(CFG["seed"], first, n))
    smp.close()


@pytest.mark.parametrize("nb,adapt", [(64, (True, True, True)), (1, (True, True, True)), (100, (True, False, True)),
                                      (512, (True, True, True)), (7, (False, False, False))])
def test_draw_matches_the_oracle(gpu_lib, nb, adapt):
    cfg = dict(CFG, n_bins=nb, adapt=adapt, dist_min_mpc=3.5, dist_max_mpc=870.25, t_ref_lo_s=-0.013, t_ref_hi_s=0.021)
    smp = gpu_lib.Sampler(cfg)
    for h in (osm.uniform_tables(nb), random_tables(nb, nb)):
        smp.set_tables(h)
        hg, Cg = smp.get_tables()
        assert np.array_equal(hg, h)
        for j in range(3):
            assert np.array_equal(Cg[j], osm.cumulative(h[j]))          # sequential sum: bit-exact
        n, first = 50_001, 123_456_789
        s, lw, bins = smp.draw(first, n)
        rs, rlw, rbins, ru = osm.draw(cfg, h, first, n)
        assert np.array_equal(bins.cpu().numpy(), rbins)                  # bin indices bit-exact
        # unit-cube coordinates recovered from the parameters that are exact products of them
        assert np.array_equal(s["ra"].cpu().numpy(), rs["ra"]) and np.array_equal(s["phi_ref"].cpu().numpy(), rs["phi_ref"])
        assert np.array_equal(s["psi"].cpu().numpy(), rs["psi"]) and np.array_equal(s["t_ref"].cpu().numpy(), rs["t_ref"])
        for k in ("dec", "incl", "dist_mpc"):
            got = s[k].cpu().numpy()
            assert np.max(np.abs(got - rs[k]) / np.maximum(np.abs(rs[k]), 1.0)) <= 1e-14, k
        assert rel_err(rlw, lw.cpu().numpy()) <= TOL
    smp.close()


def test_refit_matches_the_oracle(gpu_lib):
    import torch

    rng = np.random.default_rng(3)
    for nb, n, temper, fl in ((64, 10_000, 1.0, 0.1), (512, 100_000, 0.3, 0.02), (16, 777, 1.0, 0.0)):
        cfg = dict(CFG, n_bins=nb, temper=temper, floor_frac=fl, adapt=(True, False, True))
        smp = gpu_lib.Sampler(cfg)
        h0 = random_tables(9, nb)
        smp.set_tables(h0)
        bins = rng.integers(0, nb, size=(n, 3)).astype(np.int32)
        lnL = rng.normal(0, 4, n)
        lnL[::53] = -np.inf
        lw = rng.normal(0, 0.7, n)
        smp.refit(torch.from_numpy(bins).cuda(), torch.from_numpy(lnL).cuda(), torch.from_numpy(lw).cuda())
        hg, Cg = smp.get_tables()
        hr = osm.refit(cfg, h0, bins, lnL, lw)
        assert np.max(np.abs(hg - hr) / np.maximum(hr, 1.0)) <= TOL
        assert np.array_equal(hg[1], h0[1])                               # the non-adaptive dimension is untouched
        for j in range(3):
            assert np.array_equal(Cg[j], osm.cumulative(hg[j]))
            assert abs(hg[j].sum() / nb - 1.0) < 1e-12
        # no finite sample: unchanged
        smp.refit(torch.from_numpy(bins).cuda(), torch.full((n,), float("-inf"), dtype=torch.float64, device="cuda"), None)
        assert np.array_equal(smp.get_tables()[0], hg)
        smp.close()


def test_draw_eval_evidence_chain_on_device_equals_oracle_chain(gpu_lib):
    """One adaptive step by hand through the public entries: draw -> ile_eval -> ile_evidence(log_w) -> refit -> draw."""
    cfg_ile = gi.make_config(1, n=20_000)
    ctx = gpu_lib.Context(cfg_ile)
    smp = gpu_lib.Sampler(CFG)
    n = 20_000
    s, lw, bins = smp.draw(0, n)
    lnL, _ = ctx.eval(s, want_idx=False)
    lnZ, neff = ctx.evidence(lnL, lw)
    rs, rlw, rbins, _ = osm.draw(CFG, osm.uniform_tables(CFG["n_bins"]), 0, n)
    ref = oracle.eval_batch(cfg_ile, rs, n_threads=ORACLE_THREADS)[0]
    assert rel_err(ref, lnL.cpu().numpy()) <= TOL
    rZ, rN = oracle.evidence(ref, rlw)
    assert rel_err([rZ], lnZ.cpu().numpy()) <= TOL and rel_err([rN], neff.cpu().numpy()) <= TOL
    smp.refit(bins, lnL, lw)
    hr = osm.refit(CFG, osm.uniform_tables(CFG["n_bins"]), rbins, ref, rlw)
    hg, _ = smp.get_tables()
    assert np.max(np.abs(hg - hr) / np.maximum(hr, 1.0)) <= 1e-9
    s2, lw2, bins2 = smp.draw(n, n)
    rs2, rlw2, rbins2, _ = osm.draw(CFG, hr, n, n)
    assert np.mean(bins2.cpu().numpy() == rbins2) > 0.9999               # a bin flips only if v sits within 1e-9 of an edge
    assert np.max(np.abs(lw2.cpu().numpy() - rlw2)) <= 1e-8
    ctx.close()
    smp.close()


@pytest.mark.parametrize("case", ["config0_adaptive", "config1_streaming", "stop_rule", "prior_only"])
def test_integrate_matches_the_oracle_loop(gpu_lib, case):
    """Tolerances in north_star's terms (lnL and log-evidence within 1e-10 relative, fp64): a run that never refits
    (prior_only) and the FIRST chunk of every run, which is drawn from the prior, are held to TOL = 1e-10.  Later chunks of
    an adaptive run are held to 1e-9, ten times looser than north_star, and this is the only place in the suite where that
    happens: the refit turns the GPU's own lnL (within 1e-10 of the oracle's, not bit-equal) into INTEGER histogram counts
    rint(W 2^40) (reading S6), whose roundings differ on a few samples per chunk, so the two sides draw later chunks from
    densities that agree to ~1e-10, not exactly; a sample within that distance of a bin edge changes bin, and its ln w with
    it.  The refit densities themselves are compared at 1e-8 below for the same reason, and the sampler's
    own pieces (draws, bins, weights, one refit from identical inputs) are bit-exact / 1e-10 in the tests above."""
    if case == "config1_streaming":      # chunks of 20,000: every ile_eval takes the sorted streaming path
        cfg_ile, n_chunk, max_chunks, n_adapt, thr, scfg = gi.make_config(1, n=1), 20_000, 5, 5, 1e30, dict(CFG, temper=0.5)
    elif case == "config0_adaptive":     # the paper's block size (L97, L119)
        cfg_ile, n_chunk, max_chunks, n_adapt, thr, scfg = gi.make_config(0), 10_000, 8, 3, 1e30, CFG
    elif case == "prior_only":
        cfg_ile, n_chunk, max_chunks, n_adapt, thr, scfg = gi.make_config(0), 4_001, 6, 0, 1e30, dict(CFG, adapt=(False, False, False))
    else:
        cfg_ile, n_chunk, max_chunks, n_adapt, scfg = gi.make_config(0), 10_000, 12, 12, CFG
        thr = None
    ev = lambda s: oracle.eval_batch(cfg_ile, s, n_threads=ORACLE_THREADS)[0]
    if thr is None:  # a threshold that the oracle's run crosses in its 5th chunk
        full = osm.integrate(scfg, ev, n_chunk, max_chunks, n_adapt, 1e30)
        thr = 0.5 * (full["history"][3][1] + full["history"][4][1]) if full["history"][4][1] > full["history"][3][1] else full["history"][4][1]
    r = osm.integrate(scfg, ev, n_chunk, max_chunks, n_adapt, thr)
    ctx = gpu_lib.Context(cfg_ile)
    smp = gpu_lib.Sampler(scfg)
    g = gpu_lib.integrate(ctx, smp, n_chunk, max_chunks, n_adapt, thr)
    assert g["n_chunks"] == r["n_chunks"] and g["n_samples"] == r["n_samples"]
    rh = np.array(r["history"])
    tol = 1e-9 if n_adapt else TOL
    assert np.max(np.abs(g["history"][0] - rh[0]) / np.maximum(np.abs(rh[0]), 1.0)) <= TOL   # chunk 0: prior draws, north_star's bar
    assert np.max(np.abs(g["history"][:, 0] - rh[:, 0]) / np.maximum(np.abs(rh[:, 0]), 1.0)) <= tol
    assert np.max(np.abs(g["history"][:, 1] - rh[:, 1]) / np.maximum(np.abs(rh[:, 1]), 1.0)) <= tol
    assert abs(g["lnZ"] - r["lnZ"]) <= tol * max(abs(r["lnZ"]), 1.0)
    hg, _ = smp.get_tables()
    assert np.max(np.abs(hg - r["h"]) / np.maximum(r["h"], 1.0)) <= 1e-8
    n_bad, _ = ctx.status()
    assert n_bad == 0
    ctx.close()
    smp.close()
