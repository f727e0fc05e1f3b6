"""GPU-vs-oracle parity of the posterior harvesting (NEXT-3) through the C ABI: ile_resample and ile_harvest against
oracle/harvest.py (which reads the lnL_j series from the hot-path oracle).

Bar: indices are integers -> bit-exact wherever the decision is unique.  A decision taken by comparing floating-point
numbers (which bin holds the maximum, where a cumulative crosses a threshold) is unique unless the two sides of the
comparison agree to within the hot path's own tolerance; there both answers are correct (the prompt's "compare what is unique
and check that the rest is valid"): the test then requires the GPU's choice to be a neighbour that the oracle's numbers
cannot tell apart at 1e-10."""
import numpy as np
import pytest

import ile_inputs as gi
import oracle
from oracle import harvest as oh
from parity_util import ORACLE_THREADS, TOL, rel_err

pytestmark = pytest.mark.gpu


def to_dev(s):
    import torch

    return {k: torch.from_numpy(v).cuda() for k, v in s.items()}


@pytest.mark.parametrize("n,n_out", [(5_000, 1_777), (100_000, 20_000), (1_000_003, 50_000), (7, 40), (1, 3)])
def test_resample_matches_the_oracle(gpu_lib, n, n_out):
    import torch

    cfg = gi.make_config(0)
    ctx = gpu_lib.Context(cfg)
    rng = np.random.default_rng(n)
    lnL = rng.normal(0, 4, n)
    lw = rng.normal(0, 1, n)
    lnL[::41] = -np.inf
    if n == 1:
        lnL[0] = 0.3
    for v0 in (0.0, 0.37, 0.999999):
        for use_w in (True, False):
            ids = ctx.resample(torch.from_numpy(lnL).cuda(), torch.from_numpy(lw).cuda() if use_w else None, n_out, v0).cpu().numpy()
            ref = oh.systematic_resample(lnL, lw if use_w else None, n_out, v0)
            assert len(ids) == n_out and np.all(np.diff(ids) >= 0)
            diff = np.flatnonzero(ids != ref)
            if len(diff):  # only where the point (i + v0) / n_out sits on a cumulative edge to within rounding
                cdf = oh.resample_cdf(lnL, lw if use_w else None)
                for i in diff:
                    p = (i + v0) / n_out
                    lo, hi = sorted((ids[i], ref[i]))
                    assert np.all(np.abs(cdf[lo:hi] - p) <= 1e-12), (i, ids[i], ref[i])
            assert len(diff) <= max(1, n_out // 10_000)
    none = ctx.resample(torch.full((50,), float("-inf"), dtype=torch.float64, device="cuda"), None, 10, 0.5).cpu().numpy()
    assert np.all(none == -1) and len(oh.systematic_resample(np.full(50, -np.inf), None, 10, 0.5)) == 0
    ctx.close()


@pytest.mark.parametrize("cid,shift_mode", [(0, 0), (1, 0), (2, 0), (0, 1), (1, 1)])
def test_harvest_matches_the_oracle_series(gpu_lib, cid, shift_mode):
    """shift_mode 1: the harvested series is the linearly interpolated one of reading R8' (oracle/subsample.py), so that the
    interpolated variant of the path (NEXT-4) has its arg-max and time draw too."""
    import torch

    from oracle import subsample as osub

    n = 600 if cid < 2 else 150
    cfg = gi.make_config(cid, n=n)
    cfg["shift_mode"] = shift_mode

    def series_of(sample):
        if shift_mode:
            r = osub.sample_series_lin(cfg, sample)
            return r[0], None, None, r[4]
        return oracle.sample_series(cfg, sample)

    s = gi.make_samples(cfg["sample_seeds"][0] + 3, n)
    s["t_ref"][11] = 0.9                                   # out of range: -1 / -inf / -1
    rng = np.random.default_rng(cid)
    v = rng.random(n)
    ctx = gpu_lib.Context(cfg)
    amax, lmax, drawn = ctx.harvest(to_dev(s), v=torch.from_numpy(v).cuda())
    amax, lmax, drawn = amax.cpu().numpy(), lmax.cpu().numpy(), drawn.cpu().numpy()
    n_amb = 0
    for a in range(n):
        series, _, _, oob = series_of({k: s[k][a] for k in s})
        if oob:
            assert amax[a] == -1 and drawn[a] == -1 and lmax[a] == -np.inf
            continue
        j, val = oh.argmax_bin(series)
        scale = max(abs(val), 1.0)
        assert abs(lmax[a] - val) <= TOL * scale
        if amax[a] != j:                                   # two bins the oracle itself cannot tell apart at 1e-10
            assert abs(series[amax[a]] - val) <= TOL * scale
            n_amb += 1
        jd = oh.draw_time_bin(series, v[a])
        if drawn[a] != jd:
            cdf = oh.time_cdf(series)
            lo, hi = sorted((drawn[a], jd))
            assert np.all(np.abs(cdf[lo:hi] - v[a]) <= 1e-10), (a, drawn[a], jd)
            n_amb += 1
    assert n_amb <= 2
    assert series_of({k: s[k][11] for k in s})[3]
    ctx.close()


def test_resample_then_harvest_chain(gpu_lib):
    """The final iteration as a user runs it: ile_eval -> ile_resample (ids on the device) -> ile_harvest(ids): equal-weight
    posterior samples with their best-fit and drawn time bins, all compared with the oracle chain."""
    import torch

    cfg = gi.make_config(1, n=30_000)
    s = gi.make_samples(cfg["sample_seeds"][0], cfg["n"])
    lw = gi.make_log_weights(8, cfg["n"])
    ctx = gpu_lib.Context(cfg)
    d = to_dev(s)
    lnL, _ = ctx.eval(d, want_idx=False)
    lwd = torch.from_numpy(lw).cuda()
    n_out = 400
    ids = ctx.resample(lnL, lwd, n_out, 0.25)
    v = torch.from_numpy(np.random.default_rng(4).random(n_out)).cuda()
    amax, lmax, drawn = ctx.harvest(d, ids=ids, v=v)
    ref = oracle.eval_batch(cfg, s, n_threads=ORACLE_THREADS)[0]
    rids = oh.systematic_resample(ref, lw, n_out, 0.25)
    ids = ids.cpu().numpy()
    assert np.mean(ids == rids) >= 0.99                      # the GPU's lnL differs from the oracle's in the 13th digit
    vv = v.cpu().numpy()
    for i in range(0, n_out, 7):
        a = int(ids[i])
        series = oracle.sample_series(cfg, {k: s[k][a] for k in s})[0]
        j, val = oh.argmax_bin(series)
        assert abs(lmax[i].item() - val) <= TOL * max(abs(val), 1.0)
        assert amax[i].item() == j or abs(series[amax[i].item()] - val) <= TOL * max(abs(val), 1.0)
        jd = oh.draw_time_bin(series, vv[i])
        if drawn[i].item() != jd:
            cdf = oh.time_cdf(series)
            lo, hi = sorted((drawn[i].item(), jd))
            assert np.all(np.abs(cdf[lo:hi] - vv[i]) <= 1e-10)
    # bad ids are flagged, not dereferenced
    bad = torch.tensor([-1, cfg["n"], 5], dtype=torch.int64, device="cuda")
    am, lm, _ = ctx.harvest(d, ids=bad)
    assert am[0].item() == -1 and am[1].item() == -1 and am[2].item() >= 0
    ctx.close()
