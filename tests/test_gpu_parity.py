"""GPU-vs-oracle parity through the C ABI (pytest -m gpu, on a B200).

Same seeded inputs go to both sides.  Bar (north_star): shift indices bit-exact as integers; lnL_margT, lnZ, n_eff
within TOL = 1e-10 * max(|ref|, 1).  All five BASELINE.json configs are run at FULL size in the launch configuration
bench.py times and compared element by element with the oracle (every lnL_margT, every index, every lnZ / n_eff).
"""
import numpy as np
import pytest

import ile_inputs as gi
import oracle
from parity_util import ORACLE_THREADS, TOL, assert_indices_equal, rel_err, subset

pytestmark = pytest.mark.gpu


def to_dev(s):
    import torch

    return {k: torch.from_numpy(v).cuda() for k, v in s.items()}


def run_gpu(ile, cfg, samples, point=0, variant=0):
    ctx = ile.Context(cfg)
    if variant:
        ctx.set_variant(variant)
    lnL, idx = ctx.eval(to_dev(samples), point=point)
    n_bad, _ = ctx.status()
    return ctx, lnL, idx, n_bad


def full_compare(ile, cfg, samples, point=0, variant=0, log_w=None):
    import torch

    ctx, lnL, idx, n_bad = run_gpu(ile, cfg, samples, point, variant)
    ref, ref_idx, ref_bad = oracle.eval_batch(cfg, samples, point=point, n_threads=ORACLE_THREADS)
    assert n_bad == ref_bad
    assert_indices_equal(cfg, samples, ref_idx, idx.cpu().numpy())
    e = rel_err(ref, lnL.cpu().numpy())
    assert e <= TOL, f"lnL_margT rel err {e:.3e}"
    lw = None if log_w is None else torch.from_numpy(log_w).cuda()
    lnZ, neff = ctx.evidence(lnL, lw)
    rZ, rN = oracle.evidence(ref, log_w)
    assert rel_err([rZ], lnZ.cpu().numpy()) <= TOL
    assert rel_err([rN], neff.cpu().numpy()) <= TOL
    ctx.close()
    return e


# ---------------------------------------------------------------------------------------------- configs 0, 1
def test_config0_full(gpu_lib):
    cfg = gi.make_config(0)
    s = gi.make_samples(cfg["sample_seeds"][0], cfg["n"])
    full_compare(gpu_lib, cfg, s)


def test_config1_full(gpu_lib):
    cfg = gi.make_config(1)
    s = gi.make_samples(cfg["sample_seeds"][0], cfg["n"])
    full_compare(gpu_lib, cfg, s)


def test_config1_concentrated_and_weighted(gpu_lib):
    cfg = gi.make_config(1)
    s = gi.make_concentrated_samples(cfg["sample_seeds"][0] + 1, 20_000)
    lw = gi.make_log_weights(cfg["sample_seeds"][0] + 2, 20_000)
    full_compare(gpu_lib, cfg, s, log_w=lw)


# ---------------------------------------------------------------------------------------------- config 2 (21 modes)
def test_config2_small_elementwise(gpu_lib):
    cfg = gi.make_config(2)
    s = gi.make_samples(cfg["sample_seeds"][0], 3_001)       # several tiles and a ragged tail
    full_compare(gpu_lib, cfg, s)


def test_config2_full_size_every_sample(gpu_lib):
    """BASELINE.json configs[2] at full size (1,000,000 samples, 21 modes) in the launch configuration bench.py times:
    EVERY lnL_margT and EVERY shift index against the oracle, lnZ / n_eff against oracle.evidence of the whole set,
    chunked evidence against the same oracle values."""
    cfg = gi.make_config(2)
    n = cfg["n"]
    s = gi.make_samples(cfg["sample_seeds"][0], n)
    ctx, lnL, idx, n_bad = run_gpu(gpu_lib, cfg, s)
    ref, ref_idx, ref_bad = oracle.eval_batch(cfg, s, n_threads=ORACLE_THREADS)
    assert n_bad == ref_bad == 0
    assert_indices_equal(cfg, s, ref_idx, idx.cpu().numpy())
    assert rel_err(ref, lnL.cpu().numpy()) <= TOL
    rZ, rN = oracle.evidence(ref)
    lnZ, neff = ctx.evidence(lnL)
    assert rel_err([rZ], lnZ.cpu().numpy()) <= TOL and rel_err([rN], neff.cpu().numpy()) <= TOL
    st = ctx.new_state()
    for lo in range(0, n, 300_000):
        lnZc, neffc = ctx.evidence(lnL[lo:lo + 300_000].contiguous(), state=st)
    assert rel_err([rZ], lnZc.cpu().numpy()) <= TOL and rel_err([rN], neffc.cpu().numpy()) <= TOL
    ctx.close()


# ---------------------------------------------------------------------------------------------- config 3 (batch sweep)
@pytest.mark.parametrize("n", [1_000, 10_000, 100_000])
def test_config3_sweep_elementwise(gpu_lib, n):
    cfg = gi.make_config(3, n=n)
    s = gi.make_samples(cfg["sample_seeds"][0], n)
    full_compare(gpu_lib, cfg, s)


def test_config3_1e6_evidence_parity(gpu_lib):
    cfg = gi.make_config(3, n=1_000_000)
    s = gi.make_samples(cfg["sample_seeds"][0], cfg["n"])
    full_compare(gpu_lib, cfg, s)


def test_config3_1e7_chunked_from_one_stream_every_sample(gpu_lib):
    """Largest batch (1e7): processed in chunks on one stream with the evidence state carried on the device.  EVERY
    lnL_margT and EVERY shift index against the oracle; the chunked lnZ / n_eff against the oracle's evidence of the
    whole set."""
    import torch

    cfg = gi.make_config(3)
    n, chunk = cfg["n"], 1_000_000
    s = gi.make_samples(cfg["sample_seeds"][0], n)
    ctx = gpu_lib.Context(cfg)
    st = ctx.new_state()
    out = torch.empty(n, dtype=torch.float64, device="cuda")
    idx = torch.empty((n, cfg["n_det"]), dtype=torch.int32, device="cuda")
    for lo in range(0, n, chunk):
        d = to_dev(subset(s, slice(lo, lo + chunk)))
        _, ix = ctx.eval(d, want_idx=True, out=out[lo:lo + chunk])
        idx[lo:lo + chunk].copy_(ix)
        lnZc, neffc = ctx.evidence(out[lo:lo + chunk], state=st)
    n_bad, _ = ctx.status()
    ref, ref_idx, ref_bad = oracle.eval_batch(cfg, s, n_threads=ORACLE_THREADS)
    assert n_bad == ref_bad == 0
    assert abs(st.cpu().numpy()[0, 2] - n) == 0
    assert_indices_equal(cfg, s, ref_idx, idx.cpu().numpy())
    assert rel_err(ref, out.cpu().numpy()) <= TOL
    rZ, rN = oracle.evidence(ref)
    assert rel_err([rZ], lnZc.cpu().numpy()) <= TOL and rel_err([rN], neffc.cpu().numpy()) <= TOL
    lnZ, neff = ctx.evidence(out)                       # one call over the whole set
    assert rel_err([rZ], lnZ.cpu().numpy()) <= TOL and rel_err([rN], neff.cpu().numpy()) <= TOL
    ctx.close()


def test_one_call_above_the_launch_group_size_every_sample(gpu_lib):
    """ONE ile_eval call and ONE ile_run_host call with n = 2,500,000 on config 3's shape: more than the 1,048,576 samples
    of a launch group, so the library itself cuts the call into three groups with shifted pointers, the last one ragged
    (the paths bench.py --config 3 --n 10000000 takes).  EVERY lnL_margT, EVERY shift index, lnZ and n_eff against the
    oracle (eq. 7, 9: L64-L67, L81-L86; eq. 4: L42-L47)."""
    import torch

    n = 2_500_000
    cfg = gi.make_config(3, n=n)
    s = gi.make_samples(cfg["sample_seeds"][0], n)
    lw = gi.make_log_weights(9, n)
    ref, ref_idx, ref_bad = oracle.eval_batch(cfg, s, n_threads=ORACLE_THREADS)
    rZ, rN = oracle.evidence(ref, lw)
    ctx = gpu_lib.Context(cfg)
    lnL, idx = ctx.eval(to_dev(s), want_idx=True)                      # one call, three launch groups
    n_bad, _ = ctx.status()
    assert n_bad == ref_bad == 0
    assert_indices_equal(cfg, s, ref_idx, idx.cpu().numpy())
    assert rel_err(ref, lnL.cpu().numpy()) <= TOL
    lnZ, neff = ctx.evidence(lnL, torch.from_numpy(lw).cuda())
    assert rel_err([rZ], lnZ.cpu().numpy()) <= TOL and rel_err([rN], neff.cpu().numpy()) <= TOL
    del lnL, idx
    host = {k: torch.from_numpy(v).pin_memory() for k, v in s.items()}
    out, lnZh, neffh = ctx.run_host(host, torch.from_numpy(lw).pin_memory())   # one call from host buffers
    assert rel_err(ref, out.numpy()) <= TOL
    assert rel_err([rZ], [lnZh]) <= TOL and rel_err([rN], [neffh]) <= TOL
    ctx.close()


# ---------------------------------------------------------------------------------------------- config 4 (many points)
def test_config4_small_all_points_elementwise(gpu_lib):
    import torch

    cfg = gi.make_config(4, n=777, n_points=5)
    P, n = cfg["n_points"], cfg["n"]
    per = [gi.make_samples(cfg["sample_seeds"][p], n) for p in range(P)]
    allS = {k: np.ascontiguousarray(np.stack([per[p][k] for p in range(P)])) for k in per[0]}
    ctx = gpu_lib.Context(cfg)
    lnL, idx = ctx.eval_all(to_dev(allS), want_idx=True)
    lnZ, neff = ctx.evidence(lnL, n_segments=P)
    for p in range(P):
        ref, ref_idx, _ = oracle.eval_batch(cfg, per[p], point=p, n_threads=ORACLE_THREADS)
        assert_indices_equal(cfg, per[p], ref_idx, idx[p].cpu().numpy())
        assert rel_err(ref, lnL[p].cpu().numpy()) <= TOL
        rZ, rN = oracle.evidence(ref)
        assert rel_err([rZ], lnZ[p:p + 1].cpu().numpy()) <= TOL
        assert rel_err([rN], neff[p:p + 1].cpu().numpy()) <= TOL
        # single-point entry gives the same numbers as the all-points launch, up to the summation order of the
        # log-sum-exp (the sorted kernel splits a window over warps by the tile's time range, and the order of equal
        # keys in its counting sort is free): a few ulp, far inside TOL
        one, _ = ctx.eval(to_dev(per[p]), point=p, want_idx=False)
        assert rel_err(lnL[p].cpu().numpy(), one.cpu().numpy()) <= 1e-13
    ctx.close()


def test_config4_full_size_every_point(gpu_lib):
    """BASELINE.json configs[4] at full size: 256 intrinsic points x 100,000 samples in one ile_eval_all, as bench.py
    --config 4 --points 256 launches it.  EVERY lnL_margT and shift index of EVERY point against the oracle, and all
    256 lnZ / n_eff."""
    import torch

    cfg = gi.make_config(4)
    P, n = cfg["n_points"], cfg["n"]
    ctx = gpu_lib.Context(cfg)
    dev = {k: torch.empty((P, n), dtype=torch.float64, device="cuda") for k in gi.SAMPLE_FIELDS}
    per = []
    for p in range(P):
        s = gi.make_samples(cfg["sample_seeds"][p], n)
        per.append(s)
        for k in gi.SAMPLE_FIELDS:
            dev[k][p].copy_(torch.from_numpy(s[k]))
    lnL, idx = ctx.eval_all(dev, want_idx=True)
    lnZ, neff = ctx.evidence(lnL, n_segments=P)
    n_bad, _ = ctx.status()
    assert n_bad == 0
    got, got_idx = lnL.cpu().numpy(), idx.cpu().numpy()
    gZ, gN = lnZ.cpu().numpy(), neff.cpu().numpy()
    worst = 0.0
    for p in range(P):
        ref, ref_idx, ref_bad = oracle.eval_batch(cfg, per[p], point=p, n_threads=ORACLE_THREADS)
        assert ref_bad == 0
        assert_indices_equal(cfg, per[p], ref_idx, got_idx[p])
        e = rel_err(ref, got[p])
        worst = max(worst, e)
        assert e <= TOL, f"point {p}: lnL_margT rel err {e:.3e}"
        rZ, rN = oracle.evidence(ref)
        assert rel_err([rZ], gZ[p:p + 1]) <= TOL, f"point {p}: lnZ"
        assert rel_err([rN], gN[p:p + 1]) <= TOL, f"point {p}: n_eff"
    ctx.close()


# ---------------------------------------------------------------------------------------------- edge cases
# Every edge case runs through the automatic choice (small n: the tiled / direct kernels) AND through the streaming
# FP64-MMA kernel (variant 4), which is what every production-size batch uses.
VARIANTS = [0, 4]


@pytest.mark.parametrize("variant", VARIANTS)
def test_edge_empty_one_and_ragged(gpu_lib, variant):
    import torch

    cfg = gi.make_config(0)
    ctx = gpu_lib.Context(cfg)
    if variant:
        ctx.set_variant(variant)
    empty = {k: torch.empty(0, dtype=torch.float64, device="cuda") for k in gi.SAMPLE_FIELDS}
    lnL, idx = ctx.eval(empty)
    assert lnL.numel() == 0
    ctx.close()
    for n in (1, 7, 8, 9, 31, 33, 255, 257):
        s = gi.make_samples(99 + n, n)
        full_compare(gpu_lib, cfg, s, variant=variant)


@pytest.mark.parametrize("variant", VARIANTS)
def test_edge_out_of_range_windows(gpu_lib, variant):
    cfg = gi.make_config(0)
    s = gi.make_samples(5, 64)
    s["t_ref"][3] = 0.2
    s["t_ref"][40] = -0.2
    s["t_ref"][63] = 0.124   # window end beyond N_Q
    ctx, lnL, idx, n_bad = run_gpu(gpu_lib, cfg, s, variant=variant)
    ref, ref_idx, ref_bad = oracle.eval_batch(cfg, s)
    assert n_bad == ref_bad and ref_bad >= 2
    assert_indices_equal(cfg, s, ref_idx, idx.cpu().numpy())
    assert rel_err(ref, lnL.cpu().numpy()) <= TOL
    lnZ, neff = ctx.evidence(lnL)
    rZ, rN = oracle.evidence(ref)
    assert rel_err([rZ], lnZ.cpu().numpy()) <= TOL
    n_bad2, code = ctx.status(reset=True)
    assert n_bad2 == ref_bad and code == -5
    assert ctx.status() == (0, 0)
    ctx.close()


@pytest.mark.parametrize("variant", VARIANTS)
def test_edge_all_out_of_range_gives_minus_inf_evidence(gpu_lib, variant):
    cfg = gi.make_config(0)
    s = gi.make_samples(6, 40)
    s["t_ref"][:] = 0.3
    ctx, lnL, idx, n_bad = run_gpu(gpu_lib, cfg, s, variant=variant)
    assert n_bad == 40
    lnZ, neff = ctx.evidence(lnL)
    assert lnZ.item() == -np.inf and neff.item() == 0.0
    assert oracle.evidence(oracle.eval_batch(cfg, s)[0]) == (-np.inf, 0.0)
    ctx.close()


def test_edge_streaming_batch_touching_both_ends_of_Q(gpu_lib):
    """A production-size batch (>= 10,000 samples: the automatic choice is the streaming kernel) whose windows reach the
    first and the last stored Q sample -- the kernel then reads the zero padding in front of and behind the packed
    series -- with a few samples just out of range (reading R9: -inf + counter, never wrapped or clamped)."""
    cfg = gi.make_config(1)
    n = 20_011
    s = gi.make_samples(4242, n)
    half = (cfg["n_q"] - cfg["n_t"]) / (2.0 * cfg["fs_hz"])     # |t_ref| at which a geocentre window touches an end of Q
    rng = np.random.default_rng(7)
    edge = rng.choice(n, 3_000, replace=False)
    s["t_ref"][edge[:1400]] = half - rng.uniform(0.0, 0.03, 1400)       # delays up to +-21 ms: some leave the range
    s["t_ref"][edge[1400:2800]] = -half + rng.uniform(0.0, 0.03, 1400)
    s["t_ref"][edge[2800:]] = rng.choice([-1.0, 1.0], 200) * (half + rng.uniform(0.03, 0.2, 200))   # surely out
    ctx, lnL, idx, n_bad = run_gpu(gpu_lib, cfg, s)
    ref, ref_idx, ref_bad = oracle.eval_batch(cfg, s, n_threads=ORACLE_THREADS)
    assert n_bad == ref_bad and 200 <= ref_bad < 3_000
    i0 = ref_idx[np.isfinite(ref)]
    assert i0.min() == 0 and i0.max() == cfg["n_q"] - cfg["n_t"], "the case is meant to touch both ends of Q"
    assert_indices_equal(cfg, s, ref_idx, idx.cpu().numpy())
    assert rel_err(ref, lnL.cpu().numpy()) <= TOL
    lnZ, neff = ctx.evidence(lnL)
    rZ, rN = oracle.evidence(ref)
    assert rel_err([rZ], lnZ.cpu().numpy()) <= TOL and rel_err([rN], neff.cpu().numpy()) <= TOL
    ctx.close()


def test_edge_asymmetric_U_and_generic_V(gpu_lib):
    """Reading R15: U is not assumed Hermitian, V not assumed symmetric."""
    cfg = gi.make_config(1, n=500)
    rng = np.random.default_rng(8)
    cfg["U"] = cfg["U"] * (1.0 + 0.3 * rng.standard_normal(cfg["U"].shape)) + 50j * rng.standard_normal(cfg["U"].shape)
    cfg["V"] = cfg["V"] + 30.0 * (rng.standard_normal(cfg["V"].shape) + 1j * rng.standard_normal(cfg["V"].shape))
    s = gi.make_samples(77, 500)
    full_compare(gpu_lib, cfg, s)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("n_t", [1, 2, 7, 8, 9, 16, 32, 33, 128, 129, 1000])
def test_edge_window_lengths(gpu_lib, n_t, variant):
    cfg = gi.make_config(0, n=300)
    cfg["n_t"] = n_t
    s = gi.make_samples(123, 300)
    if n_t == 1000:
        s["t_ref"] = s["t_ref"] * 0.0   # the window nearly fills Q: only small shifts stay in range
    full_compare(gpu_lib, cfg, s, variant=variant)


@pytest.mark.parametrize("n_det", [1, 2])
@pytest.mark.parametrize("n_t", [1, 8, 33, 410])
def test_edge_streaming_kernel_one_and_two_detectors(gpu_lib, n_det, n_t):
    """The K = 1 and K = 2 instantiations of the streaming kernel (config 1 cut down to its first detectors), on a batch
    large enough for several groups per warp, window lengths below / at / above one 8-row block."""
    full = gi.make_config(1, n=5_003)
    cfg = dict(full)
    cfg.update(n_det=n_det, n_t=n_t, Q=np.ascontiguousarray(full["Q"][:, :n_det]), U=np.ascontiguousarray(full["U"][:, :n_det]),
               V=np.ascontiguousarray(full["V"][:, :n_det]), vertex_m=full["vertex_m"][:n_det], arm_x=full["arm_x"][:n_det],
               arm_y=full["arm_y"][:n_det])
    full_compare(gpu_lib, cfg, gi.make_samples(808 + n_det, 5_003), variant=4)


@pytest.mark.parametrize("variant", VARIANTS)
def test_edge_window_equals_series(gpu_lib, variant):
    """N_t = N_Q with a detector at the geocentre: the only in-range window is the whole series."""
    cfg = gi.make_config(0, n=64)
    cfg["n_t"] = cfg["n_q"]
    cfg["vertex_m"] = np.zeros_like(cfg["vertex_m"])
    s = gi.make_samples(321, 64)
    s["t_ref"][:] = 0.0
    s["t_ref"][7] = 1.0 / 4096.0   # one sample off: out of range
    ctx, lnL, idx, n_bad = run_gpu(gpu_lib, cfg, s, variant=variant)
    ref, ref_idx, ref_bad = oracle.eval_batch(cfg, s)
    assert n_bad == ref_bad == 1
    assert_indices_equal(cfg, s, ref_idx, idx.cpu().numpy())
    assert rel_err(ref, lnL.cpu().numpy()) <= TOL
    ctx.close()


def test_edge_single_detector_single_mode_and_max_sizes(gpu_lib):
    rng = np.random.default_rng(4)
    # K = 1, M = 1
    cfg = gi.make_config(0, n=100)
    one = dict(cfg)
    one.update(n_det=1, n_modes=1, Q=np.ascontiguousarray(cfg["Q"][:, :1, :1]), U=np.ascontiguousarray(cfg["U"][:, :1, :1, :1]),
               V=np.ascontiguousarray(cfg["V"][:, :1, :1, :1]), l=cfg["l"][:1], m=cfg["m"][:1], vertex_m=cfg["vertex_m"][:1],
               arm_x=cfg["arm_x"][:1], arm_y=cfg["arm_y"][:1])
    full_compare(gpu_lib, one, gi.make_samples(11, 100))
    full_compare(gpu_lib, one, gi.make_samples(11, 100), variant=4)
    # K = ILE_MAX_DET = 8 detectors, M = ILE_MAX_MODES = 32 modes (l = 2..5 truncated), generic complex inputs
    K, M, n_q = 8, 32, 512
    modes = gi.modes_up_to(5)[:M]
    big = dict(n_points=1, n_det=K, n_modes=M, n_q=n_q, n_t=65, fs_hz=4096.0, t0_q_s=-n_q / 8192.0, gmst_rad=1.0,
               d_ref_mpc=100.0, l=np.array([x[0] for x in modes], dtype=np.int32), m=np.array([x[1] for x in modes], dtype=np.int32),
               Q=(rng.standard_normal((1, K, M, n_q)) + 1j * rng.standard_normal((1, K, M, n_q))) * 3.0,
               U=(rng.standard_normal((1, K, M, M)) + 1j * rng.standard_normal((1, K, M, M))),
               V=(rng.standard_normal((1, K, M, M)) + 1j * rng.standard_normal((1, K, M, M))),
               vertex_m=6.0e6 * rng.standard_normal((K, 3)) / np.sqrt(3.0), arm_x=np.tile(cfg["arm_x"][:1], (K, 1)),
               arm_y=np.tile(cfg["arm_y"][:1], (K, 1)))
    s = gi.make_samples(12, 200)
    s["t_ref"] *= 0.2
    full_compare(gpu_lib, big, s)


def test_psi_plus_pi_invariance_on_gpu(gpu_lib):
    cfg = gi.make_config(1, n=4096)
    s = gi.make_samples(31, 4096)
    ctx = gpu_lib.Context(cfg)
    a, ia = ctx.eval(to_dev(s))
    s2 = dict(s)
    s2["psi"] = s["psi"] + np.pi
    b, ib = ctx.eval(to_dev(s2))
    assert (ia == ib).all()
    assert rel_err(a.cpu().numpy(), b.cpu().numpy()) <= 1e-11
    ctx.close()


def test_run_host_matches_device_path(gpu_lib):
    import torch

    cfg = gi.make_config(1, n=50_000)
    s = gi.make_samples(cfg["sample_seeds"][0], cfg["n"])
    lw = gi.make_log_weights(5, cfg["n"])
    ctx = gpu_lib.Context(cfg)
    host = {k: torch.from_numpy(v).pin_memory() for k, v in s.items()}
    out, lnZ, neff = ctx.run_host(host, torch.from_numpy(lw).pin_memory())
    ref, _, _ = oracle.eval_batch(cfg, s, n_threads=ORACLE_THREADS)
    rZ, rN = oracle.evidence(ref, lw)
    assert rel_err(ref, out.numpy()) <= TOL
    assert rel_err([rZ], [lnZ]) <= TOL and rel_err([rN], [neff]) <= TOL
    out2, lnZ2, _ = ctx.run_host(host, None, want_lnL=False)
    assert out2 is None and rel_err([oracle.evidence(ref)[0]], [lnZ2]) <= TOL
    assert ctx.launch_count >= 6
    ctx.close()


@pytest.mark.parametrize("n", [200_000, 237_777, 430_001])
def test_run_host_sliced_pipeline_every_sample(gpu_lib, n):
    """From 200,000 samples on (one point, one launch group) ile_run_host cuts the batch into 2-4 slices and uploads slice
    i + 1 / downloads slice i - 1 while slice i computes, with the evidence state carried over the slices on the device.
    EVERY lnL_margT, lnZ and n_eff against the oracle, with and without weights and the lnL download; repeated on one
    context so that a second call finds the staging buffers and events of the first."""
    import torch

    cfg = gi.make_config(1, n=n)
    s = gi.make_samples(cfg["sample_seeds"][0] + 1, n)
    lw = gi.make_log_weights(6, n)
    ref, _, _ = oracle.eval_batch(cfg, s, n_threads=ORACLE_THREADS)
    rZ, rN = oracle.evidence(ref, lw)
    ctx = gpu_lib.Context(cfg)
    host = {k: torch.from_numpy(v).pin_memory() for k, v in s.items()}
    for rep in range(2):
        out, lnZ, neff = ctx.run_host(host, torch.from_numpy(lw).pin_memory())
        assert rel_err(ref, out.numpy()) <= TOL
        assert rel_err([rZ], [lnZ]) <= TOL and rel_err([rN], [neff]) <= TOL
    out2, lnZ2, neff2 = ctx.run_host(host, None, want_lnL=False)
    r0 = oracle.evidence(ref)
    assert out2 is None and rel_err([r0[0]], [lnZ2]) <= TOL and rel_err([r0[1]], [neff2]) <= TOL
    pageable = {k: torch.from_numpy(v.copy()) for k, v in s.items()}          # not pinned: the copies are staged by the driver
    out3, lnZ3, _ = ctx.run_host(pageable, None)
    assert rel_err(ref, out3.numpy()) <= TOL and rel_err([r0[0]], [lnZ3]) <= TOL
    n_bad, _ = ctx.status()
    assert n_bad == 0
    ctx.close()


def test_run_host_all_matches_the_oracle_per_point(gpu_lib):
    """ile_run_host_all: host [P][n] arrays through ONE C-ABI call (H2D, ile_eval_all, ile_evidence per point, D2H);
    n large enough that the streaming path runs, weighted."""
    import torch

    cfg = gi.make_config(4, n=17_000, n_points=3)
    P, n = cfg["n_points"], cfg["n"]
    per = [gi.make_samples(cfg["sample_seeds"][p], n) for p in range(P)]
    lw = gi.make_log_weights(9, P * n).reshape(P, n)
    host = {k: torch.from_numpy(np.ascontiguousarray(np.stack([per[p][k] for p in range(P)]))).pin_memory() for k in per[0]}
    ctx = gpu_lib.Context(cfg)
    out, lnZ, neff = ctx.run_host_all(host, torch.from_numpy(lw).pin_memory())
    for p in range(P):
        ref, _, _ = oracle.eval_batch(cfg, per[p], point=p, n_threads=ORACLE_THREADS)
        assert rel_err(ref, out[p].numpy()) <= TOL
        rZ, rN = oracle.evidence(ref, lw[p])
        assert rel_err([rZ], lnZ[p:p + 1]) <= TOL and rel_err([rN], neff[p:p + 1]) <= TOL
    out2, lnZ2, _ = ctx.run_host_all(host, None, want_lnL=False)
    assert out2 is None
    for p in range(P):
        ref, _, _ = oracle.eval_batch(cfg, per[p], point=p, n_threads=ORACLE_THREADS)
        assert rel_err([oracle.evidence(ref)[0]], lnZ2[p:p + 1]) <= TOL
    ctx.close()


def test_evidence_merge_of_split_batch_equals_whole(gpu_lib):
    """ile_evidence_merge: states of disjoint parts of one sample set merge to the evidence of the whole (what several
    GPUs sharing one intrinsic point exchange); also across segments and with an empty (all -inf) part."""
    import torch

    cfg = gi.make_config(1, n=30_000)
    s = gi.make_samples(cfg["sample_seeds"][0], cfg["n"])
    lw = gi.make_log_weights(3, cfg["n"])
    ctx = gpu_lib.Context(cfg)
    lnL, _ = ctx.eval(to_dev(s))
    lwd = torch.from_numpy(lw).cuda()
    cuts = [0, 7_001, 7_001 + 16_384, 30_000]
    states = []
    for a, b in zip(cuts[:-1], cuts[1:]):
        st = ctx.new_state(1)
        ctx.evidence(lnL[a:b].contiguous(), lwd[a:b].contiguous(), state=st)
        states.append(st)
    dead = ctx.new_state(1)  # a rank whose samples were all out of range
    ctx.evidence(torch.full((5,), float("-inf"), dtype=torch.float64, device="cuda"), None, state=dead)
    states.append(dead)
    merged, lnZ, neff = ctx.evidence_merge(torch.stack(states, 0).contiguous())
    ref, _, _ = oracle.eval_batch(cfg, s, n_threads=ORACLE_THREADS)
    e = ref + lw
    m = e.max()
    rN = float(np.sum(np.exp(e - m)))
    rZ = m + np.log(rN) - np.log(cfg["n"] + 5)  # the dead part still counts its 5 samples (eq. 4: 1/n of ALL draws)
    assert rel_err([rZ], lnZ.cpu().numpy()) <= TOL
    assert rel_err([rN], neff.cpu().numpy()) <= TOL
    assert merged.cpu().numpy()[0, 2] == cfg["n"] + 5
    ctx.close()


def test_streaming_kernel_extreme_amplitudes(gpu_lib):
    """The streaming kernel's fixed-point exp keeps lin / ln 2 - reference in a 2^19-step window around a running reference of a
    whole number of octaves: samples whose linear term runs to 1e3 ... 1e8 (sources at 1 kpc ... 30 Mpc, a = D_ref / D up to 1e5, where
    quad ~ a^2 dwarfs everything) or to 1e-7 (D = 1e9 Mpc) must come out like the oracle's within TOL of |lnL|, next to ordinary ones."""
    cfg = gi.make_config(1, n=20_000)
    s = gi.make_samples(cfg["sample_seeds"][0], cfg["n"])
    m = len(s["dist_mpc"][::7])
    s["dist_mpc"][::7] = np.tile(np.array([1e-3, 5e-2, 1.0, 3.0, 10.0, 30.0, 1e9]), m // 7 + 1)[:m]
    full_compare(gpu_lib, cfg, s, variant=4)


@pytest.mark.parametrize("variant", [1, 2, 4])
def test_every_variant_matches_the_oracle(gpu_lib, variant):
    """ile_set_variant: each evaluation kernel family on the same 20,000 samples of config 1 (indices bit-exact, values
    within TOL); variant 0 (automatic) is what every other test and bench.py run."""
    cfg = gi.make_config(1, n=20_000)
    s = gi.make_samples(cfg["sample_seeds"][0], cfg["n"])
    full_compare(gpu_lib, cfg, s, variant=variant)


def test_many_modes_quadratic_term_as_mma_with_generic_U_V(gpu_lib):
    """21 modes through the streaming variant (n >= 10000): the quadratic term runs as the FP64-MMA contraction of
    ile_quad_mma.cu.  U deliberately not Hermitian, V not symmetric (reading R15); ragged sample count (not a multiple
    of 8) so the last group of 8 is partial."""
    cfg = gi.make_config(2, n=20_003)
    rng = np.random.default_rng(21)
    cfg["U"] = cfg["U"] * (1.0 + 0.3 * rng.standard_normal(cfg["U"].shape)) + 20j * rng.standard_normal(cfg["U"].shape)
    cfg["V"] = cfg["V"] + 10.0 * (rng.standard_normal(cfg["V"].shape) + 1j * rng.standard_normal(cfg["V"].shape))
    s = gi.make_samples(99, cfg["n"])
    full_compare(gpu_lib, cfg, s, variant=4)


def test_many_modes_many_points_in_one_launch(gpu_lib):
    """ile_eval_all with 21 modes and several intrinsic points through the streaming kernel: the multi-point scan and
    prefix kernels together with the FP64-MMA quadratic term (n_per_point a multiple of 8, as that path requires) and,
    with a ragged n_per_point, with the coefficient kernel's own quadratic term."""
    base = gi.make_config(2, n=8)
    c4 = gi.CONFIGS[2]
    P = 3
    pts = [gi.make_point(gi.point_seed(2, 0) + 31 * p, c4["dets"], c4["modes"], c4["n_q"], 12.0 + 5 * p, admix=c4["admix"]) for p in range(P)]
    cfg = dict(base)
    cfg.update(n_points=P, Q=np.ascontiguousarray(np.stack([q[0] for q in pts])), U=np.ascontiguousarray(np.stack([q[1] for q in pts])),
               V=np.ascontiguousarray(np.stack([q[2] for q in pts])))
    for n in (6_000, 5_999):
        per = [gi.make_samples(700 + p, n) for p in range(P)]
        allS = {k: np.ascontiguousarray(np.stack([per[p][k] for p in range(P)])) for k in per[0]}
        ctx = gpu_lib.Context(cfg)
        ctx.set_variant(4)
        lnL, idx = ctx.eval_all(to_dev(allS), want_idx=True)
        lnZ, neff = ctx.evidence(lnL, n_segments=P)
        for p in range(P):
            ref, ref_idx, _ = oracle.eval_batch(cfg, per[p], point=p, n_threads=ORACLE_THREADS)
            assert_indices_equal(cfg, per[p], ref_idx, idx[p].cpu().numpy())
            assert rel_err(ref, lnL[p].cpu().numpy()) <= TOL
            rZ, rN = oracle.evidence(ref)
            assert rel_err([rZ], lnZ[p:p + 1].cpu().numpy()) <= TOL and rel_err([rN], neff[p:p + 1].cpu().numpy()) <= TOL
        ctx.close()


def test_evidence_layouts_on_one_context(gpu_lib):
    """Successive ile_evidence calls with different (n_segments, blocks per segment) layouts on ONE context: the ticket
    words of every segment start at zero whatever the previous layout left behind (two layouts with the same
    n_segments x blocks product used to share stale tickets)."""
    import torch

    cfg = gi.make_config(0)
    ctx = gpu_lib.Context(cfg)
    rng = np.random.default_rng(11)
    for n_seg, per in [(1, 100_000), (1, 8_000), (8, 1_000), (2, 4_000), (4, 2_000), (16, 500), (1, 8_000), (8, 1_000), (3, 70_001)]:
        x = rng.standard_normal(n_seg * per) * 5.0
        lnZ, neff = ctx.evidence(torch.from_numpy(x).cuda(), n_segments=n_seg)
        for g in range(n_seg):
            rZ, rN = oracle.evidence(x[g * per:(g + 1) * per])
            assert rel_err([rZ], lnZ[g:g + 1].cpu().numpy()) <= TOL, (n_seg, per, g)
            assert rel_err([rN], neff[g:g + 1].cpu().numpy()) <= TOL, (n_seg, per, g)
    ctx.close()


# ---------------------------------------------------------------------------------------------- NEXT-4: the paper's own windows
@pytest.mark.parametrize("n", [1_500, 20_000])
@pytest.mark.parametrize("cid", [5, 6, 7, 8])
def test_paper_windows_T03s_at_4096_and_16384_Hz(gpu_lib, cid, n):
    """T = 0.3 s with two detectors and 2 or 4 modes (Tables I/II) at 4096 Hz (N_t = 1229,
    N_Q = 8192) and at the legacy 16384 Hz (N_t = 4915, N_Q = 32768; L121).  1,500 samples take the small-batch kernels,
    20,000 the sorted streaming FP64-MMA path."""
    cfg = gi.make_config(cid, n=n)
    s = gi.make_samples(cfg["sample_seeds"][0], n)
    full_compare(gpu_lib, cfg, s)


def test_paper_window_concentrated_batch_16384_Hz(gpu_lib):
    """Late-in-the-run shape at the legacy rate: samples crowded around one point (a handful of sort cells, long windows)."""
    cfg = gi.make_config(8, n=20_000)
    s = gi.make_concentrated_samples(5150, 20_000)
    full_compare(gpu_lib, cfg, s, log_w=gi.make_log_weights(2, 20_000))


# ---------------------------------------------------------------------------------------------- four detectors on the streaming path
@pytest.mark.parametrize("modes,n", [("l2", 20_000), ("l2", 1_003), ("l4", 10_000)])
def test_four_detector_network_on_the_streaming_kernel(gpu_lib, modes, n):
    """H1, L1, V1 and a fourth site (F is (detectors) x (extrinsic), no limit of three): the K = 4 instantiation of the
    streaming kernel -- sort cells over (d1, d2, d3), three realigned detectors per group -- with 5 and with 21 modes."""
    dets = ("H1", "L1", "V1", "K1")
    ml = gi.modes_up_to(2) if modes == "l2" else gi.modes_up_to(4)
    n_q = 2048 if modes == "l2" else 4096
    Q, U, V, meta = gi.make_point(4004, dets, ml, n_q, 22.0, admix=0.0 if modes == "l2" else 0.1)
    v, ax, ay = gi.detector_arrays(dets)
    cfg = dict(config_id=1, dets=dets, modes=ml, Q=Q[None], U=U[None], V=V[None], l=np.array([x[0] for x in ml], dtype=np.int32),
               m=np.array([x[1] for x in ml], dtype=np.int32), n_points=1, n_det=4, n_modes=len(ml), n_q=n_q, n_t=410, fs_hz=gi.FS_HZ,
               t0_q_s=meta["t0_q_s"], gmst_rad=gi.GMST_RAD, d_ref_mpc=gi.D_REF_MPC, vertex_m=v, arm_x=ax, arm_y=ay, n=n)
    s = gi.make_samples(4005, n)
    full_compare(gpu_lib, cfg, s, variant=4)
    if n == 20_000:
        full_compare(gpu_lib, cfg, s)          # the automatic choice takes the same path


# ---------------------------------------------------------------------------------------------- NEXT-4: interpolated (sub-sample) shifts
@pytest.mark.parametrize("cid,n", [(0, 1_000), (1, 3_001), (5, 400)])
def test_linear_interpolated_shifts_match_the_oracle(gpu_lib, cid, n):
    """shift_mode = 1 (reading R8'): per-detector linear interpolation of Q between samples, against oracle/subsample.py; the floor
    indices bit-exact, lnL_margT within TOL; windows that need the sample beyond the series are out of range."""
    from oracle import subsample as osub

    cfg = gi.make_config(cid, n=n)
    cfg["shift_mode"] = 1
    s = gi.make_samples(cfg["sample_seeds"][0] + 9, n)
    s["t_ref"][3] = 0.9
    ctx, lnL, idx, n_bad = run_gpu(gpu_lib, cfg, s)
    ref, ref_idx, ref_bad = osub.eval_batch_lin(cfg, s)
    assert n_bad == ref_bad >= 1
    assert_indices_equal(cfg, s, ref_idx, idx.cpu().numpy())
    assert rel_err(ref, lnL.cpu().numpy()) <= TOL
    with pytest.raises(gpu_lib.IleError):
        ctx.set_variant(2)
    ctx.close()


@pytest.mark.parametrize("cid,n", [(1, 20_011), (5, 12_000), (6, 3_000), (0, 2_500)])
def test_linear_interpolated_shifts_streaming_kernel(gpu_lib, cid, n):
    """shift_mode = 1 through the streaming FP64-MMA kernel: the packed Q carries every series twice (row i and row i + 1), the
    coefficient records (1 - phi_k) a F_k Y_lm and phi_k a F_k Y_lm, and the contraction is the nearest-sample one over 4M channels.
    Automatic choice from 10,000 samples, variant 4 forced below; floor indices bit-exact, values within TOL, evidence included."""
    from oracle import subsample as osub

    cfg = gi.make_config(cid, n=n)
    cfg["shift_mode"] = 1
    s = gi.make_samples(cfg["sample_seeds"][0] + 11, n)
    s["t_ref"][5] = 0.9
    s["t_ref"][6] = -0.9
    ctx = gpu_lib.Context(cfg)
    if n < 10_000:
        ctx.set_variant(4)
    lnL, idx = ctx.eval(to_dev(s))
    n_bad, _ = ctx.status()
    ref, ref_idx, ref_bad = osub.eval_batch_lin(cfg, s)
    assert n_bad == ref_bad >= 2
    assert_indices_equal(cfg, s, ref_idx, idx.cpu().numpy())
    assert rel_err(ref, lnL.cpu().numpy()) <= TOL
    assert ctx.launch_count >= 5  # index, scan, scatter, coefficient, streaming kernels
    lnZ, neff = ctx.evidence(lnL)
    rZ, rN = oracle.evidence(ref)
    assert rel_err([rZ], lnZ.cpu().numpy()) <= TOL and rel_err([rN], neff.cpu().numpy()) <= TOL
    ctx.close()
