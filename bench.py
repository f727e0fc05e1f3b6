#!/usr/bin/env python
"""bench.py -- the driver's benchmark contract for the ILE hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config C] [--variant V]

A "step" is one pass of the whole hot path (ile_eval + ile_evidence) over one batch of
synthetic extrinsic samples.  Default workload: BASELINE.json configs[1] -- 3 detectors (H1, L1, V1), the five l = 2
modes, Q of 2048 complex128 samples at 4096 Hz per (detector, mode), 100,000 prior-drawn extrinsic samples, 410 time
bins.  Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.

N > 1 (torchrun): the paper's own parallelism is independent workers, one GPU each, no communication
(PAPER.md L134-L141), so each rank evaluates its own seeded intrinsic point and batch; there is no data-path
collective; `value` = samples of all ranks / max-over-ranks device time ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "time-marginalized ILE lnL samples/sec (3 det, l<=2)"
UNIT = "samples/s"


# ------------------------------------------------------------------------------------------------------------------
# algorithmic work per sample in DFMA-equivalents
# ------------------------------------------------------------------------------------------------------------------
EXP_DFMA = 20.0      # "Total DFMA-equivalents with exp ~ 20" (subtract, range reduction, polynomial, accumulate)
NOMINAL_FP64_TFLOPS = 37.2  # 148 SMs x 64 FP64 lanes x 2 flop x 1.965 GHz


def dfma_per_sample(K: int, M: int, n_t: int, exp_cost: float = EXP_DFMA, interp: bool = False) -> float:
    """config 1 -> 12,300 + 720 + 8,200 + 400 = 21,620 DFMA-equivalents per sample.
    `exp_cost` = FP64-pipe instructions per time bin of step 6: 20 is the survey's convention; the kernel's own count
    (from the committed ncu SASS mix) gives the "measured exp" accounting of SURVEY.md §8(d)."""
    # step 5: Re sum conj(A) Q, 2 DFMA per complex element.  Interpolated shifts (R8'): the contraction at n_t + 1 rows, then one
    # (1 - phi) T_j + phi T_{j+1} per detector and bin -- that the streaming kernel runs it as twice the channels is its own choice
    linear = 2.0 * K * M * (n_t + 1) + 2.0 * K * n_t if interp else 2.0 * K * M * n_t
    quad = 2.0 * K * (4.0 * M * M + 4.0 * M)        # step 4: Y^dagger U Y and Y^T V Y per detector
    lse = n_t * exp_cost                            # step 6
    geom = 250.0 + 30.0 * M                         # steps 1-3: five sincos, F_k, dt_k, Y_lm, K*M coefficient products
    return linear + quad + lse + geom


def rank_sample_seed(base_seed: int, rank: int) -> int:
    """Seed of rank `rank`'s batch of extrinsic samples: every rank is an independent worker."""
    return int(base_seed) + 7919 * int(rank)


def rank_point_seed(base_seed: int, rank: int) -> int:
    """Seed of rank `rank`'s intrinsic point (rank 0 keeps the configuration's own point)."""
    return int(base_seed) + 7919 * int(rank)


def max_over_ranks(values, device):
    """Timing rule of the bench contract: every device-timed figure is the MAX over ranks."""
    import torch
    import torch.distributed as dist

    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.0005):
        super().__init__(daemon=True)
        self.index, self.period = index, period_s
        self.samples, self.reasons, self.stop_flag = [], set(), False
        self.max_mhz = None
        self.edge = {}  # one reading taken by the launching thread right before and right after the event loop
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _read(self):
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown", nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown", nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
        r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        return mhz, [nm for bit, nm in names.items() if r & bit]

    def read_edge(self, which: str):
        """One reading by the calling thread (`which` = "before" / "after" the event loop): a timed region of a few
        milliseconds may end before the polling thread has run once."""
        if self.nv is None:
            return
        try:
            mhz, rs = self._read()
            self.edge[which] = mhz
            self.reasons.update(rs)
        except Exception:
            pass

    def run(self):
        if self.nv is None:
            return
        while not self.stop_flag:
            try:
                mhz, rs = self._read()
                self.samples.append(mhz)
                self.reasons.update(rs)
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self):
        allv = sorted(self.samples + list(self.edge.values()))
        out = {"sm_mhz": allv[len(allv) // 2] if allv else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
               "n_samples": len(self.samples), "poll_ms": self.period * 1e3}
        out.update({"sm_mhz_" + k: v for k, v in self.edge.items()})
        return out


def read_stream_counters():
    """Counters of the dominant kernel (the streaming FP64-MMA kernel, config 1, one launch = 100,000 samples) from the
    committed `ncu --set full` capture: profiles/stream_counters.csv, last row (its .md names the command).  Returns a
    dict or None.  Columns: dram_bytes_read, dram_bytes_write, dmma_inst, fp64_other_inst (DFMA + DADD + DMUL warp
    instructions), cycles_elapsed_max, pipe_fp64_pct (ncu sm__inst_executed_pipe_fp64 % of peak), samples, n_t."""
    p = os.path.join(ROOT, "profiles", "stream_counters.csv")
    try:
        import csv

        row = [r for r in csv.DictReader(open(p))][-1]
        return {k: (v if k in ("capture", "kernel", "source", "commit") else float(v)) for k, v in row.items()}
    except Exception:
        return None


def counters_describe_run(sc_, cfg, n, P, variant, shift_mode) -> bool:
    """The committed ncu row is ONE launch of the streaming kernel on config 1: its traffic, pipe fraction and per-bin exp
    cost are attached to a run only if that run launches the same kernel on the same sizes."""
    return bool(sc_) and cfg["config_id"] == 1 and P == 1 and n == int(sc_["samples"]) and cfg["n_t"] == int(sc_["n_t"]) \
        and variant in (0, 4) and not shift_mode


# ------------------------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle, as it stands, on the host cores
# ------------------------------------------------------------------------------------------------------------------
def run_reference(args, rank: int):
    if rank != 0:
        return
    import ile_inputs as gi
    import oracle

    cores = os.cpu_count() or 1
    cfg = gi.make_config(args.config, n_points=1)
    n_step = min(cfg["n"], args.ref_samples_per_step)
    s = gi.make_samples(cfg["sample_seeds"][0], n_step)
    for _ in range(args.warmup):
        out, _, _ = oracle.eval_batch(cfg, s, n_threads=cores)
        oracle.evidence(out)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        out, _, _ = oracle.eval_batch(cfg, s, n_threads=cores)
        oracle.evidence(out)
    dt = time.perf_counter() - t0
    val = n_step * args.steps / dt
    sample = f"{n_step} of the {cfg['n']} samples of the workload per step, {args.steps} steps, OpenMP over samples"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, n_step, args, extra={"note": "CPU oracle (oracle/ile_oracle.c) on host cores"}),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_precompute(args, rank: int):
    """SURVEY.md §8(f) NEXT-1, single GPU: ile_precompute over --points intrinsic points of --config's shape per step.
    HBM-bound by construction (every spectrum is read once, every Q written once); roofline against MEASURED_PEAKS.json."""
    if rank != 0:
        return None
    import numpy as np
    import torch

    import ile_inputs as gi
    import paper_1902_04934_b200 as ile

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    ile.load()
    c = gi.CONFIGS[args.config]
    P = max(1, args.points)
    snr = c["snr"] if not isinstance(c["snr"], tuple) else 20.0
    _, _, _, meta = gi.make_point(gi.point_seed(args.config, 0), c["dets"], c["modes"], c["n_q"], snr, admix=c["admix"], spectra=True)
    rng = np.random.Generator(np.random.PCG64(4934))
    x = torch.from_numpy(np.ascontiguousarray(np.broadcast_to(meta["x"], (P,) + meta["x"].shape))).cuda()
    d = torch.from_numpy(np.ascontiguousarray(np.broadcast_to(meta["d"], (P,) + meta["d"].shape))).cuda()
    x = x * torch.from_numpy(1.0 + 0.01 * rng.standard_normal(P)).cuda().view(P, 1, 1, 1)  # P different points of one shape
    K, M, N = x.shape[1:]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(max(args.warmup, 3)):
        ile.precompute(x, d, meta["fs_hz"], meta["t0_q_s"])
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(0)
    sampler.start()
    sampler.read_edge("before")
    for i in range(args.steps):
        flush.fill_(i & 1)
        ev[i][0].record()
        ile.precompute(x, d, meta["fs_hz"], meta["t0_q_s"])
        ev[i][1].record()
    torch.cuda.synchronize()
    sampler.read_edge("after")
    sampler.stop_flag = True
    ms = sum(a.elapsed_time(b) for a, b in ev) / args.steps
    nbytes = 16 * P * K * (2 * M * N + N + 2 * M * M)  # x in, d in, Q out, U and V out (x counted once)
    peak = None
    try:
        peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
        src = "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        peak, src = 6550.0, "B200_PROFILING.md fallback"
    ach = nbytes / (ms * 1e-3) * 1e-9
    line = {"metric": "overlap pre-computation (eq. 8: Q, U, V) intrinsic points/sec", "value": P / (ms * 1e-3), "unit": "points/s",
            "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "c128", "data": "synthetic",
            "config": {"workload": f"ile_precompute: {P} intrinsic point(s) of BASELINE.json configs[{args.config}]'s shape "
                                   f"({K} detectors, {M} modes, {N}-point spectra)", "l2": "flushed between timed steps (256 MiB write)"},
            "roofline": {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None,
                         "kernel": "ile_overlap_q_radix8_kernel + ile_overlap_uv_bulk_kernel", "peak_source": src, "algorithmic_bytes": nbytes},
            "gpu_launches": 2 * args.steps, "clocks": sampler.summary()}
    return line


def run_integrate(args, rank: int):
    """SURVEY.md §8(f) NEXT-2, single GPU: the whole adaptive Monte Carlo integral of one intrinsic point through
    ile_integrate -- Philox draws, sampling-prior refits, ile_eval and the evidence all on the device; per chunk two
    doubles cross the bus.  Workload: BASELINE.json configs[--config], chunks of --n samples (default 10,000: the paper's
    block size, L97 / n_chunk L119), --chunks chunks per step (default 200: N_it = 2e6, L119), adapting in RA, dec and
    distance after each of the first --adapt-chunks chunks (default 10; L125: "only adapt until a marginalized likelihood evaluation
    returns significant lnL_marg"), no early stop (n_eff threshold = inf) so that every step does the same work.  With frozen
    densities the remaining chunks are drawn and evaluated about 2^20 samples at a time; results are those of the chunk-by-chunk loop."""
    if rank != 0:
        return None
    import numpy as np
    import torch

    import ile_inputs as gi
    import paper_1902_04934_b200 as ile

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    ile.load()
    cfg = gi.make_config(args.config, n_points=1)
    n_chunk = args.n if args.n is not None else 10_000
    chunks = args.chunks
    scfg = dict(seed=4934, n_bins=100, adapt=(True, True, True), floor_frac=0.1, temper=0.5, dist_min_mpc=1.0, dist_max_mpc=1000.0,
                t_ref_lo_s=-0.05, t_ref_hi_s=0.05)
    ctx = ile.Context(cfg)
    if args.variant:
        ctx.set_variant(args.variant)
    smp = ile.Sampler(scfg)
    for _ in range(max(args.warmup, 3)):
        ile.integrate(ctx, smp, n_chunk, chunks, min(chunks, args.adapt_chunks), float("inf"))
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    l0, s0 = ctx.launch_count, smp.launch_count
    sampler.start()
    sampler.read_edge("before")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    e0.record()
    for _ in range(args.steps):
        r = ile.integrate(ctx, smp, n_chunk, chunks, min(chunks, args.adapt_chunks), float("inf"))
    e1.record()
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    sampler.read_edge("after")
    sampler.stop_flag = True
    ms = max(e0.elapsed_time(e1), wall * 1e3) / args.steps      # the call synchronises: device and wall time agree
    launches = (ctx.launch_count - l0) + (smp.launch_count - s0)
    K, M, n_t = cfg["n_det"], cfg["n_modes"], cfg["n_t"]
    w = dfma_per_sample(K, M, n_t)
    peak = max(ile.measure_fp64_peak(1 << 15)[0], ile.measure_dmma_peak(1 << 12)[0])
    val = n_chunk * chunks / (ms * 1e-3)
    ach = 2.0 * w * val * 1e-12
    line = {"metric": "adaptive Monte Carlo integral (draw + lnL_margT + evidence + refit on the device) samples/sec", "value": val,
            "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"ile_integrate on BASELINE.json configs[{args.config}] ({K} detectors, {M} modes, {n_t} bins): {chunks} chunks "
                                   f"of {n_chunk} Philox-drawn samples per step, refit of the (RA, dec, distance) sampling prior after each of the first "
                                   f"{min(chunks, args.adapt_chunks)} chunks",
                       "n_chunk": n_chunk, "chunks_per_step": chunks, "adapt_chunks": min(chunks, args.adapt_chunks), "variant": args.variant},
            "roofline": {"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak, "traffic": None,
                         "kernel": "whole loop (draw, index/sort, coefficients, contraction + marginalisation, evidence, refit)",
                         "dfma_equiv_per_sample": w},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 16 * chunks, "ms_per_step": ms,
                    "api": "ile_integrate (samples are generated on the device: no per-block H2D)"},
            "gpu_launches": int(launches), "clocks": sampler.summary(), "lnZ": r["lnZ"], "n_eff": r["n_eff"],
            "us_per_chunk": ms * 1e3 / chunks}
    if not args.no_cpu_baseline:
        import oracle  # cpu_baseline leg
        from oracle import sampler as osm

        cores = os.cpu_count() or 1
        nchk = 3
        t0 = time.perf_counter()
        osm.integrate(scfg, lambda sd: oracle.eval_batch(cfg, sd, n_threads=cores)[0], n_chunk, nchk, min(nchk, args.adapt_chunks), float("inf"))
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": n_chunk * nchk / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"the first {nchk} chunks of the same run: oracle/sampler.py (numpy) around oracle.eval_batch (OpenMP)"}
    ctx.close()
    smp.close()
    return line


# ------------------------------------------------------------------------------------------------------------------
# sweep: every other workload of BASELINE.json / SURVEY.md 8(f), short runs attached to the headline's JSON line
# ------------------------------------------------------------------------------------------------------------------
SWEEP_HOTPATH = [  # (config, samples per point, points): configs 0, 2, 3 at every batch size (1e7 as ONE call), 4, the paper's windows 5-8
    (0, None, 1), (2, 1_000_000, 1), (3, 1_000, 1), (3, 10_000, 1), (3, 100_000, 1), (3, 1_000_000, 1), (3, 10_000_000, 1),
    (4, 100_000, 256), (5, 100_000, 1), (6, 100_000, 1), (7, 100_000, 1), (8, 100_000, 1)]
ORACLE_BUDGET = 3.0e10  # detector x mode x bin x sample products the oracle is asked for per entry (about 10 s on 16 cores)


def sweep_hotpath_entry(cid, n, P, steps, peak_tflops, exp_meas, with_oracle, local_rank=0):
    """One hot-path workload, timed like the headline: warm-up 3, `steps` steps with an L2 flush in front of each, CUDA events
    on the launching stream around ile_eval + ile_evidence, NVML polled at 0.5 ms and read before / after the loop."""
    import numpy as np
    import torch

    import ile_inputs as gi
    import paper_1902_04934_b200 as ile

    cfg = gi.make_config(cid, n_points=P)
    n = cfg["n"] if n is None else n
    if P == 1:
        s_np = gi.make_samples(cfg["sample_seeds"][0], n)
    else:
        parts = [gi.make_samples(cfg["sample_seeds"][p], n) for p in range(P)]
        s_np = {k: np.ascontiguousarray(np.concatenate([q[k] for q in parts])) for k in parts[0]}
        del parts
    ctx = ile.Context(cfg)
    dev = ile.samples_to_device(s_np)
    lnL = torch.empty(P * n, dtype=torch.float64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def do_eval():
        if P == 1:
            ctx.eval(dev, want_idx=False, out=lnL)       # ONE call whatever n (above 2^20 samples the library cuts it into launch groups)
        else:
            ctx.eval_all(dev, want_idx=False, out=lnL.view(P, n))

    for _ in range(3):
        flush.fill_(1)
        do_eval()
        ctx.evidence(lnL, n_segments=P)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    sampler = ClockSampler(local_rank)
    l0 = ctx.launch_count
    sampler.start()
    sampler.read_edge("before")
    for i in range(steps):
        flush.fill_(i & 1)
        ev[i][0].record(stream)
        do_eval()
        ev[i][1].record(stream)
        lnZ, neff = ctx.evidence(lnL, n_segments=P)
        ev[i][2].record(stream)
    torch.cuda.synchronize()
    sampler.read_edge("after")
    sampler.stop_flag = True
    launches = ctx.launch_count - l0
    step_ms = sum(a.elapsed_time(c) for a, _, c in ev) / steps
    eval_ms = sum(a.elapsed_time(b) for a, b, _ in ev) / steps
    n_bad, _ = ctx.status()
    K, M, n_t = cfg["n_det"], cfg["n_modes"], cfg["n_t"]
    w = dfma_per_sample(K, M, n_t)
    e = {"stage": "hotpath", "config": cid, "samples_per_point": n, "points": P, "steps": steps,
         "workload": workload_config(cfg, n, argparse.Namespace(gpus=1))["workload"],
         "value": P * n / (step_ms * 1e-3), "unit": UNIT, "ms_per_step": step_ms, "ile_eval_ms": eval_ms,
         "frac": 2.0 * w * P * n / (eval_ms * 1e-3) * 1e-12 / peak_tflops,
         "frac_model_measured_exp": (2.0 * dfma_per_sample(K, M, n_t, exp_meas) * P * n / (eval_ms * 1e-3) * 1e-12 / peak_tflops) if exp_meas else None,
         "gpu_launches": int(launches), "n_out_of_range": int(n_bad), "clocks": sampler.summary(),
         "lnZ": float(lnZ[0].item()), "n_eff": float(neff[0].item()), "lnZ_oracle": None}
    if with_oracle and float(K) * M * n_t * n <= ORACLE_BUDGET:  # intrinsic point 0, every sample of it
        import oracle  # cpu_baseline leg

        pb = dict(cfg)
        if P > 1:
            pb["Q"], pb["U"], pb["V"], pb["n_points"] = cfg["Q"][:1], cfg["U"][:1], cfg["V"][:1], 1
        ref, _, _ = oracle.eval_batch(pb, {k: v[:n] for k, v in s_np.items()}, n_threads=os.cpu_count() or 1)
        rZ, rN = oracle.evidence(ref)
        e["lnZ_oracle"], e["n_eff_oracle"] = rZ, rN
        e["lnZ_rel_err"] = abs(e["lnZ"] - rZ) / max(abs(rZ), 1.0)
    ctx.close()
    del dev, lnL, flush
    torch.cuda.empty_cache()
    return e


def run_sweep(args, peak_tflops, exp_meas):
    """Short runs of every workload the headline does not cover.  Entries are independent: one that fails is reported as
    {"error": ...} and the sweep goes on."""
    out = []
    steps = max(3, min(args.steps, 10))
    with_oracle = not args.no_cpu_baseline
    for cid, n, P in SWEEP_HOTPATH:
        try:
            k = 3 if (n or 0) * P >= 5_000_000 else steps
            out.append(sweep_hotpath_entry(cid, n, P, k, peak_tflops, exp_meas, with_oracle))
        except Exception as ex:  # noqa: BLE001
            out.append({"stage": "hotpath", "config": cid, "samples_per_point": n, "points": P, "error": repr(ex)})
    keep = ("metric", "value", "unit", "ms_per_step", "steps", "clocks", "gpu_launches", "lnZ", "n_eff", "us_per_chunk")
    for stage, kw in [("precompute", dict(config=4, points=256)), ("precompute", dict(config=2, points=16)),
                      ("integrate", dict(config=1, n=10_000, chunks=200, adapt_chunks=10)),      # densities frozen after 10 chunks (L125)
                      ("integrate", dict(config=1, n=10_000, chunks=200, adapt_chunks=200))]:    # refit after every chunk
        a = argparse.Namespace(**vars(args))
        for k_, v_ in kw.items():
            setattr(a, k_, v_)
        a.steps, a.warmup, a.variant, a.no_cpu_baseline = (steps if stage == "precompute" else 3), 3, 0, True
        try:
            line = run_precompute(a, 0) if stage == "precompute" else run_integrate(a, 0)
            e = {"stage": stage, **kw, **{k_: line[k_] for k_ in keep if k_ in line}, "workload": line["config"]["workload"],
                 "frac": line["roofline"]["frac"], "bound": line["roofline"]["bound"]}
        except Exception as ex:  # noqa: BLE001
            e = {"stage": stage, **kw, "error": repr(ex)}
        out.append(e)
    return out



def workload_config(cfg, n, args, extra=None):
    src = f"BASELINE.json configs[{cfg['config_id']}]" if cfg["config_id"] <= 4 else f"paper window config {cfg['config_id']} (NEXT-4: T = 0.3 s, PAPER.md L86, L121)"
    c = {"workload": f"{src}: {cfg['n_det']} detectors ({','.join(cfg['dets'])}), "
                     f"{cfg['n_modes']} modes (l<= {int(max(cfg['l']))}), Q {cfg['n_q']} complex128 @ {int(cfg['fs_hz'])} Hz, "
                     f"{cfg['n_points']} intrinsic point(s) x {n} extrinsic samples/step/GPU, {cfg['n_t']} time bins",
         "n_det": cfg["n_det"], "n_modes": cfg["n_modes"], "n_q": cfg["n_q"], "n_t": cfg["n_t"],
         "samples_per_step_per_gpu": n * cfg["n_points"], "points_per_gpu": cfg["n_points"],
         "parallelism": f"independent intrinsic points, {cfg['n_points']} per GPU x{args.gpus}", "l2": "flushed between timed steps (256 MiB write)"}
    if extra:
        c.update(extra)
    return c


# ------------------------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--n", type=int, default=None, help="samples per step per GPU (default: the config's)")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--points", type=int, default=1, help="intrinsic points evaluated concurrently per step (config 4: 256), ile_eval_all")
    ap.add_argument("--samples", default="prior", choices=["prior", "concentrated"])
    ap.add_argument("--shift-mode", type=int, default=0, choices=[0, 1],
                    help="1: linear interpolation of Q between samples (NEXT-4, reading R8'); hot-path stage only, no cpu_baseline leg")
    ap.add_argument("--ref-samples-per-step", type=int, default=100_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--stage", default="hotpath", choices=["hotpath", "precompute", "integrate"],
                    help="precompute: time ile_precompute (eq. 8: Q, U, V of --points intrinsic points); integrate: time ile_integrate "
                         "(the adaptive Monte Carlo loop with on-device sampling) instead of the hot path")
    ap.add_argument("--chunks", type=int, default=200, help="--stage integrate: chunks per step")
    ap.add_argument("--no-sweep", action="store_true", help="skip the sweep over the other workloads (the default N = 1 run attaches it as \"sweep\")")
    ap.add_argument("--adapt-chunks", type=int, default=10,
                    help="--stage integrate: chunks after which the sampling prior is frozen (PAPER.md L125: adapt only early in the run)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        if args.steps > 20:
            args.steps = 20
        run_reference(args, rank)
        return
    if args.stage == "precompute":
        line = run_precompute(args, rank)
        if line:
            print(json.dumps(line), flush=True)
        return
    if args.stage == "integrate":
        if args.steps > 20:
            args.steps = 20
        line = run_integrate(args, rank)
        if line:
            print(json.dumps(line), flush=True)
        return

    import numpy as np
    import torch
    import torch.distributed as dist

    import ile_inputs as gi
    import paper_1902_04934_b200 as ile

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    ile.load()
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    # ---- workload: one intrinsic point and one batch per rank (independent workers)
    P = max(1, args.points)
    base = gi.make_config(args.config, n_points=P)
    if args.shift_mode:
        base["shift_mode"] = 1
        args.no_cpu_baseline = True
    n = args.n if args.n is not None else base["n"]
    if rank > 0:  # a different seeded intrinsic point per rank, same recipe
        c = gi.CONFIGS[args.config]
        snr = c["snr"] if not isinstance(c["snr"], tuple) else 20.0
        Q, U, V, meta = gi.make_point(rank_point_seed(gi.point_seed(args.config, 0), rank), c["dets"], c["modes"], c["n_q"], snr, admix=c["admix"])
        base["Q"], base["U"], base["V"] = Q[None], U[None], V[None]
    seed = rank_sample_seed(base["sample_seeds"][0], rank)
    mk = gi.make_samples if args.samples == "prior" else gi.make_concentrated_samples
    if P == 1:
        s_np = mk(seed, n)
    else:  # [P][n]: every point its own seeded batch
        parts = [mk(rank_sample_seed(base["sample_seeds"][p], rank), n) for p in range(P)]
        s_np = {k: np.ascontiguousarray(np.concatenate([q[k] for q in parts])) for k in parts[0]}
    ctx = ile.Context(base)
    if args.variant:
        ctx.set_variant(args.variant)
    dev = ile.samples_to_device(s_np)
    host = {k: torch.from_numpy(v).pin_memory() for k, v in s_np.items()}
    host_out = torch.empty(n, dtype=torch.float64).pin_memory()
    lnL = torch.empty(P * n, dtype=torch.float64, device="cuda")
    host_out = torch.empty(P * n, dtype=torch.float64).pin_memory() if P > 1 else host_out
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def do_eval():
        if P == 1:
            ctx.eval(dev, want_idx=False, out=lnL)
        else:
            ctx.eval_all(dev, want_idx=False, out=lnL.view(P, n))

    def do_e2e():
        if P == 1:
            return ctx.run_host(host, None, out_host=host_out)
        return ctx.run_host_all(host, None, out_host=host_out)  # [P][n] arrays, one C-ABI call

    def step():
        do_eval()
        return ctx.evidence(lnL, n_segments=P)

    for _ in range(args.warmup):
        flush.fill_(1)
        step()
        do_e2e()
    torch.cuda.synchronize()

    peak_dfma, _ = ile.measure_fp64_peak(1 << 15)
    peak_dmma, _ = ile.measure_dmma_peak(1 << 12)
    peak_tflops = max(peak_dfma, peak_dmma)

    # ---- timed region: exactly K steps, device-timed with CUDA events on the launching stream
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    launches0 = ctx.launch_count
    sampler.start()
    sampler.read_edge("before")
    wall0 = time.perf_counter()
    for i in range(args.steps):
        flush.fill_(i & 1)                      # L2 flush, outside the event pair
        ev[i][0].record(stream)
        do_eval()
        ev[i][1].record(stream)
        lnZ, neff = ctx.evidence(lnL, n_segments=P)
        ev[i][2].record(stream)
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    sampler.read_edge("after")
    sampler.stop_flag = True
    launches = ctx.launch_count - launches0
    if world > 1:
        dist.barrier()
    step_ms = sum(a.elapsed_time(c) for a, _, c in ev)
    eval_ms = sum(a.elapsed_time(b) for a, b, _ in ev)
    n_bad, _ = ctx.status()

    # ---- end to end through the C ABI with HOST buffers (ile_run_host): H2D + kernels + D2H inside the timed region
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(args.steps):
        _, lnZ_h, neff_h = do_e2e()
    e1.record(stream)
    torch.cuda.synchronize()
    e2e_ms = e0.elapsed_time(e1)
    e2e_wall = time.perf_counter() - t0
    e2e_ms = max(e2e_ms, e2e_wall * 1e3)        # the call synchronises: wall clock and device time agree; take the larger

    step_ms, eval_ms, e2e_ms = max_over_ranks([step_ms, eval_ms, e2e_ms], "cuda")

    if rank == 0:
        K, M, n_t = base["n_det"], base["n_modes"], base["n_t"]
        w = dfma_per_sample(K, M, n_t, interp=bool(args.shift_mode))
        value = world * P * n * args.steps / (step_ms * 1e-3)
        eval_avg_ms = eval_ms / args.steps
        achieved = 2.0 * w * P * n / (eval_avg_ms * 1e-3) * 1e-12
        # the same with the exp cost the kernel really pays (FP64-pipe instructions per bin outside the contraction, from the
        # committed ncu SASS mix) and the FP64 pipe's busy fraction in that capture (DMMA 16 cycles, DFMA/DADD/DMUL 2 cycles
        # per warp instruction and SMSP): SURVEY.md §8(d) "model fraction" and "pipe fraction"
        sc_ = read_stream_counters()
        if not counters_describe_run(sc_, base, n, P, args.variant, args.shift_mode):
            sc_ = None  # another config, variant or shift mode: the capture says nothing about this run
        exp_meas = frac_meas = frac_pipe = None
        if sc_:
            sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
            exp_meas = sc_["fp64_other_inst"] * 32.0 / (sc_["samples"] * sc_["n_t"])
            frac_meas = 2.0 * dfma_per_sample(K, M, n_t, exp_meas, bool(args.shift_mode)) * P * n / (eval_avg_ms * 1e-3) * 1e-12 / peak_tflops
            frac_pipe = (16.0 * sc_["dmma_inst"] + 2.0 * sc_["fp64_other_inst"]) / (sc_["cycles_elapsed_max"] * 4.0 * sms)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": step_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": workload_config(base, n, args, extra={"variant": args.variant, "samples": args.samples, "shift_mode": args.shift_mode}),
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                         "frac_model_measured_exp": frac_meas,
                         "fractions": "two accountings of the SAME measured time, to be read side by side: `frac` credits 20 DFMA-equivalents "
                                      "per exp (SURVEY.md 8(d)'s table, comparable across rounds); `frac_model_measured_exp` credits what the "
                                      "shipped table exp costs (8(d)'s 'model fraction'), the stricter of the two",
                         "traffic": int(sc_["dram_bytes_read"] + sc_["dram_bytes_write"]) if sc_ else None,
                         "kernel": "ile_eval (steps 1-6)", "kernel_ms": eval_avg_ms, "dfma_equiv_per_sample": w,
                         "peak_dfma": peak_dfma, "peak_dmma": peak_dmma, "peak_nominal": NOMINAL_FP64_TFLOPS,
                         "frac_vs_nominal": achieved / NOMINAL_FP64_TFLOPS,
                         "exp_fp64_inst_per_bin_measured": exp_meas,
                         "frac_pipe": frac_pipe, "pipe_fp64_pct_ncu": sc_["pipe_fp64_pct"] if sc_ else None,
                         "counters_capture": sc_["capture"] if sc_ else None, "counters_commit": sc_.get("commit") if sc_ else None,
                         "peak_source": "max(ile_measure_fp64_peak: register-resident DFMA chains, ile_measure_dmma_peak: DMMA.8x8x4 chains), "
                         "both measured in this run; frac counts exp at 20 DFMA-equivalents per bin (SURVEY.md 8(d)), "
                         "frac_model_measured_exp at the kernel's own FP64 instruction count per bin, frac_pipe is the FP64 pipe's "
                         "busy fraction in the committed ncu capture"},
            "e2e": {"value": world * P * n * args.steps / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 7 * 8 * P * n,
                    "d2h_bytes_per_step": 8 * P * n + 16 * P, "ms_per_step": e2e_ms / args.steps,
                    "api": "ile_run_host (pinned host buffers)" if P == 1 else "ile_run_host_all (pinned host buffers)"},
            "gpu_launches": int(launches), "clocks": sampler.summary(), "wall_ms_per_step": wall / args.steps * 1e3,
            "lnZ": float(lnZ[0].item()), "n_eff": float(neff[0].item()), "n_out_of_range": int(n_bad),
        }
        if not args.no_cpu_baseline:
            import oracle  # cpu_baseline leg: the one place bench.py's product arm may execute oracle/

            cores = os.cpu_count() or 1
            n_cpu = min(n, 100_000)  # of intrinsic point 0
            sub = {k: v[:n_cpu] for k, v in s_np.items()}
            if P > 1:  # the oracle takes one intrinsic point at a time: time point 0
                pb = dict(base)
                pb["Q"], pb["U"], pb["V"], pb["n_points"] = base["Q"][:1], base["U"][:1], base["V"][:1], 1
            else:
                pb = base
            oracle.eval_batch(pb, {k: v[:2000] for k, v in s_np.items()}, n_threads=cores)  # page in / spin up
            passes, t0 = 0, time.perf_counter()
            while passes < 4 or time.perf_counter() - t0 < 10.0:  # a bounded sample: about 10 s of CPU work
                ref, _, _ = oracle.eval_batch(pb, sub, n_threads=cores)
                rZ, _ = oracle.evidence(ref)
                passes += 1
            dt = time.perf_counter() - t0
            n_one = min(n_cpu, 20_000)  # single thread: a smaller bounded sample of the same batch
            sub1 = {k: v[:n_one] for k, v in s_np.items()}
            t1 = time.perf_counter()
            ref1, _, _ = oracle.eval_batch(pb, sub1, n_threads=1)
            oracle.evidence(ref1)
            dt1 = time.perf_counter() - t1
            line["cpu_baseline"] = {"value": n_cpu * passes / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{passes} passes over the first {n_cpu} samples of the same batch (eval + evidence), OpenMP over samples",
                                    "value_1thread": n_one / dt1, "sample_1thread": f"one pass over the first {n_one} samples, 1 thread",
                                    "lnZ_oracle": rZ if n_cpu == n else None}
        default_run = (world == 1 and args.config == 1 and P == 1 and args.n is None and not args.variant and not args.shift_mode
                       and args.samples == "prior")
        if default_run and not args.no_sweep:
            ctx.close()
            del dev, lnL, flush
            torch.cuda.empty_cache()
            line["sweep_note"] = ("the other workloads, each timed like the headline (L2 flush, CUDA events, NVML at 0.5 ms) over fewer steps; "
                                  "frac counts exp at 20 DFMA-equivalents, frac_model_measured_exp at the per-bin cost of the committed capture "
                                  "of the same streaming kernel; lnZ_oracle is the CPU oracle on intrinsic point 0 where it fits in about 10 s")
            line["sweep"] = run_sweep(args, peak_tflops, exp_meas)
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
