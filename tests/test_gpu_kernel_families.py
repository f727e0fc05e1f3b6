"""Every kernel family of the library on reduced sizes, in one process, each result checked against the oracle: configs 0 and 1
through variants 1, 2 and 4 (with one out-of-range window), a multi-point launch, segmented / chunked / merged evidence,
ile_run_host / ile_run_host_all, the 21-mode path with the FP64-MMA quadratic term, and ile_precompute.

Collected by pytest (-m gpu).  The same file is the workload for compute-sanitizer (SURVEY.md 5 "race detection / sanitizers"),
sized for its 10-100x slowdown, where that tool is available (it is closed on this pool: profiles/r02_sanitizer.md):

    for t in memcheck racecheck initcheck synccheck; do compute-sanitizer --tool $t python tests/test_gpu_kernel_families.py; done
"""
import os
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import ile_inputs as gi  # noqa: E402
import oracle  # noqa: E402
import paper_1902_04934_b200 as ile  # noqa: E402


def dev(s):
    return {k: torch.from_numpy(v).cuda() for k, v in s.items()}


def check(ref, got, what):
    ref, got = np.asarray(ref), np.asarray(got)
    fin = np.isfinite(ref)
    assert np.array_equal(fin, np.isfinite(got)), what
    e = float(np.max(np.abs(got[fin] - ref[fin]) / np.maximum(np.abs(ref[fin]), 1.0))) if fin.any() else 0.0
    assert e <= 1e-10, (what, e)
    print(f"  ok {what}: max rel err {e:.2e}", flush=True)


def main():
    ile.load()
    torch.cuda.set_device(0)
    thr = min(16, os.cpu_count() or 1)
    # configs 0 and 1, every variant
    for cid, n in ((0, 1_000), (1, 20_000)):
        cfg = gi.make_config(cid, n=n)
        s = gi.make_samples(cfg["sample_seeds"][0], n)
        s["t_ref"][5] = 0.3  # one out-of-range window (reading R9)
        ref, ref_idx, _ = oracle.eval_batch(cfg, s, n_threads=thr)
        for v in (1, 2, 4):
            ctx = ile.Context(cfg)
            ctx.set_variant(v)
            lnL, idx = ctx.eval(dev(s))
            assert np.array_equal(ref_idx, idx.cpu().numpy())
            check(ref, lnL.cpu().numpy(), f"config {cid} variant {v}")
            st = ctx.new_state()
            for lo in range(0, n, 7_000):
                lnZ, neff = ctx.evidence(lnL[lo:lo + 7_000].contiguous(), state=st)
            check([oracle.evidence(ref)[0]], lnZ.cpu().numpy(), f"config {cid} variant {v} chunked evidence")
            ctx.status(reset=True)
            ctx.close()
    # many points in one launch + segmented evidence + merge + host entries
    cfg = gi.make_config(4, n=6_000, n_points=3)
    P, n = 3, 6_000
    per = [gi.make_samples(cfg["sample_seeds"][p], n) for p in range(P)]
    allS = {k: np.ascontiguousarray(np.stack([per[p][k] for p in range(P)])) for k in per[0]}
    ctx = ile.Context(cfg)
    ctx.set_variant(4)
    lnL, _ = ctx.eval_all(dev(allS))
    lnZ, neff = ctx.evidence(lnL, n_segments=P)
    refs = [oracle.eval_batch(cfg, per[p], point=p, n_threads=thr)[0] for p in range(P)]
    check(np.stack(refs), lnL.cpu().numpy(), "eval_all, 3 points")
    check([oracle.evidence(r)[0] for r in refs], lnZ.cpu().numpy(), "segmented evidence")
    sts = []
    for lo, hi in ((0, 2_500), (2_500, 6_000)):
        st = ctx.new_state(1)
        ctx.evidence(lnL[0, lo:hi].contiguous(), state=st)
        sts.append(st)
    _, mz, _ = ctx.evidence_merge(torch.stack(sts, 0).contiguous())
    check([oracle.evidence(refs[0])[0]], mz.cpu().numpy(), "evidence merge")
    host = {k: torch.from_numpy(v).pin_memory() for k, v in allS.items()}
    out, hz, _ = ctx.run_host_all(host, None)
    check(np.stack(refs), out.numpy(), "run_host_all")
    out1, z1, _ = ctx.run_host({k: torch.from_numpy(per[1][k]).pin_memory() for k in per[1]}, None, point=1)
    check(refs[1], out1.numpy(), "run_host")
    ctx.close()
    # 21 modes: FP64-MMA quadratic term, chain ping-pong fragments
    cfg = gi.make_config(2, n=4_000)
    s = gi.make_samples(3, 4_000)
    ctx = ile.Context(cfg)
    ctx.set_variant(4)
    lnL, _ = ctx.eval(dev(s))
    check(oracle.eval_batch(cfg, s, n_threads=thr)[0], lnL.cpu().numpy(), "config 2 variant 4")
    ctx.close()
    # overlap pre-computation
    from oracle import precompute as opre

    c = gi.CONFIGS[1]
    _, _, _, meta = gi.make_point(77, c["dets"], c["modes"], c["n_q"], 20.0, spectra=True)
    x, d = torch.from_numpy(meta["x"][None]).cuda(), torch.from_numpy(meta["d"][None]).cuda()
    Q, U, V = ile.precompute(x, d, meta["fs_hz"], meta["t0_q_s"])
    Qr, Ur, Vr = opre.overlaps(meta["x"], meta["d"], meta["fs_hz"], meta["t0_q_s"])
    for nm, a, b in (("Q", Qr, Q), ("U", Ur, U), ("V", Vr, V)):
        g = b.cpu().numpy()[0]
        assert np.max(np.abs(g - a)) <= 1e-10 * np.max(np.abs(a)), nm
    print("  ok ile_precompute", flush=True)
    torch.cuda.synchronize()
    print("kernel-family workload finished", flush=True)


@pytest.mark.gpu
def test_every_kernel_family_on_reduced_sizes(gpu_lib):
    main()


if __name__ == "__main__":
    main()
