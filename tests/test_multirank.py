"""N > 1 host logic on CPU: two `gloo` ranks (world_size 2, 127.0.0.1).

The hot path has no data-path collective: ranks are independent workers.  What the ranks do share
is (1) bench.py's bookkeeping -- distinct seeded workloads per rank, MAX-over-ranks timing, rank 0 alone printing the
reference arm -- and (2), when several GPUs split ONE intrinsic point, the 24-byte evidence state per segment, gathered
with `gather_evidence_states` and merged on the device by ile_evidence_merge.  Here the gathered states are merged with
plain numpy (test code) and compared with the oracle's evidence of the unsplit sample set.
"""
import json
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys, json
import numpy as np
import torch
import torch.distributed as dist
sys.path.insert(0, os.environ["ILE_ROOT"])
import bench
import ile_inputs as gi
import oracle
import paper_1902_04934_b200 as ile

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)

# (1) bench bookkeeping: distinct workloads, MAX-over-ranks timing
seed = bench.rank_sample_seed(1234, rank)
seeds = [None] * world
dist.all_gather_object(seeds, seed)
assert len(set(seeds)) == world, seeds
mx = bench.max_over_ranks([1.0 + rank, 5.0 - rank], "cpu")
assert mx == [float(world), 5.0], mx

# (2) one intrinsic point split over the ranks: each rank evaluates its slice (oracle stands in for the GPU here),
# reduces it to an evidence state, the states are gathered
cfg = gi.make_config(0, n=600)
s = gi.make_samples(cfg["sample_seeds"][0], cfg["n"])
lw = gi.make_log_weights(11, cfg["n"])
lo, hi = rank * cfg["n"] // world, (rank + 1) * cfg["n"] // world
part = {k: np.ascontiguousarray(v[lo:hi]) for k, v in s.items()}
lnL, _, _ = oracle.eval_batch(cfg, part, n_threads=1)
e = lnL + lw[lo:hi]
m = float(np.max(e))
state = torch.tensor([[m, float(np.sum(np.exp(e - m))), float(hi - lo)]], dtype=torch.float64)
allst = ile.gather_evidence_states(state)
assert tuple(allst.shape) == (world, 1, 3)
if rank == 0:
    print(json.dumps({"states": allst.numpy().tolist()}), flush=True)
dist.barrier()
dist.destroy_process_group()
'''


def _free_port():
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def test_two_gloo_ranks_bookkeeping_and_evidence_state_gather(tmp_path):
    import ile_inputs as gi
    import oracle

    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), ILE_ROOT=ROOT,
                   OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (so, se) in zip(procs, outs):
        assert p.returncode == 0, se[-2000:]
    states = np.array(json.loads(outs[0][0].strip().splitlines()[-1])["states"])  # [world][1][3]
    # merge rule of ile_evidence_merge, restated: common max, rescaled sums, added counts
    M = states[:, 0, 0].max()
    S = float(np.sum(states[:, 0, 1] * np.exp(states[:, 0, 0] - M)))
    cnt = float(states[:, 0, 2].sum())
    cfg = gi.make_config(0, n=600)
    s = gi.make_samples(cfg["sample_seeds"][0], cfg["n"])
    lw = gi.make_log_weights(11, cfg["n"])
    ref, _, _ = oracle.eval_batch(cfg, s, n_threads=2)
    rZ, rN = oracle.evidence(ref, lw)
    assert cnt == cfg["n"]
    assert abs(M + np.log(S) - np.log(cnt) - rZ) <= 1e-10 * max(abs(rZ), 1.0)
    assert abs(S - rN) <= 1e-10 * max(abs(rN), 1.0)


def test_reference_arm_prints_on_rank0_only():
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
           "--config", "0", "--ref-samples-per-step", "200"]
    r1 = subprocess.run(cmd, env=dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1"), capture_output=True, text=True, timeout=300)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = subprocess.run(cmd, env=dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0"), capture_output=True, text=True, timeout=300)
    assert r0.returncode == 0, r0.stderr[-2000:]
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
