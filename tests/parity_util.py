"""Helpers shared by the -m gpu parity tests: tolerances, comparison rules, oracle drivers."""
import os

import numpy as np

# north_star: lnL and log-evidence within 1e-10 relative (fp64); the gate is |d| <= TOL * max(|ref|, 1)
# (SURVEY.md §7 hard part 4: lnL is a difference of O(rho^2) terms, so near zero the scale is 1).
TOL = 1e-10
ORACLE_THREADS = max(1, min(32, os.cpu_count() or 1))


def rel_err(ref, got):
    ref = np.asarray(ref, dtype=np.float64)
    got = np.asarray(got, dtype=np.float64)
    fin = np.isfinite(ref)
    assert np.array_equal(fin, np.isfinite(got)), "finite / -inf pattern differs"
    assert np.array_equal(ref[~fin], got[~fin]), "non-finite values differ"
    if not fin.any():
        return 0.0
    return float(np.max(np.abs(got[fin] - ref[fin]) / np.maximum(np.abs(ref[fin]), 1.0)))


def assert_indices_equal(cfg, samples, ref_idx, got_idx):
    """Shift indices are integers: bit-exact.  Any flip is reported with its distance from the rounding tie
    (SURVEY.md §7 hard part 3), never hidden."""
    ref_idx = np.asarray(ref_idx)
    got_idx = np.asarray(got_idx)
    assert ref_idx.shape == got_idx.shape
    bad = np.argwhere(ref_idx != got_idx)
    if len(bad):
        lines = []
        for s, k in bad[:10]:
            lines.append(f"sample {s} det {k}: oracle {ref_idx[s, k]} gpu {got_idx[s, k]} t_ref={samples['t_ref'][s]!r}")
        raise AssertionError(f"{len(bad)} shift-index mismatches of {ref_idx.size}:\n" + "\n".join(lines))


def subset(samples, sel):
    return {k: np.ascontiguousarray(v[sel]) for k, v in samples.items()}
