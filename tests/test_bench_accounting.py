"""bench.py's work accounting and counter bookkeeping (host logic, no GPU): the algorithmic work per sample is SURVEY.md 8(d)'s figure, and the
committed ncu counters of the dominant kernel parse into the quantities the roofline block derives from them."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_work_per_sample_is_the_survey_figure():
    # config 1 (3 detectors, 5 modes, 410 bins) = 12,300 + 720 + 8,200 + 400 DFMA-equivalents per sample
    assert bench.dfma_per_sample(3, 5, 410) == 21620.0
    # config 2 (21 modes): 51,660 + 11,088 + 8,200 + 880
    assert bench.dfma_per_sample(3, 21, 410) == 71828.0
    # the kernel's own exp cost replaces the 20 per bin, nothing else
    assert bench.dfma_per_sample(3, 5, 410, 6.0) == 21620.0 - 14.0 * 410
    # interpolated shifts (R8'): the contraction at n_t + 1 rows plus one blend per detector and bin -- NOT twice the contraction,
    # which is how the streaming kernel happens to run it
    assert bench.dfma_per_sample(3, 5, 410, interp=True) == 21620.0 + 2 * 3 * 5 + 2 * 3 * 410


def test_committed_stream_counters_parse_and_are_consistent():
    sc = bench.read_stream_counters()
    assert sc is not None and sc["samples"] == 100000 and sc["n_t"] == 410
    # FP64 instructions per bin outside the contraction, and the pipe's busy fraction, as bench.py derives them
    per_bin = sc["fp64_other_inst"] * 32.0 / (sc["samples"] * sc["n_t"])
    assert 3.0 < per_bin < 20.0
    busy = (16.0 * sc["dmma_inst"] + 2.0 * sc["fp64_other_inst"]) / (sc["cycles_elapsed_max"] * 4.0 * 148.0)
    assert 0.3 < busy < 1.0
    # DMMA count: 18 per warp-step of 16 rows x 8 samples can never be below the unpadded work of the batch
    assert sc["dmma_inst"] * 256 >= sc["samples"] * sc["n_t"] * 3 * 10
