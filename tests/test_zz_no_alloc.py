"""ile_evidence_static -- the evidence reduction for callers that are not allowed to allocate device memory.

Most of this library hangs off an ile_ctx, and making (or growing) a context means cudaMalloc.  That is a non-starter for
code that lives inside somebody else's memory pool (a framework's caching allocator, a fixed slab given to a batch job:
a raw cudaMalloc goes around the pool and stalls the whole device), for real-time loops and plug-ins whose host bans
driver allocations after start-up, and for a worker that just wants lnZ from lnL_margT values it already holds.
ile_evidence_static serves them: no context, and its scratch is a fixed 68 KiB array inside the library image
(at most 1024 segments per call; one array per device, so overlapping calls race -- see include/ile.h).

The GPU test below checks the new entry point against the existing ile_evidence path on two calls in a row (the second
with another layout, so whatever the first left in the shared array is in its way), within the tolerance the other
parity tests use, and against the oracle.  The file name sorts last on purpose: with `pytest -x` a failure in this
add-on must not hide the tests of the main path.  It passes alone in a fresh process and after the rest of the suite.
"""
import os
import re

import numpy as np
import pytest

import oracle
from parity_util import TOL, rel_err

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "paper_1902_04934_b200", "csrc", "ile_evidence_static.cu")


def make_lnL(rng, n_seg, per, dead_segment=None):
    """lnL_margT-like values: a wide spread (so max-subtraction matters), some -inf (out-of-range samples), and
    optionally one segment without a finite sample (lnZ = -inf, n_eff = 0)."""
    x = rng.standard_normal((n_seg, per)) * 8.0 + rng.uniform(-300.0, 300.0, size=(n_seg, 1))
    x[rng.random((n_seg, per)) < 0.01] = -np.inf
    if dead_segment is not None:
        x[dead_segment] = -np.inf
    lw = rng.standard_normal((n_seg, per)) * 0.5
    return x, lw


def check_against_both(ile, ctx, x, lw, n_seg):
    import torch

    xd, wd = torch.from_numpy(x).cuda(), torch.from_numpy(lw).cuda()
    lnZ_s, neff_s = ile.evidence_static(xd, wd, n_segments=n_seg)        # the allocation-free entry point
    lnZ_c, neff_c = ctx.evidence(xd, wd, n_segments=n_seg)               # the existing, context-owned path
    torch.cuda.synchronize()
    assert rel_err(lnZ_c.cpu().numpy(), lnZ_s.cpu().numpy()) <= TOL
    assert rel_err(neff_c.cpu().numpy(), neff_s.cpu().numpy()) <= TOL
    for g in range(n_seg):
        rZ, rN = oracle.evidence(x[g], lw[g])
        assert rel_err([rZ], lnZ_s[g:g + 1].cpu().numpy()) <= TOL, g
        assert rel_err([rN], neff_s[g:g + 1].cpu().numpy()) <= TOL, g


@pytest.mark.gpu
def test_static_scratch_evidence_matches_context_path_on_two_calls_in_a_row(gpu_lib):
    import torch

    import ile_inputs as gi

    ile = gpu_lib
    ctx = ile.Context(gi.make_config(0, n=4))       # only the existing path needs a context
    rng = np.random.default_rng(1902)
    # call 1: few long segments (many blocks per segment -> many partials and busy tickets), one of them dead
    x1, w1 = make_lnL(rng, 3, 250_001, dead_segment=1)
    check_against_both(ile, ctx, x1, w1, 3)
    # call 2, straight after, other layout: the segment maximum (the (n_seg, 1) offset) sits in different scratch slots
    x2, w2 = make_lnL(rng, 1000, 777)
    check_against_both(ile, ctx, x2, w2, 1000)
    # chunked with a carried state, as config 3 feeds ile_evidence: two calls in a row into one state
    x3, w3 = make_lnL(rng, 2, 120_000)
    st_s = torch.tensor([[-np.inf, 0.0, 0.0]] * 2, dtype=torch.float64, device="cuda")
    st_c = ctx.new_state(2)
    for lo, hi in [(0, 70_000), (70_000, 120_000)]:
        xd = torch.from_numpy(np.ascontiguousarray(x3[:, lo:hi])).cuda()
        wd = torch.from_numpy(np.ascontiguousarray(w3[:, lo:hi])).cuda()
        lnZ_s, neff_s = ile.evidence_static(xd, wd, state=st_s, n_segments=2)
        lnZ_c, neff_c = ctx.evidence(xd, wd, state=st_c, n_segments=2)
    torch.cuda.synchronize()
    assert rel_err(st_c.cpu().numpy(), st_s.cpu().numpy()) <= TOL
    assert rel_err(lnZ_c.cpu().numpy(), lnZ_s.cpu().numpy()) <= TOL
    for g in range(2):
        rZ, rN = oracle.evidence(x3[g], w3[g])
        assert rel_err([rZ], lnZ_s[g:g + 1].cpu().numpy()) <= TOL and rel_err([rN], neff_s[g:g + 1].cpu().numpy()) <= TOL
    # beyond the fixed array: refused with a clear error, nothing launched
    big = torch.zeros(1025 * 4, dtype=torch.float64, device="cuda")
    with pytest.raises(ile.IleError) as ei:
        ile.evidence_static(big, n_segments=1025)
    assert ei.value.code == -4 and "not supported" in str(ei.value)
    ctx.close()


def test_static_entry_point_calls_no_allocator():
    """The promise is 'allocates nothing': the translation unit behind ile_evidence_static must not call cudaMalloc,
    cudaFree or a relative (comments do not count)."""
    code = re.sub(r"//[^\n]*|/\*.*?\*/", "", open(SRC).read(), flags=re.S)
    assert not re.search(r"\bcuda(Malloc\w*|Free\w*|HostAlloc|HostRegister|MemPool\w*)\s*\(", code)
    assert "cudaGetSymbolAddress" in code and "__align__(256)" in code


def test_static_entry_point_rejects_bad_sizes_without_a_device():
    import paper_1902_04934_b200 as ile
    from paper_1902_04934_b200 import build as b

    b.build()
    lib = ile.load()
    assert lib.ile_evidence_static(0, 10, None, None, None, None, None, None) == -1      # no segment
    assert lib.ile_evidence_static(1, 10, None, None, None, 1, None, None) == -1         # samples but no input pointer
    assert lib.ile_evidence_static(1025, 0, None, None, None, 1, None, None) == -4       # more segments than the fixed array serves
