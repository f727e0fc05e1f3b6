"""GPU-vs-oracle parity of ile_precompute (eq. 8a-c; oracle/precompute.py) through the C ABI, and the chain
ile_precompute -> ile_create -> ile_eval against the CPU oracle fed with the oracle's own Q, U, V.

Tolerance: 1e-10 (north_star), relative to the largest magnitude of the SERIES (Q) or of the matrix (U, V): an FFT's rounding
error is a fraction of the spectrum's norm, not of each output, so bins far below the peak cannot be held to 1e-10 of their
own size by any implementation (the oracle's library FFT included)."""
import numpy as np
import pytest

import ile_inputs as gi
import oracle
from oracle import precompute as pc
from parity_util import ORACLE_THREADS, TOL, assert_indices_equal, rel_err

pytestmark = pytest.mark.gpu


def spectra_of_config(cid, n_points=1):
    c = gi.CONFIGS[cid]
    xs, ds, meta = [], [], None
    for p in range(n_points):
        snr = c["snr"] if not isinstance(c["snr"], tuple) else 20.0
        _, _, _, meta = gi.make_point(gi.point_seed(cid, p), c["dets"], c["modes"], c["n_q"], snr, admix=c["admix"], spectra=True)
        xs.append(meta["x"]), ds.append(meta["d"])
    return np.stack(xs), np.stack(ds), meta


def gpu_overlaps(ile, x, d, fs, t0):
    import torch

    Q, U, V = ile.precompute(torch.from_numpy(np.ascontiguousarray(x)).cuda(), torch.from_numpy(np.ascontiguousarray(d)).cuda(), fs, t0)
    torch.cuda.synchronize()
    return Q.cpu().numpy(), U.cpu().numpy(), V.cpu().numpy()


def check(got, ref, axes):
    scale = np.max(np.abs(ref), axis=axes, keepdims=True)
    scale = np.where(scale > 0, scale, 1.0)
    err = float(np.max(np.abs(got - ref) / scale))
    assert err <= TOL, err
    return err


@pytest.mark.parametrize("cid,n_points", [(0, 1), (1, 1), (2, 1), (4, 3)])
def test_precompute_matches_oracle_on_config_shapes(gpu_lib, cid, n_points):
    x, d, meta = spectra_of_config(cid, n_points)
    Q, U, V = gpu_overlaps(gpu_lib, x, d, meta["fs_hz"], meta["t0_q_s"])
    for p in range(n_points):
        rq, ru, rv = pc.overlaps(x[p], d[p], meta["fs_hz"], meta["t0_q_s"])
        check(Q[p], rq, axes=-1)
        check(U[p], ru, axes=(-1, -2))
        check(V[p], rv, axes=(-1, -2))


@pytest.mark.parametrize("n_q", [2, 4, 64, 256, 512, 1024, 4096, 8192, 16384, 32768, 65536])
def test_precompute_edge_sizes_and_fractional_start_time(gpu_lib, n_q):
    r = np.random.default_rng(n_q)
    K, M = 1, (1 if n_q == 2 else 3)
    x = r.standard_normal((1, K, M, n_q)) + 1j * r.standard_normal((1, K, M, n_q))
    d = r.standard_normal((1, K, n_q)) + 1j * r.standard_normal((1, K, n_q))
    fs, t0 = 4096.0, 3.25 / 4096.0
    Q, U, V = gpu_overlaps(gpu_lib, x, d, fs, t0)
    ref = pc.overlaps(x[0], d[0], fs, t0) if n_q > 64 else pc.overlaps_direct(x[0], d[0], fs, t0)
    check(Q[0], ref[0], axes=-1)
    check(U[0], ref[1], axes=(-1, -2))
    check(V[0], ref[2], axes=(-1, -2))


def test_precompute_rejects_sizes_it_does_not_support(gpu_lib):
    import torch

    x = torch.zeros((1, 1, 1, 48), dtype=torch.complex128, device="cuda")
    d = torch.zeros((1, 1, 48), dtype=torch.complex128, device="cuda")
    with pytest.raises(gpu_lib.IleError) as ei:
        gpu_lib.precompute(x, d, 4096.0, 0.0)
    assert ei.value.code == -4


def test_chain_precompute_create_eval_matches_oracle_chain(gpu_lib):
    """Q, U, V made on the GPU feed ile_create / ile_eval; the oracle chain uses the oracle's Q, U, V.  Window indices
    bit-exact, lnL_margT within TOL."""
    import torch

    x, d, meta = spectra_of_config(1)
    cfg = gi.make_config(1, n=20_000)
    s = gi.make_samples(cfg["sample_seeds"][0], cfg["n"])
    Q, U, V = gpu_overlaps(gpu_lib, x, d, meta["fs_hz"], meta["t0_q_s"])
    rq, ru, rv = pc.overlaps(x[0], d[0], meta["fs_hz"], meta["t0_q_s"])
    gcfg, ocfg = dict(cfg), dict(cfg)
    gcfg["Q"], gcfg["U"], gcfg["V"] = Q, U, V
    ocfg["Q"], ocfg["U"], ocfg["V"] = rq[None], ru[None], rv[None]
    ctx = gpu_lib.Context(gcfg)
    lnL, idx = ctx.eval({k: torch.from_numpy(v).cuda() for k, v in s.items()})
    ref, ref_idx, _ = oracle.eval_batch(ocfg, s, n_threads=ORACLE_THREADS)
    assert_indices_equal(cfg, s, ref_idx, idx.cpu().numpy())
    assert rel_err(ref, lnL.cpu().numpy()) <= TOL
    ctx.close()


@pytest.mark.parametrize("n_q,M,P", [(512, 2, 1), (2048, 5, 3), (4096, 21, 1), (8192, 4, 2), (1024, 7, 1), (16384, 2, 2), (32768, 4, 1)])
def test_precompute_psd_matches_oracle(gpu_lib, n_q, M, P):
    """ile_precompute_psd: un-whitened spectra, 1 / S weighting and band mask of eq. 2 on the device, against oracle.overlaps_psd;
    few modes (register-resident pair sums) and many modes (tiled pair sums)."""
    import torch

    r = np.random.default_rng(n_q + M)
    K, fs, t0 = 2, 4096.0, -n_q / 8192.0 + 0.4 / 4096.0
    h = r.standard_normal((P, K, M, n_q)) + 1j * r.standard_normal((P, K, M, n_q))
    d = r.standard_normal((P, K, n_q)) + 1j * r.standard_normal((P, K, n_q))
    f = np.abs(pc.signed_index(n_q) * fs / n_q)
    S = np.stack([np.stack([(0.5 + p + k) * (1.0 + (f / 300.0) ** 2 + (40.0 / np.maximum(f, 1.0)) ** 4) for k in range(K)]) for p in range(P)])
    fmin, fmax, scale = 20.0, 1024.0, 2.0 * fs / n_q
    Q, U, V = gpu_lib.precompute_psd(torch.from_numpy(h).cuda(), torch.from_numpy(d).cuda(), torch.from_numpy(S).cuda(), fs, t0, fmin, fmax, scale)
    Q, U, V = Q.cpu().numpy(), U.cpu().numpy(), V.cpu().numpy()
    for p in range(P):
        rq, ru, rv = pc.overlaps_psd(h[p], d[p], S[p], fs, t0, fmin, fmax, scale)
        check(Q[p], rq, axes=-1)
        check(U[p], ru, axes=(-1, -2))
        check(V[p], rv, axes=(-1, -2))
    with pytest.raises(gpu_lib.IleError):
        gpu_lib.precompute_psd(torch.from_numpy(h).cuda(), torch.from_numpy(d).cuda(), torch.from_numpy(S).cuda(), fs, t0, 50.0, 20.0, scale)


def test_precompute_calls_on_two_streams_share_the_library_tables_safely(gpu_lib):
    """The twiddle / phase table and the two-level scratch are library-owned, one set per device.  Calls with DIFFERENT
    (n_q, start time) issued back to back on two non-blocking streams, with no event between them, must each see their
    own table: every call waits on the device for the previous call (include/ile.h, ile_precompute).  Repeated so that a
    missing order would show as a wrong Q in at least one round."""
    import torch

    r = np.random.default_rng(77)
    cases = []
    for n_q, t0 in [(2048, 3.25 / 4096.0), (16384, -1.5 / 4096.0), (1024, 0.0), (2048, 7.75 / 4096.0)]:
        x = r.standard_normal((4, 2, 3, n_q)) + 1j * r.standard_normal((4, 2, 3, n_q))
        d = r.standard_normal((4, 2, n_q)) + 1j * r.standard_normal((4, 2, n_q))
        cases.append((torch.from_numpy(x).cuda(), torch.from_numpy(d).cuda(), t0, [pc.overlaps(x[p], d[p], 4096.0, t0) for p in range(4)]))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    for rnd in range(3):
        outs = []
        for i, (xd, dd, t0, _) in enumerate(cases):
            st = streams[(i + rnd) & 1]
            with torch.cuda.stream(st):
                outs.append(gpu_lib.precompute(xd, dd, 4096.0, t0, stream=st))
        torch.cuda.synchronize()
        for (Q, U, V), (_, _, _, ref) in zip(outs, cases):
            for p in range(4):
                check(Q[p].cpu().numpy(), ref[p][0], axes=-1)
                check(U[p].cpu().numpy(), ref[p][1], axes=(-1, -2))
                check(V[p].cpu().numpy(), ref[p][2], axes=(-1, -2))
