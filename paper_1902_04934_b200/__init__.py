"""paper_1902_04934_b200 -- thin Python binding of libile_b200.so (include/ile.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels behind the C ABI.  PyTorch is used
for device memory (`tensor.data_ptr()`), streams and nothing else.  There is no CPU fallback: `load()` raises if the
shared library is missing, and every call raises `IleError` on a non-zero return code.  Nothing here imports
`oracle/`.

    ctx = Context(cfg_dict)            # ile_create  (cfg_dict as produced by ile_inputs.make_config)
    lnL, idx = ctx.eval(samples)       # ile_eval    (dict of seven CUDA float64 tensors)
    lnZ, neff = ctx.evidence(lnL)      # ile_evidence
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libile_b200.so")
_lib = None

SAMPLE_FIELDS = ("ra", "dec", "t_ref", "phi_ref", "psi", "incl", "dist_mpc")
EXPORTS = ("ile_create", "ile_eval", "ile_eval_all", "ile_evidence", "ile_evidence_reset", "ile_evidence_merge", "ile_evidence_static", "ile_precompute", "ile_precompute_psd", "ile_run_host", "ile_run_host_all", "ile_status",
           "ile_set_variant", "ile_launch_count", "ile_measure_fp64_peak", "ile_measure_dmma_peak", "ile_destroy", "ile_strerror",
           "ile_sampler_create", "ile_sampler_destroy", "ile_sampler_reset", "ile_sampler_set_tables", "ile_sampler_get_tables",
           "ile_sampler_uniforms", "ile_sampler_draw", "ile_sampler_refit", "ile_sampler_launch_count", "ile_integrate",
           "ile_resample", "ile_harvest")


class IleError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = load().ile_strerror(code).decode() if _lib is not None else str(code)
        super().__init__(f"{where} failed with code {code}: {msg}")


class _Detector(ctypes.Structure):
    _fields_ = [("vertex_m", ctypes.c_double * 3), ("arm_x", ctypes.c_double * 3), ("arm_y", ctypes.c_double * 3)]


class _SamplerConfig(ctypes.Structure):
    _fields_ = [("seed", ctypes.c_uint64), ("n_bins", ctypes.c_int32), ("adapt_ra", ctypes.c_int32), ("adapt_dec", ctypes.c_int32),
                ("adapt_dist", ctypes.c_int32), ("floor_frac", ctypes.c_double), ("temper", ctypes.c_double),
                ("dist_min_mpc", ctypes.c_double), ("dist_max_mpc", ctypes.c_double), ("t_ref_lo_s", ctypes.c_double),
                ("t_ref_hi_s", ctypes.c_double)]


class _Config(ctypes.Structure):
    _fields_ = [("n_points", ctypes.c_int32), ("n_det", ctypes.c_int32), ("n_modes", ctypes.c_int32),
                ("l", ctypes.POINTER(ctypes.c_int32)), ("m", ctypes.POINTER(ctypes.c_int32)),
                ("n_q", ctypes.c_int32), ("n_t", ctypes.c_int32), ("fs_hz", ctypes.c_double), ("t0_q_s", ctypes.c_double),
                ("gmst_rad", ctypes.c_double), ("d_ref_mpc", ctypes.c_double), ("det", ctypes.POINTER(_Detector)),
                ("shift_mode", ctypes.c_int32)]


def load():
    """dlopen libile_b200.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_1902_04934_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    L = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, dp = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.POINTER(ctypes.c_double)
    L.ile_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(_Config), vp, vp, vp]
    L.ile_eval.argtypes = [vp, i32, i64] + [vp] * 7 + [vp, vp, vp]
    L.ile_eval_all.argtypes = [vp, i64] + [vp] * 7 + [vp, vp, vp]
    L.ile_evidence.argtypes = [vp, i32, i64, vp, vp, vp, vp, vp, vp]
    L.ile_evidence_reset.argtypes = [vp, i32, vp, vp]
    L.ile_evidence_static.argtypes = [i32, i64, vp, vp, vp, vp, vp, vp]
    L.ile_evidence_merge.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp]
    L.ile_precompute.argtypes = [i32, i32, i32, i32, ctypes.c_double, ctypes.c_double, vp, vp, vp, vp, vp, vp]
    L.ile_precompute_psd.argtypes = [i32, i32, i32, i32, ctypes.c_double, ctypes.c_double, vp, vp, vp, ctypes.c_double, ctypes.c_double,
                                     ctypes.c_double, vp, vp, vp, vp]
    L.ile_run_host.argtypes = [vp, i32, i64] + [vp] * 7 + [vp, vp, dp, dp, vp]
    L.ile_run_host_all.argtypes = [vp, i64] + [vp] * 7 + [vp, vp, dp, dp, vp]
    L.ile_status.argtypes = [vp, ctypes.POINTER(i64), ctypes.c_int, vp]
    L.ile_set_variant.argtypes = [vp, i32]
    L.ile_launch_count.argtypes = [vp]
    L.ile_launch_count.restype = i64
    L.ile_measure_fp64_peak.argtypes = [i32, dp, dp]
    L.ile_measure_dmma_peak.argtypes = [i32, dp, dp]
    L.ile_destroy.argtypes = [vp]
    L.ile_destroy.restype = None
    L.ile_strerror.argtypes = [ctypes.c_int]
    L.ile_strerror.restype = ctypes.c_char_p
    L.ile_sampler_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(_SamplerConfig)]
    L.ile_sampler_destroy.argtypes = [vp]
    L.ile_sampler_destroy.restype = None
    L.ile_sampler_reset.argtypes = [vp, vp]
    L.ile_sampler_set_tables.argtypes = [vp, vp, vp]
    L.ile_sampler_get_tables.argtypes = [vp, vp, vp, vp]
    L.ile_sampler_uniforms.argtypes = [vp, i64, i64, vp, vp]
    L.ile_sampler_draw.argtypes = [vp, i64, i64] + [vp] * 7 + [vp, vp, vp]
    L.ile_sampler_refit.argtypes = [vp, i64, vp, vp, vp, vp]
    L.ile_sampler_launch_count.argtypes = [vp]
    L.ile_sampler_launch_count.restype = i64
    L.ile_integrate.argtypes = [vp, vp, i32, i64, i32, i32, ctypes.c_double, dp, dp, ctypes.POINTER(i64), vp, vp]
    L.ile_resample.argtypes = [vp, i64, vp, vp, i64, ctypes.c_double, vp, vp]
    L.ile_harvest.argtypes = [vp, i32, i64] + [vp] * 7 + [i64, vp, vp, vp, vp, vp, vp]
    for name in EXPORTS:
        if name not in ("ile_launch_count", "ile_destroy", "ile_strerror", "ile_sampler_destroy", "ile_sampler_launch_count"):
            getattr(L, name).restype = ctypes.c_int
        assert getattr(L, name).argtypes is not None, name
    _lib = L
    return L


def _check(code: int, where: str):
    if code != 0:
        raise IleError(code, where)


def _stream_ptr(stream=None):
    import torch

    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _ptr(t):
    return ctypes.c_void_p(0 if t is None else t.data_ptr())


def measure_fp64_peak(iters: int = 1 << 16):
    """(TFLOP/s, ms) of register-resident DFMA chains on the current device (ile_measure_fp64_peak)."""
    tf, ms = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(load().ile_measure_fp64_peak(int(iters), ctypes.byref(tf), ctypes.byref(ms)), "ile_measure_fp64_peak")
    return tf.value, ms.value


def measure_dmma_peak(iters: int = 1 << 13):
    """(TFLOP/s, ms) of independent DMMA.8x8x4 chains on the current device (ile_measure_dmma_peak)."""
    tf, ms = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(load().ile_measure_dmma_peak(int(iters), ctypes.byref(tf), ctypes.byref(ms)), "ile_measure_dmma_peak")
    return tf.value, ms.value


class Context:
    """Owns one ile_ctx.  `cfg` holds numpy arrays Q [P][K][M][n_q], U, V [P][K][M][M], l, m, vertex_m, arm_x, arm_y
    and the scalars of ile_config (see include/ile.h)."""

    def __init__(self, cfg):
        import numpy as np

        L = load()
        K, M = int(cfg["n_det"]), int(cfg["n_modes"])
        self.n_points, self.n_det, self.n_modes = int(cfg["n_points"]), K, M
        self.n_q, self.n_t = int(cfg["n_q"]), int(cfg["n_t"])
        l = np.ascontiguousarray(cfg["l"], dtype=np.int32)
        m = np.ascontiguousarray(cfg["m"], dtype=np.int32)
        det = (_Detector * K)()
        for k in range(K):
            for e in range(3):
                det[k].vertex_m[e] = float(cfg["vertex_m"][k][e])
                det[k].arm_x[e] = float(cfg["arm_x"][k][e])
                det[k].arm_y[e] = float(cfg["arm_y"][k][e])
        c = _Config(self.n_points, K, M, l.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                    m.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), self.n_q, self.n_t, float(cfg["fs_hz"]),
                    float(cfg["t0_q_s"]), float(cfg["gmst_rad"]), float(cfg["d_ref_mpc"]), det, int(cfg.get("shift_mode", 0)))
        Q = np.ascontiguousarray(cfg["Q"], dtype=np.complex128)
        U = np.ascontiguousarray(cfg["U"], dtype=np.complex128)
        V = np.ascontiguousarray(cfg["V"], dtype=np.complex128)
        assert Q.shape == (self.n_points, K, M, self.n_q) and U.shape == V.shape == (self.n_points, K, M, M)
        self._h = ctypes.c_void_p()
        _check(L.ile_create(ctypes.byref(self._h), ctypes.byref(c), ctypes.c_void_p(Q.ctypes.data),
                            ctypes.c_void_p(U.ctypes.data), ctypes.c_void_p(V.ctypes.data)), "ile_create")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load().ile_destroy(self._h)
            self._h = ctypes.c_void_p()

    __del__ = close

    def set_variant(self, variant: int):
        _check(load().ile_set_variant(self._h, int(variant)), "ile_set_variant")

    @property
    def launch_count(self) -> int:
        return int(load().ile_launch_count(self._h))

    def _sample_ptrs(self, samples, n_expected=None):
        import torch

        ts = [samples[f] for f in SAMPLE_FIELDS]
        n = ts[0].numel()
        for t in ts:
            assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n
        assert n_expected is None or n == n_expected
        return [_ptr(t) for t in ts], n

    def eval(self, samples, point: int = 0, want_idx: bool = True, out=None, stream=None):
        """ile_eval: dict of seven CUDA float64 tensors [n] -> (lnL_margT [n], shift_idx [n][K] or None)."""
        import torch

        ptrs, n = self._sample_ptrs(samples)
        dev = samples["ra"].device
        lnL = out if out is not None else torch.empty(n, dtype=torch.float64, device=dev)
        idx = torch.empty((n, self.n_det), dtype=torch.int32, device=dev) if want_idx else None
        _check(load().ile_eval(self._h, int(point), n, *ptrs, _ptr(lnL), _ptr(idx), _stream_ptr(stream)), "ile_eval")
        return lnL, idx

    def eval_all(self, samples, want_idx: bool = False, out=None, stream=None):
        """ile_eval_all: tensors are [P][n_per_point] -> (lnL_margT [P][n], shift_idx [P][n][K] or None)."""
        import torch

        ptrs, n = self._sample_ptrs(samples)
        assert n % self.n_points == 0
        npp = n // self.n_points
        dev = samples["ra"].device
        lnL = out if out is not None else torch.empty((self.n_points, npp), dtype=torch.float64, device=dev)
        idx = torch.empty((self.n_points, npp, self.n_det), dtype=torch.int32, device=dev) if want_idx else None
        _check(load().ile_eval_all(self._h, npp, *ptrs, _ptr(lnL), _ptr(idx), _stream_ptr(stream)), "ile_eval_all")
        return lnL, idx

    def evidence(self, lnL, log_w=None, state=None, n_segments: int = 1, stream=None):
        """ile_evidence: lnL [n_segments][n_per_segment] (any shape with that many elements) -> (lnZ, n_eff) CUDA
        tensors [n_segments].  `state` ([n_segments][3], from new_state()) carries (max, sum, count) across chunks."""
        import torch

        assert lnL.is_cuda and lnL.dtype == torch.float64 and lnL.is_contiguous()
        n = lnL.numel()
        assert n % n_segments == 0
        if log_w is not None:
            assert log_w.is_cuda and log_w.dtype == torch.float64 and log_w.is_contiguous() and log_w.numel() == n
        lnZ = torch.empty(n_segments, dtype=torch.float64, device=lnL.device)
        neff = torch.empty(n_segments, dtype=torch.float64, device=lnL.device)
        _check(load().ile_evidence(self._h, int(n_segments), n // n_segments, _ptr(lnL), _ptr(log_w), _ptr(state),
                                   _ptr(lnZ), _ptr(neff), _stream_ptr(stream)), "ile_evidence")
        return lnZ, neff

    def evidence_merge(self, states, stream=None):
        """ile_evidence_merge: states [n_states][n_segments][3] (CUDA float64, e.g. gathered from all ranks by
        gather_evidence_states) -> (merged state [n_segments][3], lnZ [n_segments], n_eff [n_segments])."""
        import torch

        assert states.is_cuda and states.dtype == torch.float64 and states.is_contiguous() and states.dim() == 3 and states.shape[2] == 3
        n_states, n_seg = int(states.shape[0]), int(states.shape[1])
        out = torch.empty((n_seg, 3), dtype=torch.float64, device=states.device)
        lnZ = torch.empty(n_seg, dtype=torch.float64, device=states.device)
        neff = torch.empty(n_seg, dtype=torch.float64, device=states.device)
        _check(load().ile_evidence_merge(self._h, n_seg, n_states, _ptr(states), _ptr(out), _ptr(lnZ), _ptr(neff),
                                         _stream_ptr(stream)), "ile_evidence_merge")
        return out, lnZ, neff

    def new_state(self, n_segments: int = 1, device="cuda", stream=None):
        import torch

        st = torch.empty((n_segments, 3), dtype=torch.float64, device=device)
        _check(load().ile_evidence_reset(self._h, int(n_segments), _ptr(st), _stream_ptr(stream)), "ile_evidence_reset")
        return st

    def run_host(self, samples_host, log_w_host=None, point: int = 0, want_lnL: bool = True, out_host=None, stream=None):
        """ile_run_host: HOST tensors/arrays in (pinned torch CPU tensors recommended), host results out:
        (lnL_margT host tensor or None, lnZ float, n_eff float)."""
        import torch

        ts = [samples_host[f] for f in SAMPLE_FIELDS]
        n = ts[0].numel()
        for t in ts:
            assert (not t.is_cuda) and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n
        out = None
        if want_lnL:
            out = out_host if out_host is not None else torch.empty(n, dtype=torch.float64).pin_memory()
        lnZ, neff = ctypes.c_double(0.0), ctypes.c_double(0.0)
        _check(load().ile_run_host(self._h, int(point), n, *[_ptr(t) for t in ts], _ptr(log_w_host), _ptr(out),
                                   ctypes.byref(lnZ), ctypes.byref(neff), _stream_ptr(stream)), "ile_run_host")
        return out, lnZ.value, neff.value

    def run_host_all(self, samples_host, log_w_host=None, want_lnL: bool = True, out_host=None, stream=None):
        """ile_run_host_all: HOST tensors [P][n_per_point] in, host results out: (lnL_margT host tensor [P][n] or None,
        lnZ numpy [P], n_eff numpy [P])."""
        import numpy as np
        import torch

        ts = [samples_host[f] for f in SAMPLE_FIELDS]
        tot = ts[0].numel()
        assert tot % self.n_points == 0
        n = tot // self.n_points
        for t in ts:
            assert (not t.is_cuda) and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == tot
        out = None
        if want_lnL:
            out = out_host if out_host is not None else torch.empty((self.n_points, n), dtype=torch.float64).pin_memory()
        lnZ, neff = np.zeros(self.n_points), np.zeros(self.n_points)
        dp = ctypes.POINTER(ctypes.c_double)
        _check(load().ile_run_host_all(self._h, n, *[_ptr(t) for t in ts], _ptr(log_w_host), _ptr(out), lnZ.ctypes.data_as(dp),
                                       neff.ctypes.data_as(dp), _stream_ptr(stream)), "ile_run_host_all")
        return out, lnZ, neff

    def resample(self, lnL, log_w, n_out: int, v0: float, stream=None):
        """ile_resample: -> CUDA int64 [n_out] sample ids (systematic resampling by w L_margT)."""
        import torch

        assert lnL.is_cuda and lnL.dtype == torch.float64 and lnL.is_contiguous()
        assert log_w is None or (log_w.is_cuda and log_w.dtype == torch.float64 and log_w.is_contiguous() and log_w.numel() == lnL.numel())
        ids = torch.empty(int(n_out), dtype=torch.int64, device=lnL.device)
        _check(load().ile_resample(self._h, lnL.numel(), _ptr(lnL), _ptr(log_w), int(n_out), float(v0), _ptr(ids),
                                   _stream_ptr(stream)), "ile_resample")
        return ids

    def harvest(self, samples, ids=None, v=None, point: int = 0, stream=None):
        """ile_harvest: -> (argmax_bin int32 [n_sel], lnL_max [n_sel], drawn_bin int32 [n_sel] or None)."""
        import torch

        ptrs, n = self._sample_ptrs(samples)
        n_sel = n if ids is None else ids.numel()
        assert ids is None or (ids.is_cuda and ids.dtype == torch.int64 and ids.is_contiguous())
        assert v is None or (v.is_cuda and v.dtype == torch.float64 and v.is_contiguous() and v.numel() == n_sel)
        dev = samples["ra"].device
        amax = torch.empty(n_sel, dtype=torch.int32, device=dev)
        lmax = torch.empty(n_sel, dtype=torch.float64, device=dev)
        drawn = torch.empty(n_sel, dtype=torch.int32, device=dev) if v is not None else None
        _check(load().ile_harvest(self._h, int(point), n, *ptrs, n_sel, _ptr(ids), _ptr(v), _ptr(amax), _ptr(lmax), _ptr(drawn),
                                  _stream_ptr(stream)), "ile_harvest")
        return amax, lmax, drawn

    def status(self, reset: bool = False, stream=None):
        """ile_status: (n_out_of_range, code).  Synchronises the stream."""
        v = ctypes.c_int64(0)
        code = load().ile_status(self._h, ctypes.byref(v), int(reset), _stream_ptr(stream))
        if code not in (0, -5):
            raise IleError(code, "ile_status")
        return int(v.value), code


class Sampler:
    """Owns one ile_sampler (NEXT-2).  cfg: dict(seed, n_bins, adapt (RA, dec, distance), floor_frac, temper, dist_min_mpc,
    dist_max_mpc, t_ref_lo_s, t_ref_hi_s)."""

    def __init__(self, cfg):
        self.n_bins = int(cfg["n_bins"])
        c = _SamplerConfig(int(cfg["seed"]), self.n_bins, int(bool(cfg["adapt"][0])), int(bool(cfg["adapt"][1])),
                           int(bool(cfg["adapt"][2])), float(cfg["floor_frac"]), float(cfg["temper"]), float(cfg["dist_min_mpc"]),
                           float(cfg["dist_max_mpc"]), float(cfg["t_ref_lo_s"]), float(cfg["t_ref_hi_s"]))
        self._h = ctypes.c_void_p()
        _check(load().ile_sampler_create(ctypes.byref(self._h), ctypes.byref(c)), "ile_sampler_create")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load().ile_sampler_destroy(self._h)
            self._h = ctypes.c_void_p()

    __del__ = close

    @property
    def launch_count(self) -> int:
        return int(load().ile_sampler_launch_count(self._h))

    def reset(self, stream=None):
        _check(load().ile_sampler_reset(self._h, _stream_ptr(stream)), "ile_sampler_reset")

    def set_tables(self, h, stream=None):
        import numpy as np

        h = np.ascontiguousarray(h, dtype=np.float64)
        assert h.shape == (3, self.n_bins)
        _check(load().ile_sampler_set_tables(self._h, ctypes.c_void_p(h.ctypes.data), _stream_ptr(stream)), "ile_sampler_set_tables")

    def get_tables(self, stream=None):
        import numpy as np

        h, C = np.empty((3, self.n_bins)), np.empty((3, self.n_bins + 1))
        _check(load().ile_sampler_get_tables(self._h, ctypes.c_void_p(h.ctypes.data), ctypes.c_void_p(C.ctypes.data),
                                             _stream_ptr(stream)), "ile_sampler_get_tables")
        return h, C

    def uniforms(self, first_index: int, n: int, stream=None):
        import torch

        u = torch.empty((n, 7), dtype=torch.float64, device="cuda")
        _check(load().ile_sampler_uniforms(self._h, int(first_index), int(n), _ptr(u), _stream_ptr(stream)), "ile_sampler_uniforms")
        return u

    def draw(self, first_index: int, n: int, stream=None):
        """-> (samples dict of CUDA float64 [n] as Context.eval takes it, log_w [n], bin_idx int32 [n][3])."""
        import torch

        s = {f: torch.empty(n, dtype=torch.float64, device="cuda") for f in SAMPLE_FIELDS}
        lw = torch.empty(n, dtype=torch.float64, device="cuda")
        bins = torch.empty((n, 3), dtype=torch.int32, device="cuda")
        _check(load().ile_sampler_draw(self._h, int(first_index), int(n), *[_ptr(s[f]) for f in SAMPLE_FIELDS], _ptr(lw), _ptr(bins),
                                       _stream_ptr(stream)), "ile_sampler_draw")
        return s, lw, bins

    def refit(self, bins, lnL, log_w=None, stream=None):
        import torch

        n = lnL.numel()
        assert bins.is_cuda and bins.dtype == torch.int32 and bins.is_contiguous() and bins.numel() == 3 * n
        assert lnL.is_cuda and lnL.dtype == torch.float64 and lnL.is_contiguous()
        assert log_w is None or (log_w.is_cuda and log_w.dtype == torch.float64 and log_w.is_contiguous() and log_w.numel() == n)
        _check(load().ile_sampler_refit(self._h, n, _ptr(bins), _ptr(lnL), _ptr(log_w), _stream_ptr(stream)), "ile_sampler_refit")


def integrate(ctx: "Context", sampler: "Sampler", n_chunk: int, max_chunks: int, n_adapt_chunks: int, n_eff_min: float,
              point: int = 0, stream=None):
    """ile_integrate: the adaptive Monte Carlo loop on the device -> dict(lnZ, n_eff, n_samples, n_chunks, history [c][2])."""
    import numpy as np

    lnZ, neff, ns = ctypes.c_double(0.0), ctypes.c_double(0.0), ctypes.c_int64(0)
    hist = np.zeros((int(max_chunks), 2))
    _check(load().ile_integrate(ctx._h, sampler._h, int(point), int(n_chunk), int(max_chunks), int(n_adapt_chunks), float(n_eff_min),
                                ctypes.byref(lnZ), ctypes.byref(neff), ctypes.byref(ns), ctypes.c_void_p(hist.ctypes.data),
                                _stream_ptr(stream)), "ile_integrate")
    nc = int(ns.value) // int(n_chunk)
    return dict(lnZ=lnZ.value, n_eff=neff.value, n_samples=int(ns.value), n_chunks=nc, history=hist[:nc])


def evidence_static(lnL, log_w=None, state=None, n_segments: int = 1, out=None, stream=None):
    """ile_evidence_static: the evidence reduction for callers that may not allocate device memory -- no Context (whose
    creation is a series of cudaMalloc calls) is needed; the kernel's scratch is a fixed 68 KiB array inside the library
    (see include/ile.h for who needs this and for the rules: at most ILE_EVIDENCE_STATIC_MAX_SEGMENTS = 1024 segments, one
    shared array per device, so calls that may overlap on the GPU race; first call on a device before any stream capture).
    lnL [n_segments][n_per_segment] CUDA float64 -> (lnZ, n_eff) CUDA tensors [n_segments].  Pass `out=(lnZ, n_eff)`
    (preallocated) if even PyTorch's allocator must stay untouched; `state` [n_segments][3] must start as (-inf, 0, 0)."""
    import torch

    assert lnL.is_cuda and lnL.dtype == torch.float64 and lnL.is_contiguous()
    n = lnL.numel()
    assert n % n_segments == 0
    if log_w is not None:
        assert log_w.is_cuda and log_w.dtype == torch.float64 and log_w.is_contiguous() and log_w.numel() == n
    if out is None:
        out = (torch.empty(n_segments, dtype=torch.float64, device=lnL.device),
               torch.empty(n_segments, dtype=torch.float64, device=lnL.device))
    lnZ, neff = out
    assert lnZ.numel() == n_segments and neff.numel() == n_segments
    with torch.cuda.device(lnL.device):
        _check(load().ile_evidence_static(int(n_segments), n // n_segments, _ptr(lnL), _ptr(log_w), _ptr(state), _ptr(lnZ),
                                          _ptr(neff), _stream_ptr(stream)), "ile_evidence_static")
    return lnZ, neff


def precompute(x, d, fs_hz: float, t0_q_s: float, stream=None):
    """ile_precompute: whitened mode spectra x [P][K][M][N] and data spectra d [P][K][N] (CUDA complex128, FFT order)
    -> (Q [P][K][M][N], U [P][K][M][M], V [P][K][M][M]) CUDA complex128 tensors, the inputs of ile_create (eq. 8a-c)."""
    import torch

    assert x.is_cuda and d.is_cuda and x.dtype == torch.complex128 and d.dtype == torch.complex128
    assert x.is_contiguous() and d.is_contiguous() and x.dim() == 4 and d.dim() == 3 and tuple(d.shape) == (x.shape[0], x.shape[1], x.shape[3])
    P, K, M, N = (int(v) for v in x.shape)
    Q = torch.empty((P, K, M, N), dtype=torch.complex128, device=x.device)
    U = torch.empty((P, K, M, M), dtype=torch.complex128, device=x.device)
    V = torch.empty((P, K, M, M), dtype=torch.complex128, device=x.device)
    _check(load().ile_precompute(P, K, M, N, float(fs_hz), float(t0_q_s), _ptr(x), _ptr(d), _ptr(Q), _ptr(U), _ptr(V),
                                 _stream_ptr(stream)), "ile_precompute")
    return Q, U, V


def precompute_psd(h, d, S, fs_hz: float, t0_q_s: float, f_min_hz: float, f_max_hz: float, scale: float, stream=None):
    """ile_precompute_psd: un-whitened mode spectra h [P][K][M][N], data spectra d [P][K][N] (CUDA complex128), one-sided PSD
    S [P][K][N] (CUDA float64, FFT order) -> (Q, U, V) with eq. 2's 1/S weighting and band cut applied on the device."""
    import torch

    assert h.is_cuda and d.is_cuda and S.is_cuda and h.dtype == torch.complex128 and d.dtype == torch.complex128 and S.dtype == torch.float64
    assert h.is_contiguous() and d.is_contiguous() and S.is_contiguous() and h.dim() == 4 and tuple(d.shape) == (h.shape[0], h.shape[1], h.shape[3])
    assert tuple(S.shape) == tuple(d.shape)
    P, K, M, N = (int(v) for v in h.shape)
    Q = torch.empty((P, K, M, N), dtype=torch.complex128, device=h.device)
    U = torch.empty((P, K, M, M), dtype=torch.complex128, device=h.device)
    V = torch.empty((P, K, M, M), dtype=torch.complex128, device=h.device)
    _check(load().ile_precompute_psd(P, K, M, N, float(fs_hz), float(t0_q_s), _ptr(h), _ptr(d), _ptr(S), float(f_min_hz), float(f_max_hz),
                                     float(scale), _ptr(Q), _ptr(U), _ptr(V), _stream_ptr(stream)), "ile_precompute_psd")
    return Q, U, V


def gather_evidence_states(state, group=None):
    """Plumbing for several GPUs working on ONE intrinsic point: all-gather every rank's evidence state
    ([n_segments][3], as ile_evidence leaves it) -> [world][n_segments][3] on every rank, ready for
    Context.evidence_merge.  No arithmetic here; works with any torch.distributed backend (nccl on GPUs, gloo on CPU)."""
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    out = [torch.empty_like(state) for _ in range(world)]
    dist.all_gather(out, state.contiguous(), group=group)
    return torch.stack(out, 0).contiguous()


def samples_to_device(samples_np, device="cuda"):
    """numpy dict (ile_inputs.make_samples) -> dict of contiguous CUDA float64 tensors."""
    import torch

    return {f: torch.from_numpy(samples_np[f]).to(device) for f in SAMPLE_FIELDS}
