"""ctypes binding of the CPU oracle (oracle/ile_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from paper_1902_04934_b200 and shares no code with it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ile_oracle.c")
_LIB = os.path.join(_HERE, "libile_oracle.so")
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int32)
_vp = ctypes.c_void_p


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp -shared; rebuilt when the source is newer than the library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-std=gnu11", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        d, i32, i64 = ctypes.c_double, ctypes.c_int32, ctypes.c_int64
        L.ile_oracle_antenna.argtypes = [_dp, _dp, d, d, d, d, _dp]
        L.ile_oracle_antenna.restype = None
        L.ile_oracle_delay.argtypes = [_dp, d, d, d]
        L.ile_oracle_delay.restype = d
        L.ile_oracle_window_index.argtypes = [d, d, d, d, i32]
        L.ile_oracle_window_index.restype = i32
        L.ile_oracle_wigner_d.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, d]
        L.ile_oracle_wigner_d.restype = d
        L.ile_oracle_sYlm.argtypes = [ctypes.c_int, ctypes.c_int, d, d, _dp]
        L.ile_oracle_sYlm.restype = None
        L.ile_oracle_quad.argtypes = [ctypes.c_int, ctypes.c_int, _vp, _vp, _vp, _vp, d]
        L.ile_oracle_quad.restype = d
        L.ile_oracle_margT.argtypes = [_dp, i32]
        L.ile_oracle_margT.restype = d
        L.ile_oracle_sample.argtypes = [ctypes.c_int, ctypes.c_int, _ip, _ip, i32, i32, d, d, d, d, _dp, _dp, _dp,
                                        _vp, _vp, _vp, d, d, d, d, d, d, d, _dp, _ip, ctypes.POINTER(ctypes.c_int)]
        L.ile_oracle_sample.restype = d
        L.ile_oracle_eval.argtypes = [ctypes.c_int, ctypes.c_int, _ip, _ip, i32, i32, d, d, d, d, _dp, _dp, _dp,
                                      _vp, _vp, _vp, i64, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _ip, ctypes.c_int]
        L.ile_oracle_eval.restype = i64
        L.ile_oracle_evidence.argtypes = [i64, _dp, _dp, _dp, _dp]
        L.ile_oracle_evidence.restype = None
        _lib = L
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a, ctypes.c_void_p(a.ctypes.data)


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(_ip)


def antenna(arm_x, arm_y, gmst, ra, dec, psi) -> complex:
    """O1: F_k = F+ + i Fx."""
    ax, pax = _d(arm_x)
    ay, pay = _d(arm_y)
    out = np.zeros(2)
    lib().ile_oracle_antenna(pax, pay, gmst, ra, dec, psi, out.ctypes.data_as(_dp))
    return complex(out[0], out[1])


def delay(vertex_m, gmst, ra, dec) -> float:
    """O2: arrival-time offset relative to the geocentre (s)."""
    v, pv = _d(vertex_m)
    return float(lib().ile_oracle_delay(pv, gmst, ra, dec))


def window_index(t_ref, dt, t0_q, fs, n_t) -> int:
    return int(lib().ile_oracle_window_index(t_ref, dt, t0_q, fs, n_t))


def wigner_d(l, mp, m, beta) -> float:
    return float(lib().ile_oracle_wigner_d(l, mp, m, beta))


def sYlm(l, m, theta, phi) -> complex:
    """O3: spin-weight -2 spherical harmonic."""
    out = np.zeros(2)
    lib().ile_oracle_sYlm(l, m, theta, phi, out.ctypes.data_as(_dp))
    return complex(out[0], out[1])


def quad(F, Y, U, V, a) -> float:
    """O4."""
    F, pF = _c(F)
    Y, pY = _c(Y)
    U, pU = _c(U)
    V, pV = _c(V)
    return float(lib().ile_oracle_quad(F.shape[0], Y.shape[0], pF, pY, pU, pV, a))


def margT(lnL) -> float:
    """O6."""
    x, px = _d(lnL)
    return float(lib().ile_oracle_margT(px, x.shape[0]))


def _cfg_args(cfg, point):
    l, pl = _i(cfg["l"])
    m, pm = _i(cfg["m"])
    v, pv = _d(cfg["vertex_m"])
    ax, pax = _d(cfg["arm_x"])
    ay, pay = _d(cfg["arm_y"])
    Q, pQ = _c(cfg["Q"][point])
    U, pU = _c(cfg["U"][point])
    V, pV = _c(cfg["V"][point])
    keep = (l, m, v, ax, ay, Q, U, V)
    args = [int(cfg["n_det"]), int(cfg["n_modes"]), pl, pm, int(cfg["n_q"]), int(cfg["n_t"]), float(cfg["fs_hz"]),
            float(cfg["t0_q_s"]), float(cfg["gmst_rad"]), float(cfg["d_ref_mpc"]), pv, pax, pay, pQ, pU, pV]
    return args, keep


def sample_series(cfg, sample, point: int = 0):
    """O1-O6 for ONE sample: (lnL_j [n_t], lnL_margT, shift_idx [K], out_of_range)."""
    args, keep = _cfg_args(cfg, point)
    series = np.zeros(int(cfg["n_t"]))
    idx = np.zeros(int(cfg["n_det"]), dtype=np.int32)
    oob = ctypes.c_int(0)
    val = lib().ile_oracle_sample(*args, *[float(sample[f]) for f in ("ra", "dec", "t_ref", "phi_ref", "psi", "incl", "dist_mpc")],
                                  series.ctypes.data_as(_dp), idx.ctypes.data_as(_ip), ctypes.byref(oob))
    return series, float(val), idx, bool(oob.value)


def eval_batch(cfg, samples, point: int = 0, n_threads: int = 1):
    """O1-O6 for a batch: (lnL_margT [n], shift_idx [n][K], n_out_of_range)."""
    args, keep = _cfg_args(cfg, point)
    arrs = [_d(samples[f]) for f in ("ra", "dec", "t_ref", "phi_ref", "psi", "incl", "dist_mpc")]
    n = arrs[0][0].shape[0]
    out = np.zeros(n)
    idx = np.zeros((n, int(cfg["n_det"])), dtype=np.int32)
    bad = lib().ile_oracle_eval(*args, n, *[p for _, p in arrs], out.ctypes.data_as(_dp), idx.ctypes.data_as(_ip),
                                int(n_threads))
    return out, idx, int(bad)


def evidence(lnL_margT, log_w=None):
    """O7, O8: (lnZ, n_eff)."""
    x, px = _d(lnL_margT)
    if log_w is None:
        pw = ctypes.cast(None, _dp)
    else:
        w, pw = _d(log_w)
    lnZ, neff = ctypes.c_double(0.0), ctypes.c_double(0.0)
    lib().ile_oracle_evidence(x.shape[0], px, pw, ctypes.byref(lnZ), ctypes.byref(neff))
    return float(lnZ.value), float(neff.value)
