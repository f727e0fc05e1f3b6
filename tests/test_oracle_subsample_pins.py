"""Pins for the interpolated-shift oracle (oracle/subsample.py, NEXT-4): a band-limited analytic signal whose value between
samples is known in closed form, the reduction to the nearest-sample oracle on integer arrival times, and shift covariance."""
import numpy as np

import ile_inputs as gi
import oracle
from oracle import subsample as osub


def _tone_config(freqs_hz, seed=3):
    """Config 0's geometry with Q_k,lm[i] = c_k,lm exp(2 pi i f_k,lm tau_i): the continuous-time Q is the same formula at any tau."""
    cfg = gi.make_config(0)
    rng = np.random.default_rng(seed)
    K, M, n_q = cfg["n_det"], cfg["n_modes"], cfg["n_q"]
    c = rng.standard_normal((K, M)) + 1j * rng.standard_normal((K, M))
    f = np.array(freqs_hz, dtype=float).reshape(K, M)
    tau = cfg["t0_q_s"] + np.arange(n_q) / cfg["fs_hz"]
    cfg = dict(cfg)
    cfg["Q"] = (c[:, :, None] * np.exp(2j * np.pi * f[:, :, None] * tau[None, None, :]))[None]
    return cfg, c, f


def _exact_series(cfg, c, f, s):
    """lnL_j with the CONTINUOUS Q at the exact arrival times t_ref + dt_k + (j - N_t/2) / f_s (test-side closed form)."""
    K, M, n_t, fs = cfg["n_det"], cfg["n_modes"], cfg["n_t"], cfg["fs_hz"]
    a = cfg["d_ref_mpc"] / s["dist_mpc"]
    F = [oracle.antenna(cfg["arm_x"][k], cfg["arm_y"][k], cfg["gmst_rad"], s["ra"], s["dec"], s["psi"]) for k in range(K)]
    Y = [oracle.sYlm(int(cfg["l"][m]), int(cfg["m"][m]), s["incl"], -s["phi_ref"]) for m in range(M)]
    qd = oracle.quad(np.array(F), np.array(Y), cfg["U"][0], cfg["V"][0], a)
    j = np.arange(n_t)
    acc = np.zeros(n_t, dtype=complex)
    for k in range(K):
        t = s["t_ref"] + oracle.delay(cfg["vertex_m"][k], cfg["gmst_rad"], s["ra"], s["dec"]) + (j - n_t // 2) / fs
        for m in range(M):
            acc += np.conj(F[k] * Y[m]) * c[k, m] * np.exp(2j * np.pi * f[k, m] * t)
    return a * acc.real - qd, F, Y, a


def test_linear_interpolation_against_band_limited_closed_form():
    """Error of linear interpolation of a tone of frequency f sampled at f_s is at most (2 pi f / f_s)^2 / 8 of its amplitude;
    the nearest-sample series is off by up to pi f / f_s.  The interpolated oracle meets the first bound and beats the
    nearest-sample oracle by an order of magnitude."""
    cfg, c, f = _tone_config([30.0, 55.0, 41.0, 72.0])
    samples = gi.make_samples(11, 40)
    worst_lin = worst_near = 0.0
    for i in range(40):
        s = {k: float(samples[k][i]) for k in samples}
        exact, F, Y, a = _exact_series(cfg, c, f, s)
        lin, _, i0, phi, oob = osub.sample_series_lin(cfg, s)
        near = oracle.sample_series(cfg, s)[0]
        assert not oob and np.all((phi >= 0) & (phi < 1))
        bound = a * sum(abs(F[k] * Y[m]) * abs(c[k, m]) * (2 * np.pi * f[k, m] / cfg["fs_hz"]) ** 2 / 8 for k in range(2) for m in range(2))
        assert np.max(np.abs(lin - exact)) <= bound * (1 + 1e-9) + 1e-12
        worst_lin = max(worst_lin, np.max(np.abs(lin - exact)))
        worst_near = max(worst_near, np.max(np.abs(near - exact)))
    assert worst_lin < 0.1 * worst_near


def test_integer_arrival_times_reduce_to_the_nearest_sample_oracle_and_shift_covariance():
    cfg = gi.make_config(0)
    cfg = dict(cfg)
    cfg["vertex_m"] = np.zeros_like(cfg["vertex_m"])          # detectors at the geocentre: dt_k = 0, x_k = (t_ref - t0) f_s
    s = {k: float(v[0]) for k, v in gi.make_samples(5, 1).items()}
    for nshift in (-7, 0, 12):
        s["t_ref"] = nshift / cfg["fs_hz"]                      # exact in binary: x_k is an integer, phi = 0
        lin, mt, i0, phi, oob = osub.sample_series_lin(cfg, s)
        near, mt2, i02, oob2 = oracle.sample_series(cfg, s)
        assert np.all(phi == 0.0) and np.array_equal(i0, i02) and not oob
        assert np.max(np.abs(lin - near)) <= 1e-12 * max(1.0, np.max(np.abs(near))) and abs(mt - mt2) <= 1e-12 * max(1.0, abs(mt2))
    # half-way between two samples the series is the mean of the two nearest-sample series
    s["t_ref"] = 3.5 / cfg["fs_hz"]
    lin, _, i0, phi, _ = osub.sample_series_lin(cfg, s)
    s["t_ref"] = 3.0 / cfg["fs_hz"]
    lo = oracle.sample_series(cfg, s)[0]
    s["t_ref"] = 4.0 / cfg["fs_hz"]
    hi = oracle.sample_series(cfg, s)[0]
    assert np.all(phi == 0.5) and np.max(np.abs(lin - 0.5 * (lo + hi))) < 1e-12 * max(1.0, np.max(np.abs(lo)))
    # range: the interpolated window needs one sample more
    cfg2 = dict(cfg)
    cfg2["n_t"] = cfg["n_q"]
    s["t_ref"] = 0.0
    assert osub.sample_series_lin(cfg2, s)[4] and not oracle.sample_series(cfg2, s)[3]
    out, idx, bad = osub.eval_batch_lin(cfg, gi.make_samples(9, 5))
    assert bad == 0 and np.all(np.isfinite(out))
