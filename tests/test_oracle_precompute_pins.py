"""Pins of oracle/precompute.py (eq. 8a-c) against what the definition and the mathematics fix.
A plausible mistake -- a missing conjugate, the wrong sign of the exponent, f -> -f on the wrong factor, a roll by the
wrong half, a transposed U -- fails at least one of these."""
import numpy as np
import pytest

from oracle import precompute as pc

FS = 4096.0


def rnd(shape, seed):
    r = np.random.default_rng(seed)
    return r.standard_normal(shape) + 1j * r.standard_normal(shape)


def test_fft_path_equals_term_by_term_definition():
    K, M, N = 2, 3, 32
    x, d = rnd((K, M, N), 1), rnd((K, N), 2)
    for t0 in (0.0, -N / (2 * FS), 3.25 / FS):  # also a start time that is not a whole number of samples
        a = pc.overlaps(x, d, FS, t0)
        b = pc.overlaps_direct(x, d, FS, t0)
        for u, v in zip(a, b):
            assert np.max(np.abs(u - v)) <= 1e-12 * np.max(np.abs(v))


def test_data_equal_to_a_mode_reproduces_U_at_zero_lag_and_V_for_the_conjugate_mode():
    """eq. 8 consistency: d = h_b gives Q_a(tau = 0) = <h_a|h_b> = U_ab; d = conj-reflected h_b gives <h_a|h_b^*> = conj(V_ba)...
    written out: sum_n conj(x_a[n]) conj(x_b[-n]) = conj(sum_n x_a[n] x_b[-n]) = conj(V_ba)."""
    M, N = 3, 64
    x = rnd((1, M, N), 3)
    neg = (-np.arange(N)) % N
    i0 = N // 2  # tau_i = 0 for t0 = -N / (2 fs)
    t0 = -N / (2 * FS)
    for b in range(M):
        Q, U, V = pc.overlaps(x, x[:, b, :], FS, t0)
        assert np.allclose(Q[0, :, i0], U[0, :, b], rtol=1e-12, atol=0)
        Qc, _, _ = pc.overlaps(x, np.conj(x[:, b, neg]), FS, t0)
        assert np.allclose(Qc[0, :, i0], np.conj(V[0, b, :]), rtol=1e-12, atol=0)


def test_delaying_the_data_by_s_samples_moves_the_peak_s_samples_later():
    """d(f) exp(-2 pi i f s / fs) is the data delayed by s samples: Q[i] -> Q[i - s] (circular), exactly."""
    K, M, N, s = 1, 2, 64, 5
    x, d = rnd((K, M, N), 4), rnd((K, N), 5)
    f = pc.signed_index(N) * FS / N
    Q0, _, _ = pc.overlaps(x, d, FS, -N / (2 * FS))
    Q1, _, _ = pc.overlaps(x, d * np.exp(-2j * np.pi * f * s / FS), FS, -N / (2 * FS))
    assert np.max(np.abs(Q1 - np.roll(Q0, s, axis=-1))) <= 1e-12 * np.max(np.abs(Q0))


def test_U_hermitian_positive_V_symmetric_and_closed_forms():
    K, M, N = 2, 4, 128
    x = rnd((K, M, N), 6)
    _, U, V = pc.overlaps(x, rnd((K, N), 7), FS, 0.0)
    for k in range(K):
        assert np.allclose(U[k], U[k].conj().T, rtol=1e-13, atol=1e-12)
        assert np.all(np.linalg.eigvalsh(U[k]) > 0)
        assert np.allclose(V[k], V[k].T, rtol=1e-13, atol=1e-12)
        assert np.allclose(np.diag(U[k]).real, np.sum(np.abs(x[k]) ** 2, axis=1), rtol=1e-13)
    # one-sided modes (support on f > 0 only): V_aa = sum x_a(-f) x_a(f) = 0, the non-precessing structure
    xs = x.copy()
    xs[:, :, pc.signed_index(N) <= 0] = 0.0
    _, _, Vs = pc.overlaps(xs, rnd((K, N), 8), FS, 0.0)
    assert np.max(np.abs(Vs)) == 0.0


def test_parseval_and_single_tone():
    N = 64
    x, d = rnd((1, 1, N), 9), rnd((1, N), 10)
    Q, _, _ = pc.overlaps(x, d, FS, 0.0)
    assert np.isclose(np.sum(np.abs(Q) ** 2), N * np.sum(np.abs(np.conj(x[0, 0]) * d[0]) ** 2), rtol=1e-12)
    # a single spectral line at signed index m: Q[i] = conj(x_m) d_m exp(2 pi i m (t0 fs + i) / N)
    m, t0 = -7, 2.0 / FS
    xt, dt = np.zeros((1, 1, N), complex), np.zeros((1, N), complex)
    xt[0, 0, m % N], dt[0, m % N] = 0.3 - 0.4j, 1.5 + 2.0j
    Qt, _, _ = pc.overlaps(xt, dt, FS, t0)
    i = np.arange(N)
    assert np.allclose(Qt[0, 0], np.conj(0.3 - 0.4j) * (1.5 + 2.0j) * np.exp(2j * np.pi * m * (t0 * FS + i) / N), rtol=1e-12, atol=1e-13)


def test_generator_and_oracle_agree_on_a_config_point():
    """The seeded input recipe (ile_inputs) and the oracle define the same Q, U, V."""
    import ile_inputs as gi

    c = gi.CONFIGS[0]
    Q, U, V, meta = gi.make_point(gi.point_seed(0, 0), c["dets"], c["modes"], c["n_q"], c["snr"], admix=c["admix"], spectra=True)
    q, u, v = pc.overlaps(meta["x"], meta["d"], meta["fs_hz"], meta["t0_q_s"])
    for got, ref in ((q, Q), (u, U), (v, V)):
        assert np.max(np.abs(got - ref)) <= 1e-13 * np.max(np.abs(ref))


# ----------------------------------------------------------------------------------------------------------
# eq. 2's weighting on un-whitened spectra: overlaps_psd
# ----------------------------------------------------------------------------------------------------------
def _unwhitened(seed, K=2, M=3, N=64, fs=256.0):
    rng = np.random.default_rng(seed)
    h = rng.standard_normal((K, M, N)) + 1j * rng.standard_normal((K, M, N))
    d = rng.standard_normal((K, N)) + 1j * rng.standard_normal((K, N))
    f = np.abs(pc.signed_index(N) * fs / N)
    S = np.stack([(1.0 + k) * (1.0 + (f / 40.0) ** 2 + (10.0 / np.maximum(f, 1.0)) ** 4) for k in range(K)])
    return h, d, S, fs


def test_psd_inner_product_is_eq2_by_brute_force():
    """U_ab with scale = 2 df is eq. 2's <h_a|h_b> = 2 int_{f_min<|f|<f_max} h_a*(f) h_b(f) / S(|f|) df as a plain Riemann sum over
    the two-sided grid, written here term by term; Q at lag 0 with d = h_b is the same number; V pairs f with -f."""
    h, d, S, fs = _unwhitened(1)
    K, M, N = h.shape
    df, fmin, fmax, t0 = fs / N, 14.0, 90.0, 0.0
    Q, U, V = pc.overlaps_psd(h, d, S, fs, t0, fmin, fmax, 2.0 * df)
    npr = pc.signed_index(N)
    for k in range(K):
        for a in range(M):
            for b in range(M):
                u = v = 0j
                for n in range(N):
                    f = abs(npr[n]) * df
                    if not (fmin < f < fmax):
                        continue
                    u += 2.0 * np.conj(h[k, a, n]) * h[k, b, n] / S[k, n] * df
                    v += 2.0 * h[k, a, (-n) % N] * h[k, b, n] / S[k, n] * df
                assert abs(U[k, a, b] - u) <= 1e-12 * abs(u) and abs(V[k, a, b] - v) <= 1e-12 * max(abs(v), 1e-3)
            Qb = pc.overlaps_psd(h, h[:, a], S, fs, 0.0, fmin, fmax, 2.0 * df)[0]
            for b in range(M):
                assert abs(Qb[k, b, 0] - U[k, b, a]) <= 1e-12 * abs(U[k, b, a])
        assert np.allclose(U[k], U[k].conj().T, rtol=1e-13) and np.allclose(V[k], V[k].T, rtol=1e-13)


def test_psd_form_equals_whitened_form_and_respects_the_band():
    """Whitening by hand -- x = h sqrt(g), d_w = d sqrt(g) -- and the plain form give the same Q, U, V (this links the new entry to
    the one pinned above); S = 1 over the whole band is the plain form itself; data outside the band changes nothing; the lag
    axis is the same (a delayed copy of the data moves the peak of Q by the delay)."""
    h, d, S, fs = _unwhitened(2)
    K, M, N = h.shape
    t0, fmin, fmax, scale = -0.07, 9.0, 100.0, 0.37
    Q, U, V = pc.overlaps_psd(h, d, S, fs, t0, fmin, fmax, scale)
    g = np.stack([pc.psd_weights(N, S[k], fs, fmin, fmax, scale) for k in range(K)])
    Qw, Uw, Vw = pc.overlaps(h * np.sqrt(g)[:, None, :], d * np.sqrt(g), fs, t0)
    for got, ref in ((Q, Qw), (U, Uw), (V, Vw)):
        assert np.max(np.abs(got - ref)) <= 1e-12 * np.max(np.abs(ref))
    Q1, U1, V1 = pc.overlaps_psd(h, d, np.ones_like(S), fs, t0, -1.0, 1e9, 1.0)
    Q0, U0, V0 = pc.overlaps(h, d, fs, t0)
    assert np.max(np.abs(Q1 - Q0)) <= 1e-12 * np.max(np.abs(Q0)) and np.allclose(U1, U0, rtol=1e-13) and np.allclose(V1, V0, rtol=1e-13)
    d2 = d.copy()
    out = g[0] == 0.0
    d2[:, out] += 100.0
    assert np.max(np.abs(pc.overlaps_psd(h, d2, S, fs, t0, fmin, fmax, scale)[0] - Q)) <= 1e-10 * np.max(np.abs(Q))
    Qd, Ud, Vd = pc.overlaps_direct_psd(h[:1, :2, :16], d[:1, :16], S[:1, :16], fs, t0, 20.0, 100.0, scale)
    Qf, Uf, Vf = pc.overlaps_psd(h[:1, :2, :16], d[:1, :16], S[:1, :16], fs, t0, 20.0, 100.0, scale)
    assert np.max(np.abs(Qd - Qf)) <= 1e-12 * np.max(np.abs(Qf)) and np.allclose(Ud, Uf, rtol=1e-12) and np.allclose(Vd, Vf, rtol=1e-12, atol=1e-12)
