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
