"""Pins for the CPU oracle (oracle/ile_oracle.c): every function is checked against something OTHER than
itself -- brute-force eq. 1+2, textbook closed forms, invariants, special cases (SURVEY.md §8(c) "What pins each
part").  Nothing here retypes an oracle formula: the independent side is vector algebra, FFT inner products,
closed forms from the literature, quadrature, or exact summation.  All CPU, -m "not gpu".

Citations are /root/reference/PAPER.md lines.
"""
import math

import numpy as np
import pytest

import ile_inputs as gi
import oracle

C_SI = 299792458.0
RNG = np.random.default_rng(20240607)


# ----------------------------------------------------------------------------------------------------------
# independent helpers (test-side only)
# ----------------------------------------------------------------------------------------------------------
def source_dir(ra, dec, gmst):
    """Unit vector Earth -> source in the Earth-fixed frame (Greenwich hour angle = gmst - ra)."""
    lon = ra - gmst
    return np.array([np.cos(dec) * np.cos(lon), np.cos(dec) * np.sin(lon), np.sin(dec)])


def pol_axes(ra, dec, psi, gmst):
    """Wave-frame axes by vector algebra: at psi = 0, X points local west and Y local north at the sub-source
    point (X x Y = propagation direction = -s); psi rotates X toward Y."""
    s = source_dir(ra, dec, gmst)
    z = np.array([0.0, 0.0, 1.0])
    east = np.cross(z, s)
    east /= np.linalg.norm(east)
    north = np.cross(s, east)
    X0, Y0 = -east, north
    X = np.cos(psi) * X0 + np.sin(psi) * Y0
    Y = -np.sin(psi) * X0 + np.cos(psi) * Y0
    return X, Y, s


def antenna_vec(arm_x, arm_y, ra, dec, psi, gmst):
    """F+, Fx = D : e+, D : ex with e+ = XX - YY, ex = XY + YX (tensor contraction written with outer products)."""
    X, Y, _ = pol_axes(ra, dec, psi, gmst)
    D = 0.5 * (np.outer(arm_x, arm_x) - np.outer(arm_y, arm_y))
    ep = np.outer(X, X) - np.outer(Y, Y)
    ec = np.outer(X, Y) + np.outer(Y, X)
    return float(np.sum(D * ep)), float(np.sum(D * ec))


def Y2m_closed(m, th, ph):
    """Textbook closed forms of the l = 2 spin-weight -2 harmonics."""
    c = np.cos(th)
    s = np.sin(th)
    if m == 2:
        v = np.sqrt(5.0 / (64.0 * np.pi)) * (1.0 + c) ** 2
    elif m == 1:
        v = np.sqrt(5.0 / (16.0 * np.pi)) * s * (1.0 + c)
    elif m == 0:
        v = np.sqrt(15.0 / (32.0 * np.pi)) * s * s
    elif m == -1:
        v = np.sqrt(5.0 / (16.0 * np.pi)) * s * (1.0 - c)
    elif m == -2:
        v = np.sqrt(5.0 / (64.0 * np.pi)) * (1.0 - c) ** 2
    else:
        raise ValueError(m)
    return v * np.exp(1j * m * ph)


def random_unit(rng):
    v = rng.standard_normal(3)
    return v / np.linalg.norm(v)


def random_orthonormal_arms(rng):
    x = random_unit(rng)
    y = random_unit(rng)
    y = y - np.dot(x, y) * x
    y /= np.linalg.norm(y)
    return x, y


# ----------------------------------------------------------------------------------------------------------
# O1 antenna response
# ----------------------------------------------------------------------------------------------------------
def test_O1_matches_vector_algebra_construction():
    for _ in range(200):
        ax, ay = random_orthonormal_arms(RNG)
        ra, dec, psi, gmst = RNG.uniform(0, 2 * np.pi), np.arcsin(RNG.uniform(-1, 1)), RNG.uniform(0, np.pi), RNG.uniform(0, 2 * np.pi)
        F = oracle.antenna(ax, ay, gmst, ra, dec, psi)
        fp, fc = antenna_vec(ax, ay, ra, dec, psi, gmst)
        assert abs(F.real - fp) < 1e-14 and abs(F.imag - fc) < 1e-14


def test_O1_textbook_detector_frame_formula():
    """Arms along Earth-fixed x, y (a detector at the pole), source at polar angles (theta, phi) in that frame:
    F+ = 1/2 (1+cos^2 th) cos 2ph cos 2ps - cos th sin 2ph sin 2ps,  Fx = 1/2 (1+cos^2 th) cos 2ph sin 2ps + cos th sin 2ph cos 2ps,
    with the textbook polarisation angle ps = pi/2 - psi: the textbook measures it from the other transverse
    reference axis and with the opposite handedness to the west/north axes about -s used here (reading R6)."""
    ax, ay = np.array([1.0, 0, 0]), np.array([0, 1.0, 0])
    for _ in range(200):
        th, ph, psi = np.arccos(RNG.uniform(-1, 1)), RNG.uniform(0, 2 * np.pi), RNG.uniform(0, np.pi)
        gmst = RNG.uniform(0, 2 * np.pi)
        F = oracle.antenna(ax, ay, gmst, ph + gmst, 0.5 * np.pi - th, psi)
        ps = 0.5 * np.pi - psi
        fp = 0.5 * (1 + np.cos(th) ** 2) * np.cos(2 * ph) * np.cos(2 * ps) - np.cos(th) * np.sin(2 * ph) * np.sin(2 * ps)
        fc = 0.5 * (1 + np.cos(th) ** 2) * np.cos(2 * ph) * np.sin(2 * ps) + np.cos(th) * np.sin(2 * ph) * np.cos(2 * ps)
        # convention-free part: the magnitude
        assert abs(abs(F) ** 2 - (fp * fp + fc * fc)) < 1e-13
        assert abs(F.real - fp) < 1e-13
        assert abs(F.imag - fc) < 1e-13


def test_O1_psi_dependence_and_invariants():
    for _ in range(100):
        ax, ay = random_orthonormal_arms(RNG)
        ra, dec, psi, gmst = RNG.uniform(0, 2 * np.pi), np.arcsin(RNG.uniform(-1, 1)), RNG.uniform(0, np.pi), 1.234
        F0 = oracle.antenna(ax, ay, gmst, ra, dec, 0.0)
        F = oracle.antenna(ax, ay, gmst, ra, dec, psi)
        assert abs(F - F0 * np.exp(-2j * psi)) < 1e-14            # F(psi) = F(0) e^{-2 i psi}
        assert abs(oracle.antenna(ax, ay, gmst, ra, dec, psi + np.pi) - F) < 1e-14       # check (d) at the F level
        assert abs(oracle.antenna(ax, ay, gmst, ra, dec, psi + 0.5 * np.pi) + F) < 1e-14  # psi + pi/2 flips the sign
        # only ra - gmst matters
        assert abs(oracle.antenna(ax, ay, gmst + 0.3, ra + 0.3, dec, psi) - F) < 1e-13


def test_O1_transversality_single_arm():
    """With arm_y = 0 and arm_x = u:  |F| = (1 - (s.u)^2)/2 iff X, Y, s are orthonormal (convention-free)."""
    zero = np.zeros(3)
    for _ in range(100):
        u = random_unit(RNG)
        ra, dec, psi, gmst = RNG.uniform(0, 2 * np.pi), np.arcsin(RNG.uniform(-1, 1)), RNG.uniform(0, np.pi), 0.77
        s = source_dir(ra, dec, gmst)
        F = oracle.antenna(u, zero, gmst, ra, dec, psi)
        assert abs(abs(F) - 0.5 * (1.0 - np.dot(s, u) ** 2)) < 1e-14
        assert abs(oracle.antenna(s, zero, gmst, ra, dec, psi)) < 1e-15      # arm along the line of sight sees nothing


def test_O1_sky_average_one_fifth():
    """<F+^2> = <Fx^2> = 1/5 over the sky and psi for orthogonal arms (textbook), by Gauss-Legendre x uniform quadrature."""
    ax = np.array(gi.DETECTORS["H1"]["arm_x"])
    ay = np.array(gi.DETECTORS["H1"]["arm_y"])
    mu, w = np.polynomial.legendre.leggauss(8)
    n_ra, n_psi = 16, 8
    sp = sc = 0.0
    for x, wx in zip(mu, w):
        for a in range(n_ra):
            for b in range(n_psi):
                F = oracle.antenna(ax, ay, 0.3, 2 * np.pi * a / n_ra, np.arcsin(x), np.pi * b / n_psi)
                sp += wx * F.real ** 2
                sc += wx * F.imag ** 2
    sp /= 2.0 * n_ra * n_psi
    sc /= 2.0 * n_ra * n_psi
    # H1's catalogued arms are orthogonal to ~2e-7
    assert abs(sp - 0.2) < 1e-6 and abs(sc - 0.2) < 1e-6


# ----------------------------------------------------------------------------------------------------------
# O2 arrival time and window index
# ----------------------------------------------------------------------------------------------------------
def test_O2_zenith_antipode_and_sign():
    gmst = gi.GMST_RAD
    for name in ("H1", "L1", "V1"):
        v = np.array(gi.DETECTORS[name]["vertex_m"])
        r = np.linalg.norm(v)
        dec = np.arcsin(v[2] / r)
        ra = np.arctan2(v[1], v[0]) + gmst
        assert abs(oracle.delay(v, gmst, ra, dec) + r / C_SI) < 1e-15          # overhead source: earliest arrival
        assert abs(oracle.delay(v, gmst, ra + np.pi, -dec) - r / C_SI) < 1e-15  # antipode: latest arrival
        assert abs(r / C_SI - 0.02124) < 2e-4                                   # Earth radius / c ~ 21.24 ms
    assert abs(oracle.delay(np.array([6.0e6, 0, 0]), 0.4, 0.4, 0.0) + 6.0e6 / C_SI) < 1e-17


def test_O2_matches_vector_formula_and_baseline_bound():
    gmst = gi.GMST_RAD
    vH, vL, vV = (np.array(gi.DETECTORS[d]["vertex_m"]) for d in ("H1", "L1", "V1"))
    for _ in range(300):
        ra, dec = RNG.uniform(0, 2 * np.pi), np.arcsin(RNG.uniform(-1, 1))
        s = source_dir(ra, dec, gmst)
        for v in (vH, vL, vV):
            assert abs(oracle.delay(v, gmst, ra, dec) + np.dot(v, s) / C_SI) < 1e-16
        assert abs(oracle.delay(vH, gmst, ra, dec) - oracle.delay(vL, gmst, ra, dec)) <= np.linalg.norm(vH - vL) / C_SI + 1e-15
    assert abs(np.linalg.norm(vH - vL) / C_SI - 0.010013) < 2e-6               # H1-L1 light travel time


def test_O2_window_index_rounding():
    # nearest sample, ties to even, minus floor(N_t/2)  (readings R8, R10)
    assert oracle.window_index(2.5, 0.0, 0.0, 1.0, 0) == 2
    assert oracle.window_index(3.5, 0.0, 0.0, 1.0, 0) == 4
    assert oracle.window_index(-0.5, 0.0, 0.0, 1.0, 0) == 0
    assert oracle.window_index(10.4, 0.0, 0.0, 1.0, 201) == 10 - 100
    assert oracle.window_index(10.6, 0.0, 0.0, 1.0, 410) == 11 - 205
    assert oracle.window_index(0.0, 0.001, -0.25, 4096.0, 410) == round((0.001 + 0.25) * 4096.0) - 205


def test_O2_index_against_extended_precision():
    """Indices from the binary64 oracle agree with an 80-bit evaluation of the same definition on seeded samples
    (a flip needs x within ~1e-13 of a half-integer): 100,000 samples x 3 detectors."""
    n = 100_000
    cfg = gi.make_config(1, n=n)
    s = gi.make_samples(cfg["sample_seeds"][0], n)
    _, idx, bad = oracle.eval_batch(cfg, s, n_threads=4)
    assert bad == 0
    ld = np.longdouble
    assert np.finfo(ld).nmant >= 63, "needs the x87 80-bit long double"
    for k in range(cfg["n_det"]):
        v = cfg["vertex_m"][k].astype(ld)
        ra, dec, t = s["ra"].astype(ld), s["dec"].astype(ld), s["t_ref"].astype(ld)
        lon = ra - ld(cfg["gmst_rad"])
        dot = v[0] * np.cos(dec) * np.cos(lon) + v[1] * np.cos(dec) * np.sin(lon) + v[2] * np.sin(dec)
        x = ((t - dot / ld(C_SI)) - ld(cfg["t0_q_s"])) * ld(cfg["fs_hz"])
        ref = np.rint(x).astype(np.int64) - cfg["n_t"] // 2
        assert np.array_equal(ref, idx[:, k].astype(np.int64))


# ----------------------------------------------------------------------------------------------------------
# O3 spin-weighted harmonics
# ----------------------------------------------------------------------------------------------------------
def test_O3_l2_closed_forms():
    for _ in range(100):
        th, ph = np.arccos(RNG.uniform(-1, 1)), RNG.uniform(0, 2 * np.pi)
        for m in range(-2, 3):
            assert abs(oracle.sYlm(2, m, th, ph) - Y2m_closed(m, th, ph)) < 2e-15


def test_O3_higher_l_closed_forms():
    """A few l = 3, 4 closed forms from the literature (e.g. Ajith et al. 0709.0093, App.)."""
    for _ in range(50):
        th, ph = np.arccos(RNG.uniform(-1, 1)), RNG.uniform(0, 2 * np.pi)
        ch, sh = np.cos(th / 2), np.sin(th / 2)
        y33 = -np.sqrt(21.0 / (2.0 * np.pi)) * ch ** 5 * sh * np.exp(3j * ph)
        y32 = 0.5 * np.sqrt(7.0 / np.pi) * ch ** 4 * (3.0 * np.cos(th) - 2.0) * np.exp(2j * ph)
        y44 = 3.0 * np.sqrt(7.0 / np.pi) * ch ** 6 * sh ** 2 * np.exp(4j * ph)
        y3m3 = np.sqrt(21.0 / (2.0 * np.pi)) * ch * sh ** 5 * np.exp(-3j * ph)
        assert abs(oracle.sYlm(3, 3, th, ph) - y33) < 5e-15
        assert abs(oracle.sYlm(3, 2, th, ph) - y32) < 5e-15
        assert abs(oracle.sYlm(4, 4, th, ph) - y44) < 5e-15
        assert abs(oracle.sYlm(3, -3, th, ph) - y3m3) < 5e-15


def test_O3_highest_weight_closed_form_to_l8():
    """m = l has a one-term closed form for every l (Goldberg et al. 1967 eq. 3.1 with s = -2):
    -2Y_ll = (-1)^l sqrt((2l+1)/4pi) sqrt((2l)! / ((l+2)! (l-2)!)) cos^(l+2)(theta/2) sin^(l-2)(theta/2) e^{i l phi};
    l = 5 is the literature's -sqrt(330/pi) cos^7 sin^3 e^{5 i phi}.  Pins the factorial bounds of O3 up to ILE_MAX_L = 8
    (eq. 5-6)."""
    from math import factorial as f
    for _ in range(50):
        th, ph = np.arccos(RNG.uniform(-1, 1)), RNG.uniform(0, 2 * np.pi)
        ch, sh = np.cos(th / 2), np.sin(th / 2)
        assert abs(oracle.sYlm(5, 5, th, ph) + np.sqrt(330.0 / np.pi) * ch ** 7 * sh ** 3 * np.exp(5j * ph)) < 5e-15
        for l in range(2, 9):
            v = (-1) ** l * np.sqrt((2 * l + 1) / (4 * np.pi)) * np.sqrt(f(2 * l) / (f(l + 2) * f(l - 2))) * ch ** (l + 2) * sh ** (l - 2) * np.exp(1j * l * ph)
            assert abs(oracle.sYlm(l, l, th, ph) - v) < 1e-14, l


def test_O3_wigner_d_is_the_rotation_matrix_to_l8():
    """A definition that shares nothing with the finite sum: d^l_{m',m}(beta) = <l m'| exp(-i beta J_y) |l m>, J_y from the ladder
    operators J+-|l m> = sqrt(l(l+1) - m(m+-1)) |l m+-1>, exponentiated by a library routine.  -2Y_lm = sqrt((2l+1)/4pi) d^l_{m,2}(theta)
    e^{i m phi} (reading R5) for EVERY (l, m), l = 2..8: a wrong factorial bound, sign or exponent in any term fails here."""
    import scipy.linalg as sl

    for l in range(2, 9):
        ms = list(range(l, -l - 1, -1))
        Jp = np.zeros((2 * l + 1, 2 * l + 1))
        for i, m in enumerate(ms):
            if m < l:
                Jp[i - 1, i] = np.sqrt(l * (l + 1) - m * (m + 1))
        Jy = (Jp - Jp.T) / 2j
        for th in (0.0, 0.3, 1.1, np.pi / 2, 2.9, np.pi):
            D = sl.expm(-1j * th * Jy)
            for i, m in enumerate(ms):
                ref = np.sqrt((2 * l + 1) / (4 * np.pi)) * D[i, ms.index(2)] * np.exp(1j * m * 0.7)
                assert abs(oracle.sYlm(l, m, th, 0.7) - ref) < 2e-14, (l, m, th)


def test_O3_pole_values_and_sum_rule():
    for l in range(2, 9):
        for m in range(-l, l + 1):
            v = oracle.sYlm(l, m, 0.0, 0.7)
            if m == 2:
                assert abs(v - np.sqrt((2 * l + 1) / (4 * np.pi)) * np.exp(2j * 0.7)) < 1e-14
            else:
                assert abs(v) < 1e-15
        for th in (0.3, 1.1, 2.9):
            tot = sum(abs(oracle.sYlm(l, m, th, 0.2)) ** 2 for m in range(-l, l + 1))
            assert abs(tot - (2 * l + 1) / (4 * np.pi)) < 1e-14


def test_O3_orthonormality_by_quadrature():
    mu, w = np.polynomial.legendre.leggauss(20)      # exact to degree 39 >= 16 = 2 ILE_MAX_L in cos(theta)
    n_phi = 24                                       # the trapezoid in phi is exact while |m - m'| <= 16 < n_phi
    modes = gi.modes_up_to(8)
    vals = np.zeros((len(modes), len(mu), n_phi), dtype=complex)
    for a, (l, m) in enumerate(modes):
        for i, x in enumerate(mu):
            for j in range(n_phi):
                vals[a, i, j] = oracle.sYlm(l, m, np.arccos(x), 2 * np.pi * j / n_phi)
    G = np.einsum("aij,bij,i->ab", np.conj(vals), vals, w) * (2 * np.pi / n_phi)
    assert np.max(np.abs(G - np.eye(len(modes)))) < 1e-13


# ----------------------------------------------------------------------------------------------------------
# O4 + O5: check (a) -- brute-force eq. 1 with eq. 2, 5, 6 and the response of L62 on a tiny circular grid
# ----------------------------------------------------------------------------------------------------------
def _tiny_problem(rng, n_t=9, zero_data=False):
    N, fs = 64, 4096.0
    dt = 1.0 / fs
    modes = [(2, 2), (2, -2), (2, 1), (2, 0)]
    K, M = 2, len(modes)
    f = np.fft.fftfreq(N, dt)
    band = (np.abs(f) > 100.0) & (np.abs(f) < 1900.0)                    # f_min < |f| < f_max  (eq. 2)
    neg = (-np.arange(N)) % N
    S = []
    for _ in range(K):
        s = rng.uniform(0.5, 2.0, N)
        S.append(0.5 * (s + s[neg]))                                      # S(|f|)
    h = rng.standard_normal((M, N)) + 1j * rng.standard_normal((M, N))    # generic complex modes h_lm(t)
    d = np.zeros((K, N)) if zero_data else rng.standard_normal((K, N))    # real detector data

    def inner(a, b, k):                                                    # eq. 2, two-sided, discretised
        A, B = np.fft.fft(a) * dt, np.fft.fft(b) * dt
        return 2.0 * np.sum((np.conj(A) * B / S[k])[band]) / (N * dt)

    arms = [random_orthonormal_arms(rng) for _ in range(K)]
    verts = [1.2e6 * random_unit(rng) for _ in range(K)]                   # ~4 ms light time: shifts of +-16 samples
    # eq. 8a-c: Q[i] = <h_lm(. - tau_i) | d>, tau_i = i dt (t0_Q = 0); U = <h_lm|h_l'm'>; V = <h_lm^*|h_l'm'>
    Q = np.zeros((K, M, N), dtype=complex)
    U = np.zeros((K, M, M), dtype=complex)
    V = np.zeros((K, M, M), dtype=complex)
    for k in range(K):
        for a in range(M):
            for i in range(N):
                Q[k, a, i] = inner(np.roll(h[a], i), d[k].astype(complex), k)
            for b in range(M):
                U[k, a, b] = inner(h[a], h[b], k)
                V[k, a, b] = inner(np.conj(h[a]), h[b], k)
    cfg = dict(Q=Q[None], U=U[None], V=V[None], l=np.array([lm[0] for lm in modes], dtype=np.int32),
               m=np.array([lm[1] for lm in modes], dtype=np.int32), n_det=K, n_modes=M, n_q=N, n_t=n_t, fs_hz=fs,
               t0_q_s=0.0, gmst_rad=0.9, d_ref_mpc=100.0, vertex_m=np.array(verts), arm_x=np.array([a[0] for a in arms]),
               arm_y=np.array([a[1] for a in arms]))
    return cfg, dict(h=h, d=d, inner=inner, modes=modes, N=N, dt=dt)


def _brute_lnL(cfg, aux, smp):
    """eq. 1 (reading R3) evaluated literally: build h_k(t) for each candidate time, take inner products."""
    K, n_t, N, dt = cfg["n_det"], cfg["n_t"], aux["N"], aux["dt"]
    a = cfg["d_ref_mpc"] / smp["dist_mpc"]
    hc = np.zeros(N, dtype=complex)                                        # eq. 5-6: h = h+ - i hx = a sum Y_lm h_lm
    for j, (l, m) in enumerate(aux["modes"]):
        hc = hc + a * Y2m_closed(m, smp["incl"], -smp["phi_ref"]) * aux["h"][j]
    hplus, hcross = hc.real, -hc.imag
    out = np.zeros(n_t)
    idx = np.zeros(K, dtype=np.int64)
    for k in range(K):
        s = source_dir(smp["ra"], smp["dec"], cfg["gmst_rad"])
        dtk = -np.dot(cfg["vertex_m"][k], s) / C_SI                        # nearer the source -> earlier
        idx[k] = int(np.rint((smp["t_ref"] + dtk - cfg["t0_q_s"]) * cfg["fs_hz"])) - n_t // 2
    for j in range(n_t):
        tot = 0.0
        for k in range(K):
            fp, fc = antenna_vec(cfg["arm_x"][k], cfg["arm_y"][k], smp["ra"], smp["dec"], smp["psi"], cfg["gmst_rad"])
            n_shift = idx[k] + j                                           # arrival time in samples (nearest sample, R8)
            hk = fp * np.roll(hplus, n_shift) + fc * np.roll(hcross, n_shift)          # L62
            dk = aux["d"][k]
            r = (hk - dk).astype(complex)
            tot += -0.5 * (aux["inner"](r, r, k) - aux["inner"](dk.astype(complex), dk.astype(complex), k)).real
        out[j] = tot
    return out, idx


def _random_sample(rng, t_center):
    return dict(ra=rng.uniform(0, 2 * np.pi), dec=np.arcsin(rng.uniform(-1, 1)), psi=rng.uniform(0, np.pi),
                phi_ref=rng.uniform(0, 2 * np.pi), incl=np.arccos(rng.uniform(-1, 1)), dist_mpc=rng.uniform(50, 400),
                t_ref=t_center + rng.uniform(-3, 3) / 4096.0)


def test_check_a_bruteforce_eq1_equals_factored_eq7():
    rng = np.random.default_rng(7)
    cfg, aux = _tiny_problem(rng)
    for _ in range(12):
        smp = _random_sample(rng, 32 / 4096.0)
        brute, idx = _brute_lnL(cfg, aux, smp)
        series, val, oidx, oob = oracle.sample_series(cfg, smp)
        assert not oob
        assert np.array_equal(idx, oidx.astype(np.int64))
        scale = np.max(np.abs(brute))
        assert np.max(np.abs(series - brute)) < 1e-11 * scale
        # eq. 9 on top of it: direct summation
        direct = math.log(math.fsum(math.exp(x) for x in brute) / cfg["n_t"])
        assert abs(val - direct) < 1e-10 * max(1.0, abs(direct))


def test_check_b_zero_data_gives_minus_half_rho2():
    """d = 0 (hence Q = 0): lnL_j = -1/2 sum_k <h_k|h_k> for every j, so lnL_margT equals the same constant."""
    rng = np.random.default_rng(11)
    cfg, aux = _tiny_problem(rng, zero_data=True)
    assert np.all(cfg["Q"] == 0)
    for _ in range(6):
        smp = _random_sample(rng, 32 / 4096.0)
        brute, _ = _brute_lnL(cfg, aux, smp)            # = -rho^2/2 from eq. 1, bin-independent up to rounding
        series, val, _, _ = oracle.sample_series(cfg, smp)
        rho2_half = -brute[0]
        assert rho2_half > 0
        assert np.max(np.abs(brute + rho2_half)) < 1e-10 * rho2_half
        assert np.max(np.abs(series + rho2_half)) < 1e-11 * rho2_half
        assert abs(val + rho2_half) < 1e-11 * rho2_half


def test_O4_single_mode_closed_form():
    """One detector, one (2,2) mode, V = 0: quad = (a^2/4) |F|^2 |Y22|^2 U with textbook |F|^2 and |Y22|."""
    ax, ay = np.array([1.0, 0, 0]), np.array([0, 1.0, 0])
    th, ph, psi, incl, a, u = 0.8, 2.1, 0.4, 1.0, 0.37, 123.0
    F = oracle.antenna(ax, ay, 0.0, ph, 0.5 * np.pi - th, psi)
    F2 = (0.5 * (1 + np.cos(th) ** 2) * np.cos(2 * ph)) ** 2 + (np.cos(th) * np.sin(2 * ph)) ** 2
    Y = Y2m_closed(2, incl, -0.3)
    q = oracle.quad([F], [Y], np.array([[[u]]], dtype=complex), np.zeros((1, 1, 1), dtype=complex), a)
    assert abs(q - 0.25 * a * a * F2 * (5.0 / (64 * np.pi)) * (1 + np.cos(incl)) ** 4 * u) < 1e-13 * q


def test_O4_O5_distance_scan_and_linearity():
    """lnL_j(a) = a L1 - a^2 L2: linear term scales with 1/D, quadratic with 1/D^2; lnL is linear in Q (eq. 7)."""
    cfg = gi.make_config(0, n=4)
    s = gi.make_samples(1, 1)
    smp = {k: float(v[0]) for k, v in s.items()}
    smp["t_ref"] = 0.001
    ser = {}
    for D in (100.0, 200.0, 400.0):
        smp["dist_mpc"] = D
        ser[D], _, _, _ = oracle.sample_series(cfg, smp)
    # a = 1, 1/2, 1/4: solve for L1, L2 from two distances, predict the third
    L2 = 4.0 * ser[200.0] - 2.0 * ser[100.0]          # s(1) = L1 - L2, s(1/2) = L1/2 - L2/4
    L1 = ser[100.0] + L2
    pred = 0.25 * L1 - 0.0625 * L2
    assert np.max(np.abs(pred - ser[400.0])) < 1e-10 * np.max(np.abs(ser[400.0]))
    assert np.ptp(L2) < 1e-9 * abs(L2[0]) and L2[0] > 0                 # the quadratic term is time-independent and positive
    cfg2 = dict(cfg)
    cfg2["Q"] = 3.0 * cfg["Q"]
    smp["dist_mpc"] = 100.0
    ser3, _, _, _ = oracle.sample_series(cfg2, smp)
    assert np.max(np.abs((ser3 + L2) - 3.0 * L1)) < 1e-10 * np.max(np.abs(L1))


# ----------------------------------------------------------------------------------------------------------
# check (c): face-on, single (2,2) mode, one detector, V = 0
# ----------------------------------------------------------------------------------------------------------
def test_check_c_face_on_single_mode_optimum():
    rng = np.random.default_rng(3)
    n_q, n_t = 32, 1
    qv = rng.standard_normal(n_q) + 1j * rng.standard_normal(n_q)
    u = 40.0
    ax, ay = random_orthonormal_arms(rng)
    cfg = dict(Q=qv.reshape(1, 1, 1, n_q), U=np.array([[[[u]]]], dtype=complex), V=np.zeros((1, 1, 1, 1), dtype=complex),
               l=np.array([2], dtype=np.int32), m=np.array([2], dtype=np.int32), n_det=1, n_modes=1, n_q=n_q, n_t=n_t,
               fs_hz=4096.0, t0_q_s=0.0, gmst_rad=0.2, d_ref_mpc=100.0, vertex_m=np.zeros((1, 3)),
               arm_x=ax[None], arm_y=ay[None])
    ra, dec = 1.0, 0.3
    i_bin = 17
    base = dict(ra=ra, dec=dec, t_ref=i_bin / 4096.0, incl=0.0, dist_mpc=100.0)
    # degeneracy: at iota = 0, F Y22 ~ e^{-2i(psi + phi_ref)}: lnL constant along psi + phi_ref = const
    v0 = oracle.sample_series(cfg, dict(base, psi=0.3, phi_ref=1.1))[1]
    v1 = oracle.sample_series(cfg, dict(base, psi=0.8, phi_ref=0.6))[1]
    assert abs(v0 - v1) < 1e-12 * max(1.0, abs(v0))
    # analytic optimum over (distance, phase): max lnL = |Q|^2 / U at a* = 2|Q| / (|F||Y22| U), Y22(0) = sqrt(5/4pi)
    fp, fc = antenna_vec(ax, ay, ra, dec, 0.0, cfg["gmst_rad"])
    Fabs, Yabs, Qabs = math.hypot(fp, fc), math.sqrt(5.0 / (4.0 * math.pi)), abs(qv[i_bin])
    a_star = 2.0 * Qabs / (Fabs * Yabs * u)
    best = -np.inf
    phases = np.linspace(0.0, np.pi, 4001)
    for p in phases:
        best = max(best, oracle.sample_series(cfg, dict(base, psi=p, phi_ref=0.0, dist_mpc=100.0 / a_star))[1])
    assert abs(best - Qabs ** 2 / u) < 1e-6 * Qabs ** 2 / u       # grid in phase: quadratic miss ~ (dphi)^2
    for eps in (0.9, 1.1):                                            # a* is the maximum in distance
        assert oracle.sample_series(cfg, dict(base, psi=phases[0], phi_ref=0.0, dist_mpc=100.0 / (a_star * eps)))[1] < best
    # the optimal phase is where conj(F Y) Q is real positive: check the closed form value there
    F0 = complex(fp, fc)
    arg = np.angle(np.conj(F0 * Yabs) * qv[i_bin])                   # need e^{+2i(psi+phi)} e^{i arg} = 1
    psi_opt = (-0.5 * arg) % np.pi
    v = oracle.sample_series(cfg, dict(base, psi=psi_opt, phi_ref=0.0, dist_mpc=100.0 / a_star))[1]
    assert abs(v - Qabs ** 2 / u) < 1e-12 * Qabs ** 2 / u


# ----------------------------------------------------------------------------------------------------------
# check (d): psi -> psi + pi
# ----------------------------------------------------------------------------------------------------------
def test_noise_free_injection_peaks_at_half_rho_squared():
    """SURVEY.md §8(c) pin: data = the noise-free signal of a known extrinsic point theta_0, built by the input
    generator from response numbers computed HERE by independent means (vector-algebra antenna pattern, textbook l = 2
    harmonics, geometric delay), gives oracle lnL(theta_0, t_0) = <h|d> - <h|h>/2 = +rho^2/2 with rho = the SNR the
    generator scaled the signal to -- and theta_0 is a maximum: every neighbouring point and every other time bin
    gives less.  A wrong sign of F (R1), of the delay (R2), of the Y_lm phase (R4), a dropped V term or a factor in the
    quadratic term (eq. 7) fails this."""
    base = gi.make_config(1, n=1)
    dets, modes = base["dets"], base["modes"]
    rng = np.random.default_rng(99)
    snr = 17.0
    for trial in range(4):
        th = dict(ra=rng.uniform(0, 2 * np.pi), dec=np.arcsin(rng.uniform(-1, 1)), psi=rng.uniform(0, np.pi),
                  phi_ref=rng.uniform(0, 2 * np.pi), incl=np.arccos(rng.uniform(-1, 1)), dist_mpc=gi.D_TRUE_MPC, t_ref=0.0)
        resp, tau = [], []
        for k in range(len(dets)):
            fp, fc = antenna_vec(base["arm_x"][k], base["arm_y"][k], th["ra"], th["dec"], th["psi"], base["gmst_rad"])
            resp.append(complex(fp, fc))                                       # R1: F = F+ + i Fx
            dt = -float(np.dot(base["vertex_m"][k], source_dir(th["ra"], th["dec"], base["gmst_rad"]))) / C_SI   # R2
            tau.append(int(np.rint(dt * base["fs_hz"])))
        y = np.array([Y2m_closed(m, th["incl"], -th["phi_ref"]) for (_, m) in modes])      # R4: Y_lm(iota, -phi_ref)
        Q, U, V, meta = gi.make_point(1234 + trial, dets, modes, base["n_q"], snr, noise=False,
                                      truth_response=dict(y=y, resp=np.array(resp), tau_samples=np.array(tau)))
        cfg = dict(base)
        cfg.update(Q=Q[None], U=U[None], V=V[None], n_points=1)
        series, margT, idx, oob = oracle.sample_series(cfg, th)
        assert not oob
        j0 = cfg["n_t"] // 2                                                   # the bin of t = t_ref
        assert np.array_equal(idx + j0, np.array(tau) + cfg["n_q"] // 2)
        assert abs(series[j0] - 0.5 * snr ** 2) <= 1e-9 * snr ** 2
        assert np.argmax(series) == j0
        for key, step in (("ra", 0.02), ("dec", 0.02), ("psi", 0.05), ("phi_ref", 0.05), ("incl", 0.05), ("dist_mpc", 10.0)):
            for sgn in (-1.0, 1.0):
                th2 = dict(th)
                th2[key] = th[key] + sgn * step
                if key == "dec" and abs(th2["dec"]) > 0.5 * np.pi:
                    continue
                assert oracle.sample_series(cfg, th2)[0].max() < series[j0]


def test_check_d_psi_plus_pi_invariance():
    cfg = gi.make_config(0, n=64)
    s = gi.make_samples(5, 64)
    out0, idx0, _ = oracle.eval_batch(cfg, s)
    s2 = dict(s)
    s2["psi"] = s["psi"] + np.pi
    out1, idx1, _ = oracle.eval_batch(cfg, s2)
    assert np.array_equal(idx0, idx1)
    assert np.max(np.abs(out0 - out1) / np.maximum(1.0, np.abs(out0))) < 1e-12


# ----------------------------------------------------------------------------------------------------------
# O6 / check (e): time marginalisation = direct summation (eq. 9)
# ----------------------------------------------------------------------------------------------------------
def test_check_e_margT_direct_summation():
    rng = np.random.default_rng(5)
    for n in (1, 2, 201, 410):
        x = rng.uniform(-8.0, 8.0, n)
        direct = math.log(math.fsum(math.exp(v) for v in x) / n)
        assert abs(oracle.margT(x) - direct) < 1e-13 * max(1.0, abs(direct))
    assert abs(oracle.margT(np.full(410, -3.25)) + 3.25) < 1e-14                  # constant in, constant out
    x = rng.uniform(-5, 5, 201)
    assert abs(oracle.margT(x + 1000.0) - (oracle.margT(x) + 1000.0)) < 1e-12     # shift equivariance, no overflow
    spike = np.full(410, -1.0e4)
    spike[123] = 55.5
    assert abs(oracle.margT(spike) - (55.5 - math.log(410))) < 1e-13              # one dominant bin
    assert oracle.margT(np.full(7, -np.inf)) == -np.inf


# ----------------------------------------------------------------------------------------------------------
# O7, O8 evidence and n_eff
# ----------------------------------------------------------------------------------------------------------
def test_O7_O8_direct_summation_and_invariances():
    rng = np.random.default_rng(9)
    x = rng.uniform(-20, 20, 1000)
    lw = rng.standard_normal(1000)
    for w in (None, lw):
        e = x if w is None else x + w
        lnZ, neff = oracle.evidence(x, w)
        tot = math.fsum(math.exp(v) for v in e)
        assert abs(lnZ - math.log(tot / len(e))) < 1e-13 * abs(math.log(tot / len(e)))
        assert abs(neff - tot / math.exp(np.max(e))) < 1e-12 * neff
        perm = rng.permutation(len(e))
        lnZ2, neff2 = oracle.evidence(x[perm], None if w is None else w[perm])
        assert abs(lnZ2 - lnZ) < 1e-12 and abs(neff2 - neff) < 1e-10
    lnZ, neff = oracle.evidence(np.full(50, 2.5))
    assert abs(lnZ - 2.5) < 1e-14 and abs(neff - 50.0) < 1e-12                     # all equal: n_eff = n
    lnZ, neff = oracle.evidence(np.array([0.0, -np.inf, -np.inf, -np.inf]))
    assert abs(lnZ + math.log(4.0)) < 1e-15 and neff == 1.0                        # -inf samples count in n, add nothing


# ----------------------------------------------------------------------------------------------------------
# R9: a window that leaves the stored Q
# ----------------------------------------------------------------------------------------------------------
def test_R9_out_of_range_window_flags_and_minus_inf():
    cfg = gi.make_config(0, n=4)
    s = gi.make_samples(2, 4)
    s["t_ref"] = np.array([0.0, 0.2, -0.2, 0.01])
    out, idx, bad = oracle.eval_batch(cfg, s)
    assert bad == 2
    assert np.isfinite(out[0]) and np.isfinite(out[3]) and out[1] == -np.inf and out[2] == -np.inf
    lnZ, _ = oracle.evidence(out)
    assert np.isfinite(lnZ)


def test_batch_equals_single_and_threads():
    cfg = gi.make_config(0, n=32)
    s = gi.make_samples(cfg["sample_seeds"][0], 32)
    out1, idx1, _ = oracle.eval_batch(cfg, s, n_threads=1)
    out4, idx4, _ = oracle.eval_batch(cfg, s, n_threads=4)
    assert np.array_equal(out1, out4) and np.array_equal(idx1, idx4)
    for a in (0, 7, 31):
        _, v, i, _ = oracle.sample_series(cfg, {k: float(x[a]) for k, x in s.items()})
        assert v == out1[a] and np.array_equal(i, idx1[a])
