"""Seeded synthetic inputs for the ILE hot path.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_1902_04934_b200/`).  It holds none of the hot path's arithmetic: no antenna
pattern, no arrival-time delay, no spherical harmonic, no likelihood, no log-sum-exp.
It manufactures the *inputs* of the hot path -- the mode overlap time series
Q_{k,lm}(t), the mode-mode matrices U_k, V_k (eq. 8a-c), the
detector constants and the extrinsic sample arrays -- with the
shapes, sizes and value distributions of the paper's workloads
and of BASELINE.json's five configs.  The paper's own inputs come from lalsuite
waveforms and LIGO PSDs, neither of which exists here; these stand in for them.

Since the overlap pre-computation itself became a product entry (`ile_precompute`,
SURVEY.md §8(f) NEXT-1), note what that means here: `make_point` builds Q, U, V from
the whitened spectra with numpy (matrix products and one inverse FFT) because the hot
path needs inputs whether or not NEXT-1 exists.  For NEXT-1 only the spectra
(`spectra=True`: meta["x"], meta["d"]) are the shared inputs; the expected Q, U, V of
its parity tests come from `oracle/precompute.py`, never from this module, and the
test that compares this module's Q, U, V with the oracle's is a consistency check of
the generator, not a pin of the oracle (its pins are in tests/test_oracle_precompute_pins.py).

The "true signal" injected into the data is described by seeded random response
numbers (one complex amplitude per detector, one complex weight per mode, one integer
delay per detector), NOT computed from a sky position, so no response formula lives here.
A caller that wants a signal at an exact extrinsic point passes `truth_response`.
"""
from __future__ import annotations

import numpy as np

FS_HZ = 4096.0                  # 4096 Hz analyses
D_REF_MPC = 100.0               # BASELINE.json configs[0]: D_ref = 100 Mpc
D_TRUE_MPC = 200.0              # BBH source at 200 Mpc
GMST_RAD = 0.336877343721285    # GMST at GPS 1000000000 (an input; one value per event)
F_LOW_HZ, F_HIGH_HZ = 20.0, 1024.0
SEED_BASE = 190204934 * 10

# Earth-fixed vertex (m) and unit arm directions.  Inputs, parity-neutral.
DETECTORS = {
    "H1": dict(vertex_m=(-2.16141492636e6, -3.83469517889e6, 4.60035022664e6),
               arm_x=(-0.22389266154, 0.79983062746, 0.55690487831),
               arm_y=(-0.91397818574, 0.02609403989, -0.40492342125), psd_scale=1.0),
    "L1": dict(vertex_m=(-7.42760447238e4, -5.49628371971e6, 3.22425701744e6),
               arm_x=(-0.95457412153, -0.14158077340, -0.26218911324),
               arm_y=(0.29774156894, -0.48791033647, -0.82054461286), psd_scale=0.8),
    "V1": dict(vertex_m=(4.54637409900e6, 8.42989697626e5, 4.37857696241e6),
               arm_x=(-0.70045821479, 0.20848948619, 0.68256166277),
               arm_y=(-0.05379255368, -0.96908180549, 0.24080451708), psd_scale=2.5),
}


def _site(lat_deg: float, lon_deg: float, x_arm_azimuth_deg: float, psd_scale: float):
    """A site on a spherical Earth (R = 6.371e6 m) with orthogonal horizontal arms, the x arm at the given azimuth east of north."""
    lat, lon, az = np.radians(lat_deg), np.radians(lon_deg), np.radians(x_arm_azimuth_deg)
    up = np.array([np.cos(lat) * np.cos(lon), np.cos(lat) * np.sin(lon), np.sin(lat)])
    east = np.array([-np.sin(lon), np.cos(lon), 0.0])
    north = np.cross(up, east)
    ax = np.cos(az) * north + np.sin(az) * east
    ay = np.cos(az + 0.5 * np.pi) * north + np.sin(az + 0.5 * np.pi) * east
    return dict(vertex_m=tuple(6.371e6 * up), arm_x=tuple(ax), arm_y=tuple(ay), psd_scale=psd_scale)


# A fourth site for four-detector networks (PAPER.md L79 treats F as (detectors) x (extrinsic) without a limit of three): a
# detector at KAGRA's approximate geodetic position.  An input like the others, parity-neutral.
DETECTORS["K1"] = _site(36.41, 137.31, 60.4, 3.0)


def modes_up_to(l_max: int, l_min: int = 2):
    """All (l, m) with l_min <= l <= l_max, m = -l..l, in that order."""
    return [(l, m) for l in range(l_min, l_max + 1) for m in range(-l, l + 1)]


# BASELINE.json "configs" -> sizes.  `n` is samples per intrinsic point.
CONFIGS = {
    0: dict(dets=("H1", "L1"), modes=[(2, -2), (2, 2)], n_q=1024, n_t=201, n=1_000, n_points=1,
            snr=15.0, admix=0.0),
    1: dict(dets=("H1", "L1", "V1"), modes=modes_up_to(2), n_q=2048, n_t=410, n=100_000, n_points=1,
            snr=20.0, admix=0.0),
    2: dict(dets=("H1", "L1", "V1"), modes=modes_up_to(4), n_q=4096, n_t=410, n=1_000_000, n_points=1,
            snr=20.0, admix=0.1),
    3: dict(dets=("H1", "L1", "V1"), modes=modes_up_to(2), n_q=2048, n_t=410, n=10_000_000, n_points=1,
            snr=20.0, admix=0.0, sweep=(1_000, 10_000, 100_000, 1_000_000, 10_000_000)),
    4: dict(dets=("H1", "L1", "V1"), modes=modes_up_to(2), n_q=2048, n_t=410, n=100_000, n_points=256,
            snr=(8.0, 40.0), admix=0.0),
    # the paper's own window and rates (not BASELINE.json configs): T = 0.3 s, two
    # detectors (L109), modes (2,+-2) or (2,+-2),(2,+-1) (Tables I/II, L143-L159), at 4096 Hz and at the legacy 16384 Hz (L121)
    5: dict(dets=("H1", "L1"), modes=[(2, -2), (2, 2)], n_q=8192, n_t=1229, n=100_000, n_points=1, snr=20.0, admix=0.0,
            fs_hz=4096.0),
    6: dict(dets=("H1", "L1"), modes=[(2, -2), (2, -1), (2, 1), (2, 2)], n_q=8192, n_t=1229, n=100_000, n_points=1, snr=20.0,
            admix=0.0, fs_hz=4096.0),
    7: dict(dets=("H1", "L1"), modes=[(2, -2), (2, 2)], n_q=32768, n_t=4915, n=100_000, n_points=1, snr=20.0, admix=0.0,
            fs_hz=16384.0),
    8: dict(dets=("H1", "L1"), modes=[(2, -2), (2, -1), (2, 1), (2, 2)], n_q=32768, n_t=4915, n=100_000, n_points=1, snr=20.0,
            admix=0.0, fs_hz=16384.0),
}

SAMPLE_FIELDS = ("ra", "dec", "t_ref", "phi_ref", "psi", "incl", "dist_mpc")


def point_seed(config_id: int, point: int = 0) -> int:
    """PCG64(190204934*10 + config); config 4's point p adds 1000*(p+1)."""
    s = SEED_BASE + config_id
    if CONFIGS[config_id]["n_points"] > 1:
        s += 1000 * (point + 1)
    return s


def detector_arrays(dets):
    """(vertex_m, arm_x, arm_y), each float64 [K][3]."""
    v = np.array([DETECTORS[d]["vertex_m"] for d in dets], dtype=np.float64)
    ax = np.array([DETECTORS[d]["arm_x"] for d in dets], dtype=np.float64)
    ay = np.array([DETECTORS[d]["arm_y"] for d in dets], dtype=np.float64)
    return v, ax, ay


def make_point(seed: int, dets, modes, n_q: int, snr: float, *, fs_hz: float = FS_HZ,
               admix: float = 0.0, truth_response=None, noise: bool = True, spectra: bool = False):
    """One intrinsic point: Q [K][M][n_q], U [K][M][M], V [K][M][M] (complex128, C order) + metadata.

    Frequency-domain recipe.  With the whitened mode spectra
    x_{k,lm}(f) as columns of X_k and the discrete two-sided inner product
    <a|b> = sum_f conj(a_w(f)) b_w(f):
        U_k = X_k^H X_k,  V_k = X_k^T P X_k  (P: f -> -f),  Q_{k,lm}[i] = <h_lm(. - tau_i) | d_k>
    so the three are mutually consistent in the sense of PAPER.md eq. 8a-c.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    K, M = len(dets), len(modes)
    dt = 1.0 / fs_hz
    f = np.fft.fftfreq(n_q, dt)
    af = np.abs(f)
    band = (af > F_LOW_HZ) & (af < F_HIGH_HZ)
    afs = np.where(band, af, 1.0)               # avoid 0**negative outside the band
    neg = (-np.arange(n_q)) % n_q                # index of -f

    # per-mode amplitude, chirp phase coefficient (mode properties, shared by all detectors)
    c_lm = np.array([1.0 if (l == 2 and abs(m) == 2) else rng.uniform(0.05, 0.3) for (l, m) in modes])
    beta = np.array([40.0 * abs(m) / 2.0 + rng.uniform(0.0, 5.0) for (l, m) in modes])
    mix = np.eye(M, dtype=np.complex128)
    if admix > 0.0:
        ph = np.exp(2j * np.pi * rng.random((M, M)))
        for a in range(M - 1):                   # neighbouring modes only
            mix[a, a + 1] = admix * ph[a, a + 1]
            mix[a + 1, a] = admix * ph[a + 1, a]

    X = np.zeros((K, n_q, M), dtype=np.complex128)
    for k, d in enumerate(dets):
        S = DETECTORS[d]["psd_scale"] * ((40.0 / afs) ** 4 + 1.0 + (afs / 300.0) ** 2)
        for j, (l, m) in enumerate(modes):
            if m > 0:
                supp = (f < 0).astype(np.float64)
            elif m < 0:
                supp = (f > 0).astype(np.float64)
            else:
                supp = np.full(n_q, 0.3)
            amp = band * supp * c_lm[j] * (afs / 100.0) ** (-7.0 / 6.0) / np.sqrt(S)
            X[k, :, j] = amp * np.exp(1j * np.sign(f) * beta[j] * (afs / 100.0) ** (-5.0 / 3.0))
        X[k] = X[k] @ mix

    # the injected signal's response numbers (seeded; see module docstring)
    if truth_response is None:
        y = rng.standard_normal(M) + 1j * rng.standard_normal(M)
        y *= np.sqrt(5.0 / (4.0 * np.pi)) / np.linalg.norm(y)
        resp = 0.7 * np.sqrt(rng.random(K)) * np.exp(2j * np.pi * rng.random(K))
        tau = rng.integers(-60, 61, size=K)
    else:
        y = np.asarray(truth_response["y"], dtype=np.complex128)
        resp = np.asarray(truth_response["resp"], dtype=np.complex128)
        tau = np.asarray(truth_response["tau_samples"], dtype=np.int64)
    a0 = D_REF_MPC / D_TRUE_MPC

    def signal(Xk, k):
        hw = Xk @ y
        s = 0.5 * a0 * (resp[k] * hw + np.conj(resp[k]) * np.conj(hw[neg]))
        return s * np.exp(-2j * np.pi * f * (tau[k] * dt))

    rho2 = sum(float(np.sum(np.abs(signal(X[k], k)) ** 2)) for k in range(K))
    X *= snr / np.sqrt(rho2)

    t0_q_s = -n_q / (2.0 * fs_hz)
    Q = np.empty((K, M, n_q), dtype=np.complex128)
    U = np.empty((K, M, M), dtype=np.complex128)
    V = np.empty((K, M, M), dtype=np.complex128)
    D = np.empty((K, n_q), dtype=np.complex128)
    for k in range(K):
        d = signal(X[k], k)
        if noise:
            d = d + np.fft.fft(rng.standard_normal(n_q)) / np.sqrt(n_q)
        D[k] = d
        U[k] = X[k].conj().T @ X[k]
        V[k] = X[k].T @ X[k][neg]
        spec = np.conj(X[k]) * (d * np.exp(2j * np.pi * f * t0_q_s))[:, None]       # [n_q][M]
        Q[k] = (np.fft.ifft(spec, axis=0) * n_q).T
    meta = dict(seed=seed, snr=float(snr), t0_q_s=t0_q_s, fs_hz=fs_hz, truth=dict(y=y, resp=resp, tau_samples=tau, a0=a0))
    if spectra:  # inputs of the overlap pre-computation (eq. 8): whitened mode spectra [K][M][n_q] and data [K][n_q], FFT order
        meta["x"] = np.ascontiguousarray(np.transpose(X, (0, 2, 1)))
        meta["d"] = np.ascontiguousarray(D)
    return np.ascontiguousarray(Q), np.ascontiguousarray(U), np.ascontiguousarray(V), meta


def make_samples(seed: int, n: int):
    """Extrinsic samples drawn from the prior: dict of float64 [n]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    s = {}
    s["ra"] = 2.0 * np.pi * rng.random(n)
    s["dec"] = np.arcsin(2.0 * rng.random(n) - 1.0)
    s["psi"] = np.pi * rng.random(n)
    s["phi_ref"] = 2.0 * np.pi * rng.random(n)
    s["incl"] = np.arccos(2.0 * rng.random(n) - 1.0)
    s["dist_mpc"] = np.cbrt(1.0 + rng.random(n) * (1000.0 ** 3 - 1.0))
    s["t_ref"] = 0.1 * rng.random(n) - 0.05
    return {k: np.ascontiguousarray(s[k]) for k in SAMPLE_FIELDS}


def make_concentrated_samples(seed: int, n: int, width: float = 0.05):
    """Samples in a Gaussian ball around one seeded extrinsic point with t_ref ~ 0: the shape of what an
    adaptive sampler feeds the likelihood late in a run.  Same cost as prior draws."""
    rng = np.random.Generator(np.random.PCG64(seed))
    c = make_samples(seed + 17, 1)
    s = {}
    s["ra"] = np.mod(c["ra"][0] + width * rng.standard_normal(n), 2.0 * np.pi)
    s["dec"] = np.clip(c["dec"][0] + width * rng.standard_normal(n), -0.5 * np.pi, 0.5 * np.pi)
    s["psi"] = np.mod(c["psi"][0] + width * rng.standard_normal(n), np.pi)
    s["phi_ref"] = np.mod(c["phi_ref"][0] + width * rng.standard_normal(n), 2.0 * np.pi)
    s["incl"] = np.clip(c["incl"][0] + width * rng.standard_normal(n), 0.0, np.pi)
    s["dist_mpc"] = D_TRUE_MPC * np.exp(width * rng.standard_normal(n))
    s["t_ref"] = 2.0e-4 * rng.standard_normal(n)
    return {k: np.ascontiguousarray(s[k]) for k in SAMPLE_FIELDS}


def make_log_weights(seed: int, n: int):
    """ln w ~ N(0,1), for the weighted-evidence case.  Configs themselves use ln w = 0."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.standard_normal(n)


def make_config(config_id: int, *, n: int | None = None, n_points: int | None = None):
    """Everything `ile_create` needs for one BASELINE.json config, plus its samples' seeds.

    Returns a dict: Q [P][K][M][n_q], U, V [P][K][M][M], l, m (int32 [M]), n_det, n_modes, n_q, n_t,
    fs_hz, t0_q_s, gmst_rad, d_ref_mpc, vertex_m/arm_x/arm_y [K][3], n (samples per point), sample_seeds [P].
    `n` / `n_points` override the config's sizes (tests use reduced sizes; the recipe is unchanged).
    """
    c = CONFIGS[config_id]
    P = c["n_points"] if n_points is None else n_points
    Qs, Us, Vs, metas, sseeds = [], [], [], [], []
    for p in range(P):
        seed = point_seed(config_id, p)
        if isinstance(c["snr"], tuple):
            lo, hi = c["snr"]
            snr = float(np.random.Generator(np.random.PCG64(seed + 250)).uniform(lo, hi))
        else:
            snr = c["snr"]
        Q, U, V, meta = make_point(seed, c["dets"], c["modes"], c["n_q"], snr, admix=c["admix"], fs_hz=c.get("fs_hz", FS_HZ))
        Qs.append(Q), Us.append(U), Vs.append(V), metas.append(meta), sseeds.append(seed + 500)
    v, ax, ay = detector_arrays(c["dets"])
    return dict(
        config_id=config_id, dets=c["dets"], modes=list(c["modes"]),
        Q=np.ascontiguousarray(np.stack(Qs)), U=np.ascontiguousarray(np.stack(Us)), V=np.ascontiguousarray(np.stack(Vs)),
        l=np.array([lm[0] for lm in c["modes"]], dtype=np.int32), m=np.array([lm[1] for lm in c["modes"]], dtype=np.int32),
        n_points=P, n_det=len(c["dets"]), n_modes=len(c["modes"]), n_q=c["n_q"], n_t=c["n_t"],
        fs_hz=c.get("fs_hz", FS_HZ), t0_q_s=metas[0]["t0_q_s"], gmst_rad=GMST_RAD, d_ref_mpc=D_REF_MPC,
        vertex_m=v, arm_x=ax, arm_y=ay, n=c["n"] if n is None else n, sample_seeds=sseeds, meta=metas,
    )
