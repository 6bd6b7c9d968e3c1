"""Seeded synthetic workloads for the inspiral matched-filter hot path (test and bench inputs; not part of
the shipped library package).

This module is the ONLY code shared by the oracle tests and the CUDA tests/bench.
It produces *inputs* (a strain segment s(t), a one-sided PSD array S_n(f_k), a list
of mass pairs) and nothing else: it never forms a matched-filter output, a sigma
used by the filter, a band edge, an SNR or a chi^2.  It imports neither ``oracle/``
nor the CUDA binding.

Workload recipe (BASELINE.json:configs):
  * sampling 4096 Hz, low cut-off 40 Hz, segments of N = 2^14 .. 2^22 samples
    (256 s at 4096 Hz = 2^20 points);
  * noise: stationary coloured Gaussian noise whose one-sided PSD is PAPER.md Eq. 2
    (f0 = 150 Hz) -- the paper's own test data are "stationary coloured
    Gaussian noise with a spectrum matching the Initial LIGO SRD";
    Eq. 2 stands in for the SRD curve, which is not in the container;
  * injections: simulated inspiral chirps (2PN stationary-phase signal model,
    BASELINE.json:configs[0]) added in the frequency domain.  The signal simulator
    below is this module's own statement of the source model; the oracle and the
    CUDA path each carry their own, and neither calls this one;
  * banks: the (m1, m2) grids of SURVEY.md 8(d1).

Random numbers: a counter-based generator (SplitMix64 finaliser over
(seed, stream, index)) + Box-Muller, so that every value is a pure function of its
coordinates and does not depend on numpy's generator version.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

FS = 4096.0            # Hz
F_LOW = 40.0           # Hz
F0_PSD = 150.0         # Hz
T_SUN = 4.9254909476412675e-6   # G*Msun/c^3 in seconds

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)


# ----------------------------------------------------------------------------- RNG
def splitmix64(seed: int, stream: int, index) -> np.ndarray:
    """64-bit word = SplitMix64 finaliser of a linear mix of (seed, stream, index)."""
    idx = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (np.uint64(seed) * _GOLD) + (np.uint64(stream) * _C1) + (idx + np.uint64(1)) * _C2
        z = (z ^ (z >> np.uint64(30))) * _C1
        z = (z ^ (z >> np.uint64(27))) * _C2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, stream: int, index) -> np.ndarray:
    """Uniform in the open interval (0, 1) with 53 random bits."""
    w = splitmix64(seed, stream, index)
    return ((w >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed: int, stream: int, index) -> np.ndarray:
    """Standard normal: Box-Muller on the uniforms at counters 2*index, 2*index+1."""
    idx = np.asarray(index, dtype=np.uint64)
    u1 = uniform01(seed, stream, idx * np.uint64(2))
    u2 = uniform01(seed, stream, idx * np.uint64(2) + np.uint64(1))
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


# ----------------------------------------------------------------------------- PSD
def psd_eq2(f) -> np.ndarray:
    """Initial-LIGO one-sided PSD exactly as printed in PAPER.md:32 (Eq. 2), f0 = 150 Hz.

    Dimensionless (the 9e-46 scale of its source is not printed in the paper; SURVEY
    8(c2) reading 5).  Diverges at f -> 0: callers only use it at f >= 40 Hz; below
    10 Hz this returns +inf instead of overflowing.
    """
    f = np.asarray(f, dtype=np.float64)
    out = np.full(f.shape, np.inf)
    ok = f >= 10.0
    x = f[ok] / F0_PSD
    out[ok] = (4.49 * x) ** (-56.0) + 0.16 * x ** (-4.52) + 0.52 + 0.32 * x * x
    return out


def psd_array(n: int, fs: float = FS) -> np.ndarray:
    """S_n sampled at f_k = k*fs/n, k = 0..n/2 (the array handed to gwmf_load_segment)."""
    return psd_eq2(np.arange(n // 2 + 1, dtype=np.float64) * (fs / n))


# ----------------------------------------------------------------------------- noise
def noise_spectrum(n: int, seed: int, fs: float = FS, f_low: float = F_LOW) -> np.ndarray:
    """DFT-unit spectrum D[k], k = 0..n/2, of coloured Gaussian noise.

    <|n~(f_k)|^2> = S_n(f_k) / (2 df)  <=>  D[k] = 0.5*sqrt(n*fs*S_n(f_k)) * (a_k + i b_k),
    a, b ~ N(0,1) iid from streams 0 and 1, for k_low <= k < n/2; zero elsewhere
    (SURVEY.md 8(c2) reading 15; BASELINE.json:configs[0] "complex N(0,1) frequency bins
    scaled by sqrt(S_n(f)/2) ... zeroed below 40 Hz").
    """
    df = fs / n
    k_low = int(math.ceil(f_low / df))
    k = np.arange(k_low, n // 2, dtype=np.uint64)
    a = normal(seed, 0, k)
    b = normal(seed, 1, k)
    D = np.zeros(n // 2 + 1, dtype=np.complex128)
    D[k_low:n // 2] = 0.5 * np.sqrt(n * fs * psd_eq2(k.astype(np.float64) * df)) * (a + 1j * b)
    return D


# ----------------------------------------------------------------------------- signal simulator
def chirp_phase(m1: float, m2: float, f) -> np.ndarray:
    """Frequency-domain phase of a simulated inspiral with t_c = 0 (2PN, stationary phase).

    The formula is the one BASELINE.json:configs[0] prints; PAPER.md:21 only names the
    order ("second order post-Newtonian orbital phases").
    """
    f = np.asarray(f, dtype=np.float64)
    mt = (m1 + m2) * T_SUN
    eta = m1 * m2 / (m1 + m2) ** 2
    v = np.cbrt(np.pi * mt * f)
    series = (1.0
              + (3715.0 / 756.0 + 55.0 * eta / 9.0) * v ** 2
              - 16.0 * np.pi * v ** 3
              + (15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta * eta / 72.0) * v ** 4)
    return -np.pi / 4.0 + 3.0 / (128.0 * eta * v ** 5) * series


def chirp_f_cut(m1: float, m2: float, fs: float = FS) -> float:
    """min(f_ISCO, Nyquist)."""
    mt = (m1 + m2) * T_SUN
    return min(1.0 / (6.0 ** 1.5 * np.pi * mt), fs / 2.0)


def injection_spectrum(n: int, m1: float, m2: float, snr: float, j_c: int,
                       fs: float = FS, f_low: float = F_LOW) -> np.ndarray:
    """DFT-unit spectrum of a simulated chirp with optimal SNR `snr` coalescing at sample j_c.

    D[k] = fs * (A/sig) * f_k^(-7/6) * exp(-i[Psi(f_k) + 2 pi f_k t_c]) on 40 Hz <= f_k < f_cut
    (SURVEY.md 8(c2) reading 16), where sig^2 = 4 df sum f^(-7/3)/S_n over the same bins is
    the optimal SNR^2 of the unit-amplitude signal in Eq. 2 noise.  Built in the frequency
    domain, hence circular in time.
    """
    df = fs / n
    k_low = int(math.ceil(f_low / df))
    k_high = min(int(math.ceil(chirp_f_cut(m1, m2, fs) / df)), n // 2)
    D = np.zeros(n // 2 + 1, dtype=np.complex128)
    if k_high <= k_low:
        return D
    f = np.arange(k_low, k_high, dtype=np.float64) * df
    sn = psd_eq2(f)
    sig = math.sqrt(4.0 * df * float(np.sum(f ** (-7.0 / 3.0) / sn)))
    t_c = j_c / fs
    D[k_low:k_high] = fs * (snr / sig) * f ** (-7.0 / 6.0) * np.exp(
        -1j * (chirp_phase(m1, m2, f) + 2.0 * np.pi * f * t_c))
    return D


def time_series(D_half: np.ndarray, n: int) -> np.ndarray:
    """Real series whose ordinary forward DFT (e^{-2 pi i jk/n}) is the Hermitian extension of D."""
    return np.fft.irfft(D_half, n=n)


# ----------------------------------------------------------------------------- banks
def _pairs_ge(grid) -> list:
    """(m1 = g[a], m2 = g[b]) for a >= b, ordered by a then b."""
    return [(float(grid[a]), float(grid[b])) for a in range(len(grid)) for b in range(a + 1)]


def _bank_eta_mass(n_eta: int, n_m: int) -> list:
    """Grid uniform in eta and (at fixed eta) in total/chirp mass over M in [M_lo(eta), 34]."""
    eta_min = 33.0 / 1156.0                      # the (33, 1) system
    out = []
    for i in range(n_eta):
        eta = eta_min + (i + 1) * (0.25 - eta_min) / n_eta
        root = math.sqrt(max(0.0, 1.0 - 4.0 * eta))
        # M_lo(eta) <=> m2 = (M/2)(1 - root) = 1 Msun; equals 34 at eta_min, 2 at eta = 1/4
        m_lo = min(2.0 / (1.0 - root), 34.0)
        for j in range(n_m):
            mt = m_lo + j * (34.0 - m_lo) / (n_m - 1)
            out.append((0.5 * mt * (1.0 + root), 0.5 * mt * (1.0 - root)))
    return out


def bank(config: int) -> list:
    """Mass pairs of BASELINE.json:configs[config], enumerated as SURVEY.md 8(d1) proposes."""
    if config == 0:
        g = [6.0, 8.0, 10.0, 12.0]
        return [(g[a], g[b]) for a in range(4) for b in range(a, 4)][:8]
    if config == 1:
        return _pairs_ge([1.0 + 2.0 * g / 22.0 for g in range(23)])[:256]
    if config == 2:
        return _bank_eta_mass(32, 32)
    if config == 3:
        return _bank_eta_mass(64, 64)
    if config == 4:
        return _pairs_ge([1.0 + g / 31.0 for g in range(32)])[:512]
    raise ValueError(f"no such config: {config}")


# ----------------------------------------------------------------------------- configs
@dataclass
class Workload:
    config: int
    n: int
    p: int
    rho_thresh: float
    window: int
    masses: list
    seed: int
    injections: list = field(default_factory=list)   # (bank index, m1, m2, snr, j_c)
    fs: float = FS
    f_low: float = F_LOW
    n_segments: int = 1
    stream_len: int = 0

    @property
    def psd(self) -> np.ndarray:
        return psd_array(self.n, self.fs)


_SHAPES = {
    #  n      p   thresh window
    0: (1 << 14, 4, 6.0, 4096),
    1: (1 << 18, 16, 6.0, 4096),
    2: (1 << 20, 16, 6.0, 4096),
    3: (1 << 20, 16, 6.0, 4096),
    4: (1 << 22, 32, 5.5, 4096),
}
_N_INJ = {0: 1, 1: 3, 2: 10, 3: 16, 4: 4}


def workload(config: int, n_templates: int | None = None) -> Workload:
    """Parameters + injection list of a config (no arrays yet)."""
    n, p, thr, win = _SHAPES[config]
    masses = bank(config)
    if n_templates is not None:
        masses = masses[:n_templates]
    w = Workload(config=config, n=n, p=p, rho_thresh=thr, window=win, masses=masses, seed=config)
    full = bank(config)
    if config == 0:
        w.injections = [(4, 8.0, 8.0, 12.0, 9000)]
    else:
        length = n if config != 3 else (1 << 23)
        for q in range(_N_INJ[config]):
            u = uniform01(config, 2, np.arange(3 * q, 3 * q + 3))
            b = int(u[0] * len(full))
            w.injections.append((b, full[b][0], full[b][1], 8.0 + 7.0 * float(u[1]), int(u[2] * length)))
    if config == 3:
        w.n_segments = 15
        w.stream_len = 1 << 23
    return w


def segment(w: Workload, noise: bool = True, inject: bool = True) -> np.ndarray:
    """fp64 strain segment of a single-segment config (0, 1, 2, 4)."""
    assert w.config != 3, "config 3 is a stream: use stream()/stream_segment()"
    D = noise_spectrum(w.n, w.seed, w.fs, w.f_low) if noise else np.zeros(w.n // 2 + 1, np.complex128)
    if inject:
        for (_, m1, m2, snr, j_c) in w.injections:
            D = D + injection_spectrum(w.n, m1, m2, snr, j_c, w.fs, w.f_low)
    return time_series(D, w.n)


def stream(w: Workload) -> np.ndarray:
    """Config 3: one coloured-noise realisation of 2^23 samples with its injections."""
    ns = w.stream_len
    D = noise_spectrum(ns, w.seed, w.fs, w.f_low)
    for (_, m1, m2, snr, j_c) in w.injections:
        D = D + injection_spectrum(ns, m1, m2, snr, j_c, w.fs, w.f_low)
    return time_series(D, ns)


def stream_segment(x: np.ndarray, q: int, n: int = 1 << 20) -> np.ndarray:
    """Half-overlapping segment q = 0..14 of the config-3 stream."""
    return x[q * (n // 2): q * (n // 2) + n]
