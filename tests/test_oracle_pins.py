"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-types an oracle formula: they use the literal O(N^2) DFT, closed forms, invariants,
independent numpy scratch values (tests/golden/, cited there), Gaussian-noise moments and
a brute-force double sum without any FFT.
"""
import math
import os

import numpy as np
import pytest

import oracle
import workloads as inputs


def _rows(path):
    out = []
    with open(path) as fh:
        for line in fh:
            line = line.strip()
            if line and not line.startswith("#"):
                out.append([float(x) for x in line.split()])
    return out


# ----------------------------------------------------------------------------- P1: FFT
@pytest.mark.parametrize("n", [2, 4, 8, 16, 64, 256])
@pytest.mark.parametrize("sign", [+1, -1])
def test_p1_fft_vs_naive_dft(n, sign):
    x = inputs.normal(11, 0, np.arange(n)) + 1j * inputs.normal(11, 1, np.arange(n))
    a, b = oracle.fft(x, sign), oracle.dft_naive(x, sign)
    assert np.max(np.abs(a - b)) <= 1e-12 * n * np.max(np.abs(x))


def test_p1_naive_dft_is_the_definition():
    # the naive routine itself against numpy's transform (sign -1 = numpy fft; +1 = n * ifft)
    x = inputs.normal(12, 0, np.arange(32)) + 1j * inputs.normal(12, 1, np.arange(32))
    assert np.allclose(oracle.dft_naive(x, -1), np.fft.fft(x), atol=1e-12)
    assert np.allclose(oracle.dft_naive(x, +1), 32 * np.fft.ifft(x), atol=1e-12)


@pytest.mark.parametrize("n", [1 << 10, 1 << 14])
def test_p1_closed_forms(n):
    j0, k0 = 37, 101
    imp = np.zeros(n, complex); imp[j0] = 1.0
    k = np.arange(n)
    for sign in (+1, -1):
        assert np.max(np.abs(oracle.fft(imp, sign) - np.exp(sign * 2j * np.pi * ((j0 * k) % n) / n))) < 1e-12
        tone = np.exp(-sign * 2j * np.pi * ((k0 * k) % n) / n)      # -> n * delta_{k,k0}
        X = oracle.fft(tone, sign)
        want = np.zeros(n, complex); want[k0] = n
        assert np.max(np.abs(X - want)) < 1e-9 * n
    x = inputs.normal(13, 0, k) + 1j * inputs.normal(13, 1, k)
    X = oracle.fft(x, -1)
    assert abs(np.sum(np.abs(x) ** 2) - np.sum(np.abs(X) ** 2) / n) < 1e-10 * n       # Parseval
    assert np.max(np.abs(oracle.fft(X, +1) - n * x)) < 1e-12 * n * np.max(np.abs(x)) * 10   # fwd o inv = n I
    Xr = oracle.fft(x.real.astype(complex), -1)                                     # Hermitian
    assert np.max(np.abs(Xr[1:] - np.conj(Xr[1:][::-1]))) < 1e-10 * math.sqrt(n)
    # transposition pin: sign matters for an off-centre impulse
    assert np.max(np.abs(oracle.fft(imp, +1) - oracle.fft(imp, -1))) > 0.5


def test_p1_roundtrip_large():
    n = 1 << 22
    k = np.arange(n)
    x = inputs.normal(14, 0, k) + 1j * inputs.normal(14, 1, k)
    y = oracle.fft(oracle.fft(x, -1), +1) / n
    assert np.max(np.abs(y - x)) < 1e-12 * 50


def test_p1_bad_size():
    with pytest.raises(ValueError):
        oracle.fft(np.zeros(12, complex), 1)


# ----------------------------------------------------------------------------- P2: Eq. 2
def test_p2_psd_values(golden_dir):
    for f, want in _rows(os.path.join(golden_dir, "p2_psd_eq2.txt")):
        assert oracle.psd_eq2(f) == pytest.approx(want, rel=1e-13)
        assert float(inputs.psd_eq2(f)) == pytest.approx(want, rel=1e-13)     # the generator's own copy


def test_p2_psd_minimum_and_integral():
    f = np.linspace(100, 250, 150001)
    v = np.array([oracle.psd_eq2(x) for x in f[::50]])
    i = int(np.argmin(v))
    assert v[i] == pytest.approx(0.9992265, abs=2e-7)
    assert f[::50][i] == pytest.approx(152.84, abs=0.06)
    g = np.arange(40.0, 2048.0 + 1e-9, 1.0 / 64)
    s = np.array([oracle.psd_eq2(x) for x in g])
    integral = float(np.sum(0.5 * (s[1:] + s[:-1])) / 64)
    assert integral == pytest.approx(42481.4, abs=0.5)


# ----------------------------------------------------------------------------- P3: cut-offs
def test_p3_cutoffs(golden_dir):
    assert oracle.t_sun() == 4.9254909476412675e-6 == inputs.T_SUN
    assert oracle.f_isco(1.0, 1.0) * 2.0 == pytest.approx(4397.1748, abs=2e-4)
    for m1, m2, fi, kh in _rows(os.path.join(golden_dir, "p3_cutoffs.txt")):
        if fi > 0:
            assert oracle.f_isco(m1, m2) == pytest.approx(fi, rel=2e-7)
            assert oracle.f_isco(m2, m1) == oracle.f_isco(m1, m2)
        if kh > 0:
            assert oracle.k_high(m1, m2, 1 << 14) == int(kh)
    assert oracle.k_high(1, 1, 1 << 20) == 1 << 19                 # Nyquist wins, Nyquist bin is out
    assert oracle.k_low(1 << 14) == 160 and oracle.k_low(1 << 20) == 10240 and oracle.k_low(1 << 22) == 40960
    # closed form: k_high = ceil(f_cut/df)
    for (m1, m2) in [(3.0, 4.0), (11.0, 2.5)]:
        assert oracle.k_high(m1, m2, 1 << 18) == math.ceil(oracle.f_isco(m1, m2) / (4096.0 / (1 << 18)))


# ----------------------------------------------------------------------------- P4: phase
def test_p4_phase_values(golden_dir):
    for m1, m2, want in _rows(os.path.join(golden_dir, "p4_phase.txt")):
        assert oracle.phase(m1, m2, 40.0) == pytest.approx(want, abs=1e-5)
        assert oracle.phase(m2, m1, 40.0) == oracle.phase(m1, m2, 40.0)
        assert float(inputs.chirp_phase(m1, m2, 40.0)) == pytest.approx(want, abs=1e-5)   # the simulator's copy


def test_p4_phase_at_isco_is_universal_for_equal_masses():
    # v_ISCO = 6^(-1/2) whatever M, eta = 1/4  =>  Psi0(f_ISCO) is one number
    for m in (1.0, 1.4, 3.0, 8.0, 17.0):
        assert oracle.phase(m, m, oracle.f_isco(m, m)) == pytest.approx(-1.297059, abs=2e-6)
    # and that number from the series with v^2 = 1/6, eta = 1/4, evaluated here in rationals
    v = 6 ** -0.5
    eta = 0.25
    series = 1 + (3715 / 756 + 55 * eta / 9) / 6 - 16 * math.pi * v ** 3 + \
        (15293365 / 508032 + 27145 * eta / 504 + 3085 * eta ** 2 / 72) / 36
    assert oracle.phase(8, 8, oracle.f_isco(8, 8)) == pytest.approx(-math.pi / 4 + 3 / (128 * eta * v ** 5) * series, abs=1e-9)


@pytest.mark.parametrize("m1,m2,tau0", [(1.4, 1.4, 24.862863), (1.0, 1.0, 43.561002), (8.0, 8.0, 1.361281)])
def test_p4_newtonian_chirp_time(m1, m2, tau0):
    # -(1/2pi) d/df of the leading term 3/(128 eta v^5) is tau0 = 5/(256 eta) M (pi M f)^(-8/3).
    # Isolate the leading term by Richardson-free differencing of the full phase at two mass scalings is
    # not possible, so difference the full phase and compare with the full closed-form derivative.
    f, h = 40.0, 1e-3
    M = (m1 + m2) * oracle.t_sun()
    eta = m1 * m2 / (m1 + m2) ** 2
    assert 5.0 / (256.0 * eta) * M * (math.pi * M * f) ** (-8.0 / 3.0) == pytest.approx(tau0, abs=1e-6)
    v = (math.pi * M * f) ** (1.0 / 3.0)
    a2 = 3715 / 756 + 55 * eta / 9
    a3 = -16 * math.pi
    a4 = 15293365 / 508032 + 27145 * eta / 504 + 3085 * eta ** 2 / 72
    # d/df [3/(128 eta) (v^-5 + a2 v^-3 + a3 v^-2 + a4 v^-1)], dv/df = v/(3f)
    dpsi = 3 / (128 * eta) * (-5 * v ** -5 - 3 * a2 * v ** -3 - 2 * a3 * v ** -2 - a4 * v ** -1) / (3 * f)
    num = (oracle.phase(m1, m2, f + h) - oracle.phase(m1, m2, f - h)) / (2 * h)
    assert num == pytest.approx(dpsi, rel=1e-7)
    assert -dpsi / (2 * math.pi) == pytest.approx(tau0, rel=0.12)      # leading term dominates
    assert num < 0                                                      # phase decreases with f: up-chirp ends at t_c


def test_p4_horner_coefficients_of_8_8():
    # Psi0 = -pi/4 + c0 u^5 + c2 u^3 + c3 u^2 + c4 u with u = f^(-1/3): recover the
    # coefficients by least squares from oracle phases and compare with the listed values.
    f = np.linspace(40.0, 270.0, 400)
    u = f ** (-1.0 / 3.0)
    y = np.array([oracle.phase(8, 8, x) for x in f]) + math.pi / 4
    A = np.stack([u ** 5, u ** 3, u ** 2, u], axis=1)
    c, *_ = np.linalg.lstsq(A, y, rcond=None)
    want = [96037.0863088721, 2439.2654336626642, -1195.1659490677398, 69.04590419018707]
    assert np.allclose(c, want, rtol=1e-6)


# ----------------------------------------------------------------------------- P5/P6: sigma, edges, whole path
@pytest.fixture(scope="module")
def cfg0_noise_free():
    w = inputs.workload(0)
    s = inputs.segment(w, noise=False, inject=True)
    return w, s, w.psd


def test_p5_p6_config0_noise_free(golden_dir, cfg0_noise_free):
    w, s, Sn = cfg0_noise_free
    rows = _rows(os.path.join(golden_dir, "p5_p6_config0_noise_free.txt"))
    assert [(r[0], r[1]) for r in rows] == [tuple(m) for m in w.masses]
    assert float(np.sqrt(np.mean(s ** 2))) == pytest.approx(7.7228, abs=5e-4)
    assert int(np.argmax(np.abs(s))) == 8958            # chirp ends just before t_c: sign convention
    for r in rows:
        m1, m2, sig, edges, jstar, rho_w, chi_w = r[0], r[1], r[2], r[3:8], int(r[8]), r[9], r[10]
        rho, chi, sigma, e = oracle.filter_template(s, Sn, m1, m2, w.p)
        assert sigma == pytest.approx(sig, rel=2e-9)
        assert list(e) == [int(x) for x in edges]
        assert int(np.argmax(rho)) == jstar
        assert rho[jstar] == pytest.approx(rho_w, abs=1e-5)
        assert chi[jstar] == pytest.approx(chi_w, abs=1e-4)
    # closed forms for the matching template
    rho, chi, sigma, e, z = oracle.filter_template(s, Sn, 8, 8, w.p, bands=True)
    assert rho[9000] == pytest.approx(12.0, abs=1e-9)
    Ct = oracle.power_table(Sn, w.n)
    share = np.array([(Ct[e[l + 1] - 1] - (Ct[e[l] - 1] if l else 0.0)) / Ct[e[-1] - 1] for l in range(w.p)])
    assert np.allclose(share, [0.250412, 0.250668, 0.248924, 0.249997], atol=2e-6)
    assert chi[9000] == pytest.approx(w.p * 144.0 * np.sum((share - 1.0 / w.p) ** 2), rel=1e-7)
    assert chi[9000] == pytest.approx(0.001021435, abs=1e-8)
    # z_l = A sigma_l^2 / sigma at the peak (real, positive, phase of z is zero there up to -pi/4 conventions)
    assert np.allclose(np.abs(z[:, 9000]), 12.0 * share * sigma, rtol=1e-9)


def test_p5_invariants():
    n = 1 << 14
    Sn = inputs.psd_array(n)
    Ct = oracle.power_table(Sn, n)
    assert np.all(Ct[:160] == 0.0) and np.all(np.diff(Ct[160:]) > 0)
    df = 4096.0 / n
    f = np.arange(160, n // 2) * df
    assert Ct[-1] == pytest.approx(float(np.sum(f ** (-7 / 3) / inputs.psd_eq2(f))), rel=1e-12)
    for p in (1, 2, 4, 16):
        sig, e = oracle.sigma_edges(Ct, n, 1100, p)
        assert sig == pytest.approx(math.sqrt(4 * df * Ct[1099]), rel=1e-14)
        assert e[0] == 160 and e[-1] == 1100 and np.all(np.diff(e) > 0)
        shares = np.diff(np.concatenate([[0.0], Ct[e[1:] - 1]])) / Ct[1099]
        assert abs(np.sum(shares) - 1) < 1e-14
        onebin = np.max(np.diff(Ct[159:1100])) / Ct[1099]
        assert np.all(np.abs(shares - 1.0 / p) <= onebin + 1e-15)
        # definition of the edge, brute force: smallest k with C[k] >= l/p * total
        for l in range(1, p):
            kap = min(k for k in range(160, 1100) if Ct[k] >= (l / p) * Ct[1099])
            assert e[l] == kap + 1
    with pytest.raises(ValueError):
        oracle.sigma_edges(Ct, n, 160, 4)       # empty template


# ----------------------------------------------------------------------------- P7: identities
def test_p7_identities(cfg0_noise_free):
    w, _, Sn = cfg0_noise_free
    s = inputs.segment(w)                       # with noise
    rho, chi, sigma, e, z = oracle.filter_template(s, Sn, 6, 10, w.p, bands=True)
    zt = z.sum(axis=0)
    # one full-band inverse transform equals the sum of the band transforms
    h = oracle.template(6, 10, w.n)
    D = oracle.data_spectrum(s)
    spec = np.zeros(w.n, complex)
    spec[e[0]:e[-1]] = 4.0 / w.n * h[e[0]:e[-1]] * D[e[0]:e[-1]] / Sn[e[0]:e[-1]]
    zfull = oracle.fft(spec, +1)
    assert np.max(np.abs(zfull - zt)) < 1e-12 * np.max(np.abs(zt)) * 10
    assert np.allclose(rho, np.abs(zfull) / sigma, rtol=1e-10)
    lhs = np.sum(np.abs(z - zt / w.p) ** 2, axis=0)
    rhs = np.sum(np.abs(z) ** 2, axis=0) - np.abs(zt) ** 2 / w.p
    assert np.max(np.abs(lhs - rhs)) < 1e-12 * np.max(lhs)
    assert np.allclose(chi, w.p / sigma ** 2 * lhs, rtol=1e-12)
    _, chi1, _, _ = oracle.filter_template(s, Sn, 6, 10, 1)
    assert np.max(np.abs(chi1)) < 1e-20         # p = 1 => chi^2 == 0
    # against numpy's transform: z = n * ifft(spec)
    assert np.allclose(zfull, w.n * np.fft.ifft(spec), rtol=0, atol=1e-12 * np.max(np.abs(zfull)) * 10)


# ----------------------------------------------------------------------------- P8: covariances
def test_p8_covariances(cfg0_noise_free):
    w, _, Sn = cfg0_noise_free
    s = inputs.segment(w)
    rho, chi, sig, e = oracle.filter_template(s, Sn, 8, 10, w.p)
    m = 1234
    r2, c2, _, _ = oracle.filter_template(np.roll(s, m), Sn, 8, 10, w.p)
    assert np.max(np.abs(np.roll(rho, m) - r2)) < 1e-10 and np.max(np.abs(np.roll(chi, m) - c2)) < 1e-9
    r3, c3, _, _ = oracle.filter_template(3.0 * s, Sn, 8, 10, w.p)
    assert np.allclose(r3, 3 * rho, rtol=1e-12) and np.allclose(c3, 9 * chi, rtol=1e-12)
    r4, c4, s4, e4 = oracle.filter_template(2.0 * s, 4.0 * Sn, 8, 10, w.p)
    assert np.allclose(r4, rho, rtol=1e-11) and np.allclose(c4, chi, rtol=1e-10)
    assert s4 == pytest.approx(sig / 2.0, rel=1e-13) and list(e4) == list(e)
    r5, c5, s5, e5 = oracle.filter_template(s, Sn, 10, 8, w.p)
    assert np.array_equal(r5, rho) and np.array_equal(c5, chi) and s5 == sig
    # S_n below k_low is ignored
    Sn2 = Sn.copy(); Sn2[:160] = 7.0
    r6, _, _, _ = oracle.filter_template(s, Sn2, 8, 10, w.p)
    assert np.array_equal(r6, rho)


# ----------------------------------------------------------------------------- P9: noise statistics
def test_p9_noise_moments():
    # rho^2 ~ chi^2_2 (mean 2), chi^2 ~ chi^2_{2p-2} (mean 2p-2, variance 4p-4)
    n, p = 1 << 16, 8
    w = inputs.workload(0)
    D = inputs.noise_spectrum(n, 77)
    s = inputs.time_series(D, n)
    Sn = inputs.psd_array(n)
    assert np.var(s) == pytest.approx(42481.4, rel=0.05)       # var s = integral of S_n (P2)
    rho, chi, _, _ = oracle.filter_template(s, Sn, 3.0, 3.0, p)
    neff = n / 8
    assert np.mean(rho ** 2) == pytest.approx(2.0, abs=3 * 2.0 / math.sqrt(neff))
    assert np.mean(chi) == pytest.approx(2 * p - 2, abs=3 * math.sqrt(4 * p - 4) / math.sqrt(neff))
    assert np.var(chi) == pytest.approx(4 * p - 4, rel=0.15)
    # tail of rho: P(rho > x) = exp(-x^2/2)
    assert np.mean(rho > 2.0) == pytest.approx(math.exp(-2.0), rel=0.1)


# ----------------------------------------------------------------------------- P10: injection in noise
def test_p10_injection_in_noise():
    w = inputs.workload(0)
    s = inputs.segment(w)
    out = oracle.filter_bank(s, w.psd, w.masses, w.p, w.window, w.rho_thresh, keep=4)
    assert np.all(out["status"] == 0)
    trig = oracle.triggers(out, w.rho_thresh)
    mine = [t for t in trig if t[0] == 4]
    assert len(mine) == 1
    _, j, rho, chi = mine[0]
    assert abs(j - 9000) <= 3 and abs(rho - 12.0) < 3.0 and chi < 40.0
    assert out["rho_keep"][j] == rho and int(np.argmax(out["rho_keep"])) == j


# ----------------------------------------------------------------------------- P11: brute force, no FFT
def test_p11_bruteforce_whole_path():
    n, p, W = 256, 2, 64
    Sn = inputs.psd_array(n)
    D = inputs.noise_spectrum(n, 5) + inputs.injection_spectrum(n, 8, 8, 9.0, 100)
    s = inputs.time_series(D, n)
    assert oracle.k_low(n) == 3 and oracle.k_high(8, 8, n) == 18
    a = oracle.filter_template(s, Sn, 8, 8, p)
    b = oracle.filter_template_bruteforce(s, Sn, 8, 8, p)
    assert np.max(np.abs(a[0] - b[0])) < 1e-12 * max(1.0, np.max(b[0]))
    assert np.max(np.abs(a[1] - b[1])) < 1e-11 * max(1.0, np.max(b[1]))
    assert a[2] == b[2] and list(a[3]) == list(b[3])
    ta = oracle.window_maxima(a[0], a[1], W, 1.0)
    tb = oracle.window_maxima(b[0], b[1], W, 1.0)
    assert ta[0] == tb[0] and np.array_equal(ta[1], tb[1])


# ----------------------------------------------------------------------------- O9: trigger rule (definition of this build)
def test_trigger_rule():
    rho = np.zeros(24); chi = np.arange(24.0)
    rho[[2, 5]] = 7.0          # tie inside window 0 -> lowest index
    rho[9] = 6.0; rho[11] = 5.0   # window 1: max == threshold: strict '>' rejects
    rho[21] = 6.5; rho[22] = 6.4; rho[17] = 3.0
    cnt, bj, br, bc, ru = oracle.window_maxima(rho, chi, 8, 6.0)
    assert cnt == 2
    assert list(bj) == [2, 9, 21] and list(br) == [7.0, 6.0, 6.5] and list(bc) == [2.0, 9.0, 21.0]
    assert ru[0] == 7.0        # the tied sample is a competing peak
    assert ru[1] == 5.0
    assert ru[2] == 3.0        # 22 is a neighbour of the peak, not a competing peak


# ----------------------------------------------------------------------------- P12: physical amplitude / D_eff
def test_p12_amplitude_value_scaling_laws_and_horizon(golden_dir):
    # O10 (SURVEY.md 8(c2) reading 4).  (a) the value evaluated by hand, by logarithms, in the golden file;
    for m1, m2, d, want in _rows(os.path.join(golden_dir, "p12_amplitude.txt")):
        assert abs(oracle.amplitude(m1, m2, d) - want) <= 2e-11 * want
    # (b) scaling laws: A ~ 1 / D_eff; A depends on the masses through M_chirp^(5/6) only, so scaling both masses by k
    # scales A by k^(5/6), and two different pairs with one chirp mass share A
    a = oracle.amplitude(3.0, 1.2, 1.0)
    assert abs(oracle.amplitude(3.0, 1.2, 40.0) * 40.0 / a - 1.0) < 1e-14
    assert abs(oracle.amplitude(6.0, 2.4, 1.0) / a - 2.0 ** (5.0 / 6.0)) < 1e-14
    assert abs(oracle.amplitude(1.2, 3.0, 1.0) / a - 1.0) < 1e-15
    mc = (3.0 * 1.2) ** 0.6 / 4.2 ** 0.2
    m = mc * 2.0 ** 0.2                                   # the equal-mass pair with the same chirp mass
    assert abs(oracle.amplitude(m, m, 1.0) / a - 1.0) < 1e-13
    # (c) the literature's number (not this code's): the SNR-8 horizon of a 1.4+1.4 binary in the initial-LIGO design
    # curve, of which Eq. 2 x 9e-46/Hz is the fit, is about 33 Mpc (sky-averaged range 14-15 Mpc)
    n = 1 << 18
    C = oracle.power_table(inputs.psd_array(n), n)
    sigma, _ = oracle.sigma_edges(C, n, oracle.k_high(1.4, 1.4, n), 16)
    horizon = oracle.amplitude(1.4, 1.4, 1.0) * sigma / math.sqrt(9e-46) / 8.0
    assert 28.0 < horizon < 36.0, horizon
