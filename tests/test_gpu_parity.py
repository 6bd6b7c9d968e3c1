"""GPU-vs-oracle parity, element by element on the same seeded inputs, through the C ABI
(paper_0906_4175_b200.gwmf is argument marshalling only).  Run with `-m gpu` on a B200."""
import math
import os

import numpy as np
import pytest

import oracle
import parity
import workloads as inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gw():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_0906_4175_b200 import gwmf
    gwmf.load_library()
    return gwmf


@pytest.fixture(params=["decimated", "two_pass", "fused"])
def path(request):
    """The library's three paths (gwmf_params::path), each checked against the oracle."""
    return request.param


def _path_for(path, n):
    """A path the library supports at this n (fused: 2^15..2^20, decimated: >= 2^15), else auto."""
    if path == "fused" and not (1 << 15) <= n <= (1 << 20):
        return "auto"
    if path == "decimated" and n < (1 << 15):
        return "auto"
    return path


def _run_gpu(gw, w, s, Sn, masses=None, batch=0, window=None, thresh=None, p=None, path="auto"):
    masses = w.masses if masses is None else masses
    f = gw.Filter(w.n, p or w.p, window or w.window, len(masses), rho_thresh=w.rho_thresh if thresh is None else thresh,
                  batch=batch, path=_path_for(path, w.n))
    f.make_bank(masses)
    f.load_segment(s.astype(np.float32), Sn)
    f.filter()
    return f


# ----------------------------------------------------------------------------- the FFT alone
@pytest.mark.parametrize("log_n", [14, 15, 16, 17, 18, 19, 20, 21, 22])
def test_fft_inverse_alone(gw, log_n):
    import torch
    n = 1 << log_n
    k = np.arange(n)
    x = (inputs.normal(100 + log_n, 0, k) + 1j * inputs.normal(100 + log_n, 1, k)).astype(np.complex64)
    f = gw.Filter(n, 4, 4096, 1)
    X = f.fft_inverse(torch.from_numpy(x).cuda())
    f.synchronize()
    want = oracle.fft(x.astype(np.complex128), +1)
    got = X.cpu().numpy().astype(np.complex128)
    rms = math.sqrt(n) * 1.41
    err = np.max(np.abs(got - want)) / rms
    assert err < 4e-6, err
    # closed form: an impulse at j0 -> a pure tone (catches a transposed index map at any size)
    imp = np.zeros(n, np.complex64); imp[12345 % n] = 1.0
    T = f.fft_inverse(torch.from_numpy(imp).cuda()).cpu().numpy()
    tone = np.exp(2j * np.pi * ((12345 % n) * k % n) / n)
    assert np.max(np.abs(T - tone)) < 2e-6


# ----------------------------------------------------------------------------- the correlate step alone
@pytest.mark.parametrize("log_n,masses", [(14, (8.0, 8.0)), (18, (1.0, 1.0)), (20, (1.4, 1.4))])
def test_correlate_alone(gw, log_n, masses):
    # Q[k] = (4/n) D[k] f^(-7/6) e^{i Psi0} / (S_n sigma_ref) against the oracle's template and data spectrum.
    # (1,1) Msun at 40 Hz carries Psi0 = 6.7e3 rad: a phase evaluated in fp32 would be off by 1e-3 rad.
    n = 1 << log_n
    m1, m2 = masses
    s = inputs.time_series(inputs.noise_spectrum(n, 300 + log_n), n).astype(np.float32)
    Sn = inputs.psd_array(n)
    f = gw.Filter(n, 4, 4096, 1)
    f.make_bank([masses])
    f.load_segment(s, Sn)
    q = f.correlate(0).astype(np.complex128)
    D = oracle.data_spectrum(s.astype(np.float64))[: n // 2]
    h = oracle.template(m1, m2, n)                        # f^(-7/6) e^{i Psi0} on [k_low, k_high), 0 elsewhere
    Ctab = oracle.power_table(Sn, n)
    df = inputs.FS / n
    sigma_ref = math.sqrt(4.0 * df * Ctab[n // 2 - 1])
    inv_sn = np.zeros(n // 2)
    k_low = int(math.ceil(inputs.F_LOW / df))
    inv_sn[k_low:] = 1.0 / Sn[k_low:n // 2]
    want = (4.0 / n) * D * h * inv_sn / sigma_ref
    scale = np.sqrt(np.mean(np.abs(want[np.abs(want) > 0]) ** 2))
    assert np.count_nonzero(want) > 100
    assert np.all(q[want == 0] == 0)
    # the library's data spectrum comes from its fp32 FFT: absolute error ~ 1e-6 * rms(D) in every bin, carried
    # into Q by the bin's weight; the template phasor and the fp32 products add ~1e-6 relative
    weight = np.abs((4.0 / n) * h * inv_sn / sigma_ref)
    rms_d = np.sqrt(np.mean(np.abs(D[k_low:]) ** 2))
    err = np.abs(q - want) - (3e-6 * np.abs(want) + 4e-6 * rms_d * weight)
    assert np.max(err) <= 0, (int(np.argmax(err)), q[int(np.argmax(err))], want[int(np.argmax(err))], scale)
    # phase alone, bin by bin, on the bins at or above the rms (there the fp32 FFT of the data contributes
    # ~1e-6 rad, the fp64-reduced template phase 4e-7, the fp32 products 1e-7)
    big = (np.abs(D) > rms_d) & (np.abs(want) > 0)
    dphi = np.angle(q[big] / want[big])
    assert np.max(np.abs(dphi)) < 4e-6, np.max(np.abs(dphi))


# ----------------------------------------------------------------------------- config 0, everything
def test_config0_full(gw, path):
    w = inputs.workload(0)
    s = inputs.segment(w)
    Sn = w.psd
    f = _run_gpu(gw, w, s, Sn, path=path)
    out = oracle.filter_bank(s.astype(np.float32).astype(np.float64), Sn, w.masses, w.p, w.window, w.rho_thresh)
    parity.assert_sigma_edges(f.sigma(), f.band_edges(), out["sigma"], out["edges"])
    s32 = s.astype(np.float32).astype(np.float64)
    for t, (m1, m2) in enumerate(w.masses):
        rho_o, chi_o, _, _ = oracle.filter_template(s32, Sn, m1, m2, w.p)
        rho_g, chi_g = f.series(t)
        parity.assert_series(rho_g, chi_g, rho_o, chi_o, w.p, f"config0 template {t}")
    trig = f.triggers()
    compared, exempt = parity.assert_triggers(trig, out, w.rho_thresh, w.window, w.p)
    assert compared >= 1
    mine = [t for t in trig if t["template_id"] == 4]
    assert len(mine) == 1 and abs(int(mine[0]["sample"]) - 9000) <= 3


def test_config0_noise_free_closed_forms(gw):
    # P6 on the GPU: rho = A = 12 at t_c, chi^2 = 0.001021 (closed form), other templates as tabulated
    w = inputs.workload(0)
    s = inputs.segment(w, noise=False)
    f = _run_gpu(gw, w, s, w.psd)
    rho, chi = f.series(4)
    assert int(np.argmax(rho)) == 9000
    assert rho[9000] == pytest.approx(12.0, abs=1e-3 + 12e-4)
    assert chi[9000] == pytest.approx(0.001021435, abs=1e-3)
    rho1, chi1 = f.series(2)                       # (6,10): 9011, 9.245720, 25.878613
    assert int(np.argmax(rho1)) == 9011 and rho1[9011] == pytest.approx(9.245720, abs=2e-3)
    assert chi1[9011] == pytest.approx(25.878613, rel=1e-3)


# ----------------------------------------------------------------------------- ragged mid-size cases
@pytest.mark.parametrize("log_n,p,window,batch", [(15, 5, 2048, 3), (16, 7, 8192, 2), (17, 16, 4096, 0),
                                                  (19, 3, 1 << 19, 5)])
def test_midsize_full_series(gw, path, log_n, p, window, batch):
    n = 1 << log_n
    masses = [(1.0, 1.0), (1.4, 1.4), (3.0, 1.2), (5.0, 5.0), (10.0, 1.4), (12.0, 9.0), (20.0, 14.0)]
    D = inputs.noise_spectrum(n, 40 + log_n)
    D = D + inputs.injection_spectrum(n, 3.0, 1.2, 11.0, n // 3) + inputs.injection_spectrum(n, 12.0, 9.0, 9.0, n - 5)
    s = inputs.time_series(D, n).astype(np.float32)
    Sn = inputs.psd_array(n)
    w = inputs.Workload(config=-1, n=n, p=p, rho_thresh=5.0, window=window, masses=masses, seed=0)
    f = _run_gpu(gw, w, s, Sn, batch=batch, path=path)
    out = oracle.filter_bank(s.astype(np.float64), Sn, masses, p, window, 5.0)
    parity.assert_sigma_edges(f.sigma(), f.band_edges(), out["sigma"], out["edges"])
    for t, (m1, m2) in enumerate(masses):
        rho_o, chi_o, _, _ = oracle.filter_template(s.astype(np.float64), Sn, m1, m2, p)
        rho_g, chi_g = f.series(t)
        parity.assert_series(rho_g, chi_g, rho_o, chi_o, p, f"n=2^{log_n} template {t}")
    compared, _ = parity.assert_triggers(f.triggers(), out, 5.0, window, p)
    assert compared >= 2


# ----------------------------------------------------------------------------- configs 1, 2, 4: sampled templates
def _sampled_config(gw, config, sample_ids, n_templates=None, path="auto"):
    w = inputs.workload(config, n_templates)
    s = inputs.segment(w).astype(np.float32)
    Sn = w.psd
    f = _run_gpu(gw, w, s, Sn, path=path)
    trig = f.triggers()
    sub = [w.masses[i] for i in sample_ids]
    s64 = s.astype(np.float64)
    out = oracle.filter_bank(s64, Sn, sub, w.p, w.window, w.rho_thresh)
    sig, edges = f.sigma(), f.band_edges()
    parity.assert_sigma_edges(sig[sample_ids], edges[sample_ids], out["sigma"], out["edges"])
    compared, exempt = parity.assert_triggers(trig, out, w.rho_thresh, w.window, w.p, template_ids=sample_ids)
    # full series of two of the sampled templates
    for i in sample_ids[:2]:
        rho_o, chi_o, _, _ = oracle.filter_template(s64, Sn, w.masses[i][0], w.masses[i][1], w.p)
        rho_g, chi_g = f.series(i)
        parity.assert_series(rho_g, chi_g, rho_o, chi_o, w.p, f"config {config} template {i}")
    return w, trig, compared


def test_config1_all_templates(gw, path):
    w = inputs.workload(1)
    s = inputs.segment(w).astype(np.float32)
    Sn = w.psd
    f = _run_gpu(gw, w, s, Sn, path=path)
    out = oracle.filter_bank(s.astype(np.float64), Sn, w.masses, w.p, w.window, w.rho_thresh)
    parity.assert_sigma_edges(f.sigma(), f.band_edges(), out["sigma"], out["edges"])
    compared, exempt = parity.assert_triggers(f.triggers(), out, w.rho_thresh, w.window, w.p)
    assert compared >= 3
    for t in (0, 97, 255):
        rho_o, chi_o, _, _ = oracle.filter_template(s.astype(np.float64), Sn, w.masses[t][0], w.masses[t][1], w.p)
        rho_g, chi_g = f.series(t)
        parity.assert_series(rho_g, chi_g, rho_o, chi_o, w.p, f"config 1 template {t}")


# ----------------------------------------------------------------------------- the headline config in full
class _OracleCache:
    """One oracle run per workload, shared by every path and threshold (the oracle's per-window maxima do not depend
    on the threshold), and the full series of the templates that are compared element by element."""

    def __init__(self):
        self.bank = {}
        self.series = {}

    def bank_out(self, key, s64, Sn, masses, p, window, thresh):
        if key not in self.bank:
            self.bank[key] = oracle.filter_bank(s64, Sn, masses, p, window, thresh)
        return self.bank[key]

    def template_series(self, key, s64, Sn, m1, m2, p):
        if key not in self.series:
            rho, chi, _, _ = oracle.filter_template(s64, Sn, m1, m2, p)
            self.series[key] = (rho.astype(np.float32), chi.astype(np.float32))     # fp32 copies: 8 MB per template
        return self.series[key]


@pytest.fixture(scope="module")
def ocache():
    return _OracleCache()


def _stratified_ids(edges, must=()):
    """Template ids covering every class of widest-band row count (<= 4, 5-8, 9-16, 17-32, > 32 input rows of 1024
    bins) -- the classes the kernels specialise on -- two per class where the bank has them."""
    rows = ((edges[:, 1:] - 1) >> 10) - (edges[:, :-1] >> 10) + 1
    rows = np.where(edges[:, 1:] > edges[:, :-1], rows, 0).max(axis=1)
    ids = list(must)
    for lo, hi in ((0, 4), (5, 8), (9, 16), (17, 32), (33, 1 << 30)):
        cls = [int(i) for i in np.nonzero((rows >= lo) & (rows <= hi))[0] if int(i) not in ids]
        ids += cls[:1] + cls[-1:] if len(cls) > 1 else cls
    return sorted(set(ids))


def test_config2_headline_full_bank(gw, ocache, path):
    # BASELINE.json:configs[2] in the launch configuration bench.py times, ALL 1024 templates: sigma, band edges and
    # every (template, window) cell at the config's threshold 6 and again at 4 (tens of events per template, so the
    # timed kernel instantiation -- no series output, full batches -- is checked densely), plus the full series of
    # templates of every band-width class (the paper's own accuracy test ran over ~5e4 events)
    w = inputs.workload(2)
    s = inputs.segment(w).astype(np.float32)
    s64 = s.astype(np.float64)
    Sn = w.psd
    out = ocache.bank_out("c2", s64, Sn, w.masses, w.p, w.window, w.rho_thresh)
    assert np.all(out["status"] == 0)
    f = _run_gpu(gw, w, s, Sn, path=path)
    edges = f.band_edges()
    parity.assert_sigma_edges(f.sigma(), edges, out["sigma"], out["edges"])
    trig = f.triggers()
    compared, exempt = parity.assert_triggers(trig, out, w.rho_thresh, w.window, w.p)
    inj = sorted({b for (b, *_rest) in w.injections})
    assert compared >= len(inj)
    assert len(trig) < 2000                     # exp(-18) * N * T ~ 16 noise samples + the injections
    f4 = _run_gpu(gw, w, s, Sn, thresh=4.0, path=path)

    def series_of(tid):
        rho_o, chi_o, _, _ = oracle.filter_template(s64, Sn, w.masses[tid][0], w.masses[tid][1], w.p)
        return rho_o, chi_o

    compared4, exempt4 = parity.assert_triggers(f4.triggers(), out, 4.0, w.window, w.p, series_of=series_of)
    assert compared4 > 20 * len(w.masses)       # e^-8 per sample: tens of windows per template cross 4
    for i in _stratified_ids(edges, must=(992, inj[0])):       # 992 = (1,1) Msun: reaches Nyquist
        rho_o, chi_o = ocache.template_series(("c2", i), s64, Sn, w.masses[i][0], w.masses[i][1], w.p)
        rho_g, chi_g = f.series(i)
        parity.assert_series(rho_g, chi_g, rho_o.astype(np.float64), chi_o.astype(np.float64), w.p, f"config 2 template {i}")


@pytest.mark.parametrize("path4", ["decimated", "two_pass"])
def test_config4_long_segment_64_templates(gw, ocache, path4):
    # BASELINE.json:configs[4] (N = 2^22, p = 32): 64 of the 512 templates, evenly spread, every window cell
    w = inputs.workload(4)
    s = inputs.segment(w).astype(np.float32)
    s64 = s.astype(np.float64)
    Sn = w.psd
    inj = sorted({b for (b, *_rest) in w.injections})
    ids = sorted(set(list(np.linspace(0, len(w.masses) - 1, 64 - len(inj)).astype(int)) + inj))
    out = ocache.bank_out("c4", s64, Sn, [w.masses[i] for i in ids], w.p, w.window, w.rho_thresh)
    f = _run_gpu(gw, w, s, Sn, path=path4)
    parity.assert_sigma_edges(f.sigma()[ids], f.band_edges()[ids], out["sigma"], out["edges"])
    compared, exempt = parity.assert_triggers(f.triggers(), out, w.rho_thresh, w.window, w.p, template_ids=ids)
    assert compared >= len(inj)
    for i in (ids[0], inj[0]):
        rho_o, chi_o = ocache.template_series(("c4", i), s64, Sn, w.masses[i][0], w.masses[i][1], w.p)
        rho_g, chi_g = f.series(i)
        parity.assert_series(rho_g, chi_g, rho_o.astype(np.float64), chi_o.astype(np.float64), w.p, f"config 4 template {i}")


@pytest.mark.parametrize("config", [1, 2])
def test_chisq_on_demand_matches_oracle_and_every_sample_mode(gw, ocache, config):
    # SURVEY 8(f)-2 / PAPER.md:164: rho(t) from ONE full-band transform per template, chi^2 evaluated from its
    # definition at the event samples only.  Every event (rho, sample, chi^2) against the oracle over the whole bank,
    # and against the chi^2-at-every-sample run of the same library.
    w = inputs.workload(config)
    s = inputs.segment(w).astype(np.float32)
    s64 = s.astype(np.float64)
    Sn = w.psd
    out = ocache.bank_out(f"c{config}", s64, Sn, w.masses, w.p, w.window, w.rho_thresh)
    f = gw.Filter(w.n, w.p, w.window, len(w.masses), rho_thresh=w.rho_thresh, chisq_on_demand=True)
    f.make_bank(w.masses)
    f.load_segment(s, Sn)
    assert np.all(f.transform_counts() == 1)
    f.filter()
    trig = f.triggers()
    compared, exempt = parity.assert_triggers(trig, out, w.rho_thresh, w.window, w.p)
    assert compared >= 3
    ref = _run_gpu(gw, w, s, Sn).triggers()
    a = {(int(t["template_id"]), int(t["sample"])): t for t in trig}
    b = {(int(t["template_id"]), int(t["sample"])): t for t in ref}
    common = set(a) & set(b)
    assert len(common) >= 0.98 * max(len(a), len(b))      # cells within fp32 rounding of the threshold / a tie may differ
    for key in common:
        assert abs(float(a[key]["rho"]) - float(b[key]["rho"])) <= 1e-4 * float(b[key]["rho"])
        assert abs(float(a[key]["chisq"]) - float(b[key]["chisq"])) <= 1e-3 * float(b[key]["chisq"]) + 1e-3
    rho_g, chi_g = f.series(3)                             # rho(t) is still available; chi^2(t) is not formed
    rho_o, _ = ocache.template_series((f"c{config}", 3), s64, Sn, w.masses[3][0], w.masses[3][1], w.p)
    assert np.max(np.abs(rho_g - rho_o) - (1e-3 + 1e-4 * rho_o)) <= 0 and np.all(chi_g == 0.0)


def test_noise_statistics_at_full_size(gw):
    # in stationary Gaussian noise rho^2 is chi^2 with 2 degrees of freedom and the veto
    # statistic chi^2 with 2p - 2, whatever the template: properties that hold at any size, checked at the
    # headline shape (N = 2^20, p = 16) in the launch configuration bench.py times (SURVEY pin P9)
    w = inputs.workload(2)
    s = inputs.segment(w, inject=False).astype(np.float32)
    f = _run_gpu(gw, w, s, w.psd)
    n_eff = w.n / 8.0                                    # neighbouring samples are correlated
    for t in (0, 517, 1023):
        rho, chi = f.series(t)
        r2 = rho.astype(np.float64) ** 2
        assert abs(r2.mean() - 2.0) < 3 * 2.0 / math.sqrt(n_eff), (t, r2.mean())
        nu = 2 * w.p - 2
        assert abs(chi.mean() - nu) < 3 * math.sqrt(2 * nu / n_eff) + 0.02 * nu, (t, chi.mean())
        assert abs(chi.astype(np.float64).var() - 2 * nu) < 0.15 * 2 * nu, (t, chi.var())
    # exceedances of the threshold: P(rho > 6) = e^-18 per sample -> ~16 samples over the whole bank
    assert len(f.triggers()) < 200


def test_long_segment_p16_sampled(gw):
    # SURVEY 8(f)-3 / PAPER.md:119,194: N = 4 x 2^20 segments with the headline p = 16 (the paper's "another
    # factor of 2" shape): config 4's segment and bank, 16 bands
    w = inputs.workload(4, 48)
    s = inputs.segment(w).astype(np.float32)
    Sn = w.psd
    f = _run_gpu(gw, w, s, Sn, p=16)
    ids = [0, 17, 47]
    s64 = s.astype(np.float64)
    out = oracle.filter_bank(s64, Sn, [w.masses[i] for i in ids], 16, w.window, w.rho_thresh)
    parity.assert_sigma_edges(f.sigma()[ids], f.band_edges()[ids], out["sigma"], out["edges"])
    parity.assert_triggers(f.triggers(), out, w.rho_thresh, w.window, 16, template_ids=ids)
    rho_o, chi_o, _, _ = oracle.filter_template(s64, Sn, *w.masses[17], 16)
    rho_g, chi_g = f.series(17)
    parity.assert_series(rho_g, chi_g, rho_o, chi_o, 16, "N=2^22, p=16, template 17")


def test_snr_only_mode_is_p1(gw):
    # SURVEY 8(f)-2 / PAPER.md:164 (the pipeline without chi^2): p = 1 is one band = the whole template, i.e.
    # one inverse FFT per template; rho and the triggers must equal those of the p = 16 run, chi^2 == 0
    w = inputs.workload(1, 24)
    s = inputs.segment(w).astype(np.float32)
    f16 = _run_gpu(gw, w, s, w.psd)
    f1 = _run_gpu(gw, w, s, w.psd, p=1)
    t16, t1 = f16.triggers(), f1.triggers()
    out = oracle.filter_bank(s.astype(np.float64), w.psd, w.masses, 1, w.window, w.rho_thresh)
    parity.assert_triggers(t1, out, w.rho_thresh, w.window, 1)
    assert np.all(t1["chisq"] == 0.0)
    k16 = {(int(t["template_id"]), int(t["sample"])): float(t["rho"]) for t in t16}
    k1 = {(int(t["template_id"]), int(t["sample"])): float(t["rho"]) for t in t1}
    common = set(k16) & set(k1)
    assert len(common) >= 0.9 * max(len(k16), 1)          # cells within 1e-3 of threshold / a rival peak may differ
    assert all(abs(k16[c] - k1[c]) <= 1e-3 + 1e-4 * k16[c] for c in common)


def test_sub_grid_bands_and_prepass_are_exercised(gw):
    # Decimated path, the two branches that only wide bands reach: a class-S band of 8193..32768 bins is
    # transformed as 2 or 4 interleaved sub-grids of 2^14 points (k_bandpower<14, true>), and an effective band of more
    # than 32 * 6 input rows at n = 2^20 is pre-passed (k_prepass, one 32-point transform over the Horner rounds).
    # The bank is chosen so that both occur (checked from the band edges), then every sample is compared.
    n, p = 1 << 20, 7
    masses = [(1.4, 1.4), (3.0, 2.5), (8.0, 6.0)]
    D = inputs.noise_spectrum(n, 77) + inputs.injection_spectrum(n, 3.0, 2.5, 10.0, 123457)
    s = inputs.time_series(D, n).astype(np.float32)
    Sn = inputs.psd_array(n)
    w = inputs.Workload(config=-1, n=n, p=p, rho_thresh=5.5, window=4096, masses=masses, seed=0)
    f = _run_gpu(gw, w, s, Sn, path="decimated")
    edges = f.band_edges()
    widths = np.diff(edges, axis=1)
    assert np.any((widths > 8192) & (widths <= 16384)), "no band on a 2^15-point grid (2 sub-grids)"
    assert np.any((widths > 16384) & (widths <= 32768)), "no band on a 2^16-point grid (4 sub-grids)"
    rows = (edges[:, 1:] - 1) // 1024 - edges[:, :-1] // 1024 + 1
    assert np.any((widths > 32768) & (rows > 192)), "no pre-passed band"
    out = oracle.filter_bank(s.astype(np.float64), Sn, masses, p, 4096, 5.5)
    parity.assert_sigma_edges(f.sigma(), edges, out["sigma"], out["edges"])
    for t, (m1, m2) in enumerate(masses):
        rho_o, chi_o, _, _ = oracle.filter_template(s.astype(np.float64), Sn, m1, m2, p)
        rho_g, chi_g = f.series(t)
        parity.assert_series(rho_g, chi_g, rho_o, chi_o, p, f"sub-grid / pre-pass case, template {t}")
    compared, _ = parity.assert_triggers(f.triggers(), out, 5.5, 4096, p)
    assert compared >= 1


def test_config3_sweep_256_pairs_overlapped_loads(gw):
    # BASELINE.json:configs[3]: half-overlapping segments of one stream against the 4096-template bank, driven the way
    # bench.py --workload sweep drives it: the next segment is uploaded and prepared (gwmf_load_segment with Sn = NULL,
    # on the library's upload stream) while the current one is still being filtered, and the events of the current
    # one are collected afterwards.  4 segments x 64 templates = 256 (segment, template) pairs against the oracle.
    w = inputs.workload(3)
    x = inputs.stream(w).astype(np.float32)
    Sn = w.psd
    f = gw.Filter(w.n, w.p, w.window, len(w.masses), rho_thresh=w.rho_thresh)
    f.make_bank(w.masses)
    ids = [int(i) for i in np.linspace(0, len(w.masses) - 1, 64)]
    segs = (0, 1, 7, 14)
    f.load_segment(inputs.stream_segment(x, segs[0], w.n), Sn)
    trigs = []
    for i, q in enumerate(segs):
        f.filter()
        if i + 1 < len(segs):
            f.load_segment(inputs.stream_segment(x, segs[i + 1], w.n).copy())       # Sn = None: overlapped
        trigs.append(f.triggers().copy())                                           # events of segment q
    n_compared = 0
    for q, trig in zip(segs, trigs):
        seg = inputs.stream_segment(x, q, w.n).astype(np.float64)
        out = oracle.filter_bank(seg, Sn, [w.masses[i] for i in ids], w.p, w.window, w.rho_thresh)
        compared, _ = parity.assert_triggers(trig, out, w.rho_thresh, w.window, w.p, template_ids=ids)
        n_compared += compared
    assert n_compared >= 1
    # the last segment is still loaded: one full series
    seg = inputs.stream_segment(x, segs[-1], w.n).astype(np.float64)
    rho_o, chi_o, _, _ = oracle.filter_template(seg, Sn, *w.masses[ids[31]], w.p)
    rho_g, chi_g = f.series(ids[31])
    parity.assert_series(rho_g, chi_g, rho_o, chi_o, w.p, "config 3 last segment")


def test_load_segment_semantics(gw):
    # Sn = NULL before any PSD is an error; events survive a following load until the next filter; a reloaded segment
    # gives bit-identical events whichever way it was loaded
    import torch
    w = inputs.workload(1, 12)
    s = inputs.segment(w).astype(np.float32)
    s2 = np.roll(s, 1000)
    f = gw.Filter(w.n, w.p, w.window, len(w.masses), rho_thresh=5.0)
    f.make_bank(w.masses)
    with pytest.raises(gw.GwmfError) as e:
        f.load_segment(s)
    assert e.value.status == gw.E_STATE
    f.load_segment(s, w.psd)
    f.filter()
    a = f.triggers().copy()
    f.load_segment(s2)                          # overlapped path; the events of s stay readable
    assert f.triggers().tobytes() == a.tobytes()
    f.filter()
    b = f.triggers().copy()
    assert b.tobytes() != a.tobytes()
    shifted = {(int(t["template_id"]), (int(t["sample"]) + 1000) % w.n) for t in a}
    assert {(int(t["template_id"]), int(t["sample"])) for t in b} & shifted   # P8: rotating s rotates the events
    f.load_segment(torch.from_numpy(s).cuda())  # device source, same PSD
    f.filter()
    assert f.triggers().tobytes() == a.tobytes()
    f.load_segment(s, w.psd)                    # host source with the PSD again
    f.filter()
    assert f.triggers().tobytes() == a.tobytes()


def test_wide_band_inside_narrow_ones(gw, path):
    # a PSD with a strong line: the band that has to cross it becomes wide while its neighbours stay narrow, so the
    # decimated path's union of narrow bands has a hole (a class-D band inside the hull of Z) -- DESIGN.md section 5
    n = 1 << 20                                 # 70 Hz = 17920 bins > 8192: the crossing band is class D
    Sn = inputs.psd_array(n)
    df = inputs.FS / n
    lo, hi = int(95.0 / df), int(165.0 / df)
    Sn = Sn.copy()
    Sn[lo:hi] *= 1e4                            # 95-165 Hz carries almost no weight
    masses = [(1.4, 1.4), (5.0, 4.0), (12.0, 9.0)]
    D = inputs.noise_spectrum(n, 71)
    D[lo:hi] *= 100.0                           # noise consistent with the PSD
    D = D + inputs.injection_spectrum(n, 5.0, 4.0, 30.0, n // 5)
    s = inputs.time_series(D, n).astype(np.float32)
    w = inputs.Workload(config=-1, n=n, p=16, rho_thresh=5.0, window=4096, masses=masses, seed=0)
    f = _run_gpu(gw, w, s, Sn, path=path)
    out = oracle.filter_bank(s.astype(np.float64), Sn, masses, 16, 4096, 5.0)
    parity.assert_sigma_edges(f.sigma(), f.band_edges(), out["sigma"], out["edges"])
    e = np.asarray(out["edges"])
    widths = np.diff(e, axis=1)
    interior_wide = [(t, l) for t in range(len(masses)) for l in range(1, 15)
                     if widths[t, l] > 8192 and widths[t, :l].min() <= 8192 and widths[t, l + 1:].min() <= 8192]
    assert interior_wide, "this case is meant to put a wide band between narrow ones"
    for t, (m1, m2) in enumerate(masses):
        rho_o, chi_o, _, _ = oracle.filter_template(s.astype(np.float64), Sn, m1, m2, 16)
        rho_g, chi_g = f.series(t)
        parity.assert_series(rho_g, chi_g, rho_o, chi_o, 16, f"line PSD template {t}")
    parity.assert_triggers(f.triggers(), out, 5.0, 4096, 16)


@pytest.mark.parametrize("snr", [100.0, 300.0, 1000.0])
def test_loud_events(gw, path, snr):
    # The veto exists for loud events (section 1.2).  A matched injection of optimal SNR 100, 300, 1000 in
    # Eq. 2 noise at the headline shape: every sample of the matched template and of a mismatched one (large chi^2),
    # and the events of the whole bank, at the tolerances of every other test.  chi^2 at such a sample is a small
    # number next to rho^2; reading 23 says how the library evaluates it there.
    n, p, W = 1 << 20, 16, 4096
    masses = [(3.0, 1.2), (3.3, 1.25), (1.4, 1.4), (10.0, 8.0)]
    jc = 5 * n // 8 + 123
    D = inputs.noise_spectrum(n, 91) + inputs.injection_spectrum(n, 3.0, 1.2, snr, jc)
    s = inputs.time_series(D, n).astype(np.float32)
    s64 = s.astype(np.float64)
    Sn = inputs.psd_array(n)
    w = inputs.Workload(config=-1, n=n, p=p, rho_thresh=6.0, window=W, masses=masses, seed=0)
    f = _run_gpu(gw, w, s, Sn, path=path)
    out = oracle.filter_bank(s64, Sn, masses, p, W, 6.0)
    parity.assert_sigma_edges(f.sigma(), f.band_edges(), out["sigma"], out["edges"])
    assert abs(out["best_rho"][0].max() - snr) < 5.0          # the injection is found at about its SNR
    series = {}

    def series_of(tid):
        if tid not in series:
            series[tid] = oracle.filter_template(s64, Sn, masses[tid][0], masses[tid][1], p)[:2]
        return series[tid]

    compared, _ = parity.assert_triggers(f.triggers(), out, 6.0, W, p, series_of=series_of)
    assert compared >= 4
    for t in (0, 1):
        rho_o, chi_o = series_of(t)
        rho_g, chi_g = f.series(t)
        parity.assert_series(rho_g, chi_g, rho_o, chi_o, p, f"loud injection, SNR {snr}, template {t}")
    j = int(np.argmax(series_of(0)[0]))
    assert abs(j - jc) <= 1 and series_of(1)[1].max() > 50.0 * series_of(0)[1][j]   # matched: small chi^2; mismatched: large


@pytest.mark.parametrize("world", [2, 3])
def test_template_sharded_plan_on_the_cuda_path(gw, world):
    # SURVEY.md 8(e) / 8(f)-4, PAPER.md:75,196 (independent work, the multi-GPU extrapolation): bench.py's
    # template-sharded mode gives rank r the range shard_plan(world, r, T, "templates") of ONE bank against ONE segment
    # and concatenates the ranks' event lists in rank order (gather_triggers).  Here every "rank" is a context of its
    # own on cuda:0: the concatenated list must be byte-identical to the single-context list.  world = 3 cuts config
    # 1's 256 templates at odd indices, i.e. through the template pairs (2i, 2i+1) that share a transform.
    import bench
    w = inputs.workload(1)
    s = inputs.segment(w).astype(np.float32)
    T = len(w.masses)
    whole = _run_gpu(gw, w, s, w.psd, thresh=4.5)
    ref = whole.triggers()
    assert len(ref) > 2 * T                                  # a dense list: several events per template at rho* = 4.5
    parts, covered = [], 0
    for r in range(world):
        _, first, count = bench.shard_plan(world, r, T, "templates")
        assert first == covered
        covered += count
        f = gw.Filter(w.n, w.p, w.window, T, rho_thresh=4.5)
        f.make_bank(w.masses)
        f.load_segment(s, w.psd)
        f.filter(first, count)
        t = f.triggers()
        assert np.all((t["template_id"] >= first) & (t["template_id"] < first + count))
        parts.append(t)
        f.close()
    assert covered == T
    assert np.concatenate(parts).tobytes() == ref.tobytes()


# ----------------------------------------------------------------------------- edge cases and the boundary
def test_p_extremes_and_covariance(gw, path):
    n = 1 << 15
    masses = [(2.0, 1.5), (9.0, 7.0)]
    s = inputs.time_series(inputs.noise_spectrum(n, 9) + inputs.injection_spectrum(n, 2.0, 1.5, 10.0, 777), n).astype(np.float32)
    Sn = inputs.psd_array(n)
    for p in (1, 2, 32):
        w = inputs.Workload(config=-1, n=n, p=p, rho_thresh=5.5, window=n, masses=masses, seed=0)
        f = _run_gpu(gw, w, s, Sn, path=path)
        for t, (m1, m2) in enumerate(masses):
            rho_o, chi_o, _, _ = oracle.filter_template(s.astype(np.float64), Sn, m1, m2, p)
            rho_g, chi_g = f.series(t)
            parity.assert_series(rho_g, chi_g, rho_o, chi_o, p, f"p={p} template {t}")
            if p == 1:
                assert np.all(chi_g == 0.0)
    # (S_n, s) -> (c S_n, sqrt(c) s) leaves rho and chi^2 unchanged (P8), also at physical scales
    w = inputs.Workload(config=-1, n=n, p=8, rho_thresh=5.5, window=4096, masses=masses, seed=0)
    f1 = _run_gpu(gw, w, s, Sn, path=path)
    r1, c1 = f1.series(0)
    c = 9e-46
    f2 = _run_gpu(gw, w, (s.astype(np.float64) * math.sqrt(c)), Sn * c, path=path)
    r2, c2 = f2.series(0)
    assert np.max(np.abs(r1 - r2)) < 2e-4 and np.max(np.abs(c1 - c2) / np.maximum(c1, 1)) < 1e-3
    assert f2.sigma()[0] == pytest.approx(f1.sigma()[0] / math.sqrt(c), rel=1e-12)


def test_empty_bands_and_few_bins(gw, path):
    # a template that spans only a few dozen bins: with p = 32 most bands hold one bin and several are
    # empty (coinciding edges) -- their z_l must be exactly 0 in both pass-1 paths
    for log_n in (14, 15):           # n1 = 16: generic kernel only; n1 = 32: narrow kernel's empty-band path
        n = 1 << log_n
        masses = [(50.0, 50.0), (48.0, 45.0), (8.0, 8.0)]       # f_ISCO = 44.0 Hz, 47.3 Hz, 275 Hz
        s = inputs.time_series(inputs.noise_spectrum(n, 77) + inputs.injection_spectrum(n, 50.0, 50.0, 9.0, n // 2), n)
        s = s.astype(np.float32)
        Sn = inputs.psd_array(n)
        w = inputs.Workload(config=-1, n=n, p=32, rho_thresh=4.0, window=2048, masses=masses, seed=0)
        f = _run_gpu(gw, w, s, Sn, path=path)
        out = oracle.filter_bank(s.astype(np.float64), Sn, masses, 32, 2048, 4.0)
        parity.assert_sigma_edges(f.sigma(), f.band_edges(), out["sigma"], out["edges"])
        e = np.asarray(out["edges"])
        assert np.any(e[0, 1:] == e[0, :-1]), "this case is meant to have empty bands"
        for t, (m1, m2) in enumerate(masses):
            rho_o, chi_o, _, _ = oracle.filter_template(s.astype(np.float64), Sn, m1, m2, 32)
            rho_g, chi_g = f.series(t)
            parity.assert_series(rho_g, chi_g, rho_o, chi_o, 32, f"few-bin template {t}, n=2^{log_n}")
        parity.assert_triggers(f.triggers(), out, 4.0, 2048, 32)


def test_determinism_and_refilter(gw, path):
    w = inputs.workload(0)
    s = inputs.segment(w)
    f = _run_gpu(gw, w, s, w.psd, path=path)
    a = f.triggers().copy()
    r1, c1 = f.series(4)
    f.filter()                      # slots are reset, not accumulated
    b = f.triggers()
    r2, c2 = f.series(4)
    assert a.tobytes() == b.tobytes() and np.array_equal(r1, r2) and np.array_equal(c1, c2)
    f.filter(2, 3)                  # partial re-filter keeps the other templates' events
    assert f.triggers().tobytes() == a.tobytes()


def test_batching_invariance(gw, path):
    # the result must not depend on how the bank is cut into launches (double-buffered Q, side stream,
    # ragged last batch, partial filter calls)
    n = 1 << 17
    w1 = inputs.workload(1, 37)
    masses = w1.masses
    s = inputs.time_series(inputs.noise_spectrum(n, 5) + inputs.injection_spectrum(n, *masses[11], 10.0, 4242), n).astype(np.float32)
    Sn = inputs.psd_array(n)
    w = inputs.Workload(config=-1, n=n, p=16, rho_thresh=5.0, window=4096, masses=masses, seed=0)
    ref = _run_gpu(gw, w, s, Sn, batch=37, path=path).triggers().tobytes()
    for batch in (1, 5, 8, 36):
        f = _run_gpu(gw, w, s, Sn, batch=batch, path=path)
        assert f.triggers().tobytes() == ref, f"batch {batch}"
    f.filter(3, 20)                 # partial re-filter in ragged batches keeps the other templates' events
    f.filter(30, 7)
    assert f.triggers().tobytes() == ref


def test_error_codes(gw):
    assert gw.workspace_bytes(1000, 4, 8, 1) == 0             # n not a power of two
    assert gw.workspace_bytes(1 << 14, 0, 4096, 1) == 0       # p < 1
    assert gw.workspace_bytes(1 << 14, 4, 3000, 1) == 0       # window not a power of two
    f = gw.Filter(1 << 14, 4, 4096, 4)
    with pytest.raises(gw.GwmfError) as e:
        f.filter()
    assert e.value.status == gw.E_ARG or e.value.status == gw.E_STATE
    with pytest.raises(gw.GwmfError) as e:
        f.make_bank([(8.0, -1.0)])
    assert e.value.status == gw.E_ARG
    with pytest.raises(gw.GwmfError) as e:
        f.make_bank([(80.0, 80.0)])                            # f_ISCO = 27 Hz < 40 Hz
    assert e.value.status == gw.E_EMPTY_TEMPLATE
    with pytest.raises(gw.GwmfError) as e:
        f.make_bank([(8.0, 8.0)] * 5)                          # over capacity
    assert e.value.status == gw.E_ARG
    w = inputs.workload(0)
    f.make_bank(w.masses[:4])
    with pytest.raises(gw.GwmfError) as e:
        f.filter()
    assert e.value.status == gw.E_STATE
    s = inputs.segment(w)
    f.load_segment(s, w.psd)
    f.filter()
    with pytest.raises(gw.GwmfError) as e:
        f.triggers(capacity=0)                                 # config 0 has at least the injection's event
    assert e.value.status == gw.E_CAPACITY
    bad = w.psd.copy(); bad[500] = 0.0
    f.load_segment(s, bad)
    with pytest.raises(gw.GwmfError) as e:
        f.triggers()
    assert e.value.status == gw.E_ARG


def test_rejected_bank_leaves_the_old_bank_intact(gw, path):
    # gwmf_make_bank is failure-atomic: a bank that is refused half way (here its second template is empty) must not
    # disturb the loaded one, including the host mirror of k_high the correlate grid is trimmed with.  The filter of
    # templates 2, 3 in between leaves THEIR spectra in the buffers template 0 uses next, so a grid cut at the
    # rejected bank's smaller k_high would pick up foreign bins.
    n = 1 << 16
    masses = [(1.4, 1.4), (1.2, 1.0), (3.0, 1.2), (5.0, 5.0)]
    s = inputs.time_series(inputs.noise_spectrum(n, 31) + inputs.injection_spectrum(n, 1.4, 1.4, 9.0, 20000), n)
    f = gw.Filter(n, 8, 4096, 4, rho_thresh=4.0, batch=2, path=_path_for(path, n))
    f.make_bank(masses)
    f.load_segment(s.astype(np.float32), inputs.psd_array(n))
    f.filter()
    ref = f.triggers().copy()
    sig, edges = f.sigma().copy(), f.band_edges().copy()
    assert len(ref) > 8
    f.filter(2, 2)
    with pytest.raises(gw.GwmfError) as e:
        f.make_bank([(30.0, 30.0), (80.0, 80.0)])              # template 0 would get a far smaller k_high; template 1 is empty
    assert e.value.status == gw.E_EMPTY_TEMPLATE
    f.filter()
    assert f.triggers().tobytes() == ref.tobytes()
    assert np.array_equal(f.sigma(), sig) and np.array_equal(f.band_edges(), edges)


def test_effective_distance_matches_oracle(gw):
    # SURVEY.md 8(f)-4 / PAPER.md:21 (D_eff is one of the template's parameters): the distance at which each template has
    # optimal SNR 1 in the loaded PSD, D_1 = A(1 Mpc) sigma / sqrt(psd_unit), and D_eff = D_1 / rho of every event,
    # against the oracle's amplitude (O10) times the oracle's sigma, to 1e-5 relative (sigma's tolerance)
    w = inputs.workload(1)
    s = inputs.segment(w).astype(np.float32)
    f = _run_gpu(gw, w, s, w.psd)
    unit = 9e-46                                             # Eq. 2 as printed is the design curve / 9e-46
    C = oracle.power_table(w.psd, w.n)
    want = np.array([oracle.amplitude(m1, m2, 1.0) * oracle.sigma_edges(C, w.n, oracle.k_high(m1, m2, w.n), w.p)[0]
                     for m1, m2 in w.masses]) / math.sqrt(unit)
    d1 = f.effective_distance(unit)
    assert np.all(np.abs(d1 - want) <= 1e-5 * want)
    trig = f.triggers()
    assert len(trig) >= 3
    deff = f.trigger_distances(trig, unit)
    ref = want[trig["template_id"]] / trig["rho"].astype(np.float64)
    assert np.all(np.abs(deff - ref) <= 1e-5 * ref)
    assert np.allclose(f.effective_distance(1.0), d1 * math.sqrt(unit), rtol=1e-12)      # D_1 ~ 1 / sqrt(psd_unit)
    with pytest.raises(gw.GwmfError) as e:
        f.effective_distance(0.0)
    assert e.value.status == gw.E_ARG
    bad = trig[:1].copy()
    bad["template_id"] = len(w.masses)
    with pytest.raises(gw.GwmfError) as e:
        f.trigger_distances(bad, unit)
    assert e.value.status == gw.E_ARG


def test_no_triggers_when_threshold_is_high(gw):
    w = inputs.workload(0)
    f = _run_gpu(gw, w, inputs.segment(w), w.psd, thresh=50.0)
    assert len(f.triggers()) == 0


def test_device_resident_inputs(gw):
    import torch
    w = inputs.workload(0)
    s = inputs.segment(w).astype(np.float32)
    f = _run_gpu(gw, w, s, w.psd)
    a = f.triggers().copy()
    g = gw.Filter(w.n, w.p, w.window, len(w.masses), rho_thresh=w.rho_thresh)
    g.make_bank(w.masses)
    g.load_segment(torch.from_numpy(s).cuda(), torch.from_numpy(w.psd).cuda())
    g.filter()
    assert g.triggers().tobytes() == a.tobytes()
