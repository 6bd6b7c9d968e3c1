"""Seeded input generators: determinism, the noise normalisation and the bank enumerations."""
import math

import numpy as np
import pytest

import workloads as inputs


def test_rng_is_a_pure_function_of_its_coordinates():
    a = inputs.normal(3, 0, np.arange(1000))
    b = inputs.normal(3, 0, np.arange(1000)[::-1])[::-1]
    assert np.array_equal(a, b)
    assert not np.array_equal(a, inputs.normal(3, 1, np.arange(1000)))
    assert not np.array_equal(a, inputs.normal(4, 0, np.arange(1000)))
    u = inputs.uniform01(1, 2, np.arange(200000))
    assert 0.0 < u.min() and u.max() < 1.0 and abs(u.mean() - 0.5) < 3e-3
    z = inputs.normal(9, 0, np.arange(400000))
    assert abs(z.mean()) < 6e-3 and abs(z.var() - 1.0) < 1e-2
    assert abs(np.mean(z ** 4) - 3.0) < 0.06


def test_noise_variance_is_the_integral_of_the_psd():
    n = 1 << 16
    s = inputs.time_series(inputs.noise_spectrum(n, 5), n)
    assert np.var(s) == pytest.approx(42481.4, rel=0.05)
    D = np.fft.rfft(s)
    assert np.all(np.abs(D[:inputs.F_LOW.__int__() * n // 4096]) < 1e-6)      # nothing below 40 Hz
    assert abs(D[n // 2]) < 1e-6


def test_injection_lands_at_t_c():
    n = 1 << 14
    s = inputs.time_series(inputs.injection_spectrum(n, 8, 8, 12.0, 9000), n)
    assert int(np.argmax(np.abs(s))) in range(8940, 9001)                    # chirp ends at t_c


def test_banks():
    b0 = inputs.bank(0)
    assert b0 == [(6, 6), (6, 8), (6, 10), (6, 12), (8, 8), (8, 10), (8, 12), (10, 10)]
    b1 = inputs.bank(1)
    assert len(b1) == 256 and all(1.0 <= m2 <= m1 <= 3.0 for m1, m2 in b1)
    b2 = inputs.bank(2)
    assert len(b2) == 1024
    for m1, m2 in b2:
        assert m1 >= m2 >= 1.0 - 1e-9 and 2.0 - 1e-9 <= m1 + m2 <= 34.0 + 1e-9
    assert len(inputs.bank(3)) == 4096
    b4 = inputs.bank(4)
    assert len(b4) == 512 and all(1.0 <= m2 <= m1 <= 2.0 for m1, m2 in b4)
    # chirp mass uniform at fixed eta (first row of the config-2 grid)
    row = b2[:32]
    mc = [(a * b) ** 0.6 / (a + b) ** 0.2 for a, b in row]
    assert np.allclose(np.diff(mc), np.diff(mc)[0], rtol=1e-9)


def test_workloads():
    for c, (n, p) in {0: (1 << 14, 4), 1: (1 << 18, 16), 2: (1 << 20, 16), 3: (1 << 20, 16), 4: (1 << 22, 32)}.items():
        w = inputs.workload(c)
        assert (w.n, w.p) == (n, p)
        for (b, m1, m2, snr, jc) in w.injections:
            assert 8.0 <= snr <= 15.0
    assert inputs.workload(4).rho_thresh == 5.5
    w3 = inputs.workload(3)
    assert w3.n_segments == 15 and w3.stream_len == 1 << 23
