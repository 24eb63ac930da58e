"""Pins of the t -> f transform oracle (oracle/tf_oracle.py) against things other
than itself: a library FFT, closed forms, and the inverse relation used by the data recipe."""
import numpy as np
import pytest

import oracle


def test_matches_library_rfft_on_random_section():
    rng = np.random.default_rng(1)
    nt, nx = 96, 7
    d = rng.standard_normal((nt, nx))
    bins = np.array([0, 1, 5, 17, 40, 48])
    want = np.fft.rfft(d, axis=0)[bins]                     # numpy's sign: exp(-2 pi i j n / nt)
    got = oracle.section_to_fx(d, bins)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-11)


def test_cosine_closed_form():
    nt, nx, j0, A, phi = 128, 3, 9, 2.5, 0.7
    n = np.arange(nt)[:, None]
    d = A * np.cos(2 * np.pi * j0 * n / nt + phi) * np.ones((1, nx))
    bins = np.arange(0, nt // 2 + 1)
    got = oracle.section_to_fx(d, bins)
    want = np.zeros((bins.size, nx), dtype=complex)
    want[j0] = A * nt / 2 * np.exp(1j * phi)                # the e^{+i(wt+phi)} half of the cosine
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-10)


def test_delta_gives_pure_phase_with_negative_sign():
    nt, n0 = 64, 5
    d = np.zeros((nt, 2)); d[n0, 0] = 1.0; d[0, 1] = 3.0
    bins = np.array([0, 1, 2, 31, 32])
    got = oracle.section_to_fx(d, bins)
    np.testing.assert_allclose(got[:, 0], np.exp(-2j * np.pi * bins * n0 / nt), atol=1e-13)
    np.testing.assert_allclose(got[:, 1], 3.0 + 0j, atol=1e-13)


def test_inverts_the_synthesis_used_by_the_input_recipe():
    """P0(w,x) = R(w) e^{-i w t0} synthesised to a real trace (irfft) comes back unchanged."""
    nt, dt = 256, 0.004
    j = np.arange(nt // 2 + 1)
    w = 2 * np.pi * j / (nt * dt)
    spec = np.exp(-((w / (2 * np.pi) - 20.0) / 8.0) ** 2) * np.exp(-1j * w * 0.3)
    spec[0] = 0; spec[-1] = 0
    trace = np.fft.irfft(spec, n=nt) * nt                   # d[n] = sum over +-w of P e^{+iwt}
    bins = np.arange(5, 60)
    got = oracle.section_to_fx(trace[:, None], bins)[:, 0]
    np.testing.assert_allclose(got, spec[bins] * nt, rtol=0, atol=1e-9 * nt)


def test_linearity_and_bin_selection_order():
    rng = np.random.default_rng(3)
    a, b = rng.standard_normal((50, 4)), rng.standard_normal((50, 4))
    bins = np.array([7, 3, 25, 3])
    lhs = oracle.section_to_fx(2 * a - 3 * b, bins)
    rhs = 2 * oracle.section_to_fx(a, bins) - 3 * oracle.section_to_fx(b, bins)
    np.testing.assert_allclose(lhs, rhs, atol=1e-12)
    np.testing.assert_array_equal(lhs[1], lhs[3])           # repeated bin, any order


def test_rejects_bins_outside_the_real_spectrum():
    with pytest.raises(ValueError):
        oracle.section_to_fx(np.zeros((16, 2)), np.array([9]))
