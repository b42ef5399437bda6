"""CPU pins of oracle/whiten_oracle.py (PSD estimation + whitening) against closed forms and statistics."""
import math

import numpy as np

from oracle import Whitener, hann_periodic, log_median_mean, tukey_taper
from oracle.whiten_oracle import EULER_GAMMA


def test_windows():
    L = 64
    h = hann_periodic(L)
    assert np.allclose(h[:L // 2] + h[L // 2:], 1.0, atol=1e-15)       # copies shifted by L/2 sum to one
    assert h[0] == 0.0 and math.isclose(h[L // 2], 1.0)
    t = tukey_taper(40, 8)
    assert np.all(t[8:32] == 1.0) and np.allclose(t[:8], t[::-1][:8]) and 0 < t[0] < t[7] < 1
    assert np.allclose(t[:8] + t[:8][::-1], 1.0)                       # complementary ramps


def test_median_constant_closed_form_and_monte_carlo():
    assert math.isclose(log_median_mean(1), -EULER_GAMMA, abs_tol=1e-10)   # E log of an exponential variate = -gamma
    rng = np.random.default_rng(2)
    for m in (3, 5, 7):
        x = np.median(rng.exponential(size=(400000, m)), axis=1)
        assert abs(np.log(x).mean() - log_median_mean(m)) < 4e-3
    assert log_median_mean(7) > log_median_mean(3) > log_median_mean(1)


def _run(w, x):
    return np.concatenate([w.push(x[i * w.hop:(i + 1) * w.hop]) for i in range(len(x) // w.hop)])


def test_white_noise_of_any_variance_comes_out_with_unit_variance():
    f_in, f_out = 4096, 1024
    rng = np.random.default_rng(0)
    for sig in (0.01, 3.7):
        w = Whitener(f_in, f_out, f_in, f_in // 4)
        o = _run(w, sig * rng.standard_normal(300 * w.hop))[80 * w.hop_out:]
        assert abs(o.var() - 1.0) < 0.03
        k = np.arange(5, w.N_out // 2 - 5)
        assert abs((w.psd[k] * f_in / 2 / sig ** 2).mean() - 1.0) < 0.03   # one-sided PSD of white noise = 2 sigma^2 / f_in


def test_coloured_noise_is_flattened_and_its_psd_recovered():
    from scipy.signal import lfilter
    f_in, f_out = 4096, 1024
    rng = np.random.default_rng(1)
    w = Whitener(f_in, f_out, f_in, f_in // 4)
    a = 0.9
    x = lfilter([1.0], [1.0, -a], rng.standard_normal(400 * w.hop))
    o = _run(w, x)[100 * w.hop_out:]
    assert abs(o.var() - 1.0) < 0.04
    F = (np.abs(np.fft.rfft(o[:len(o) // 1024 * 1024].reshape(-1, 1024) * np.hanning(1024), axis=1)) ** 2).mean(axis=0)
    band = F[20:480].reshape(-1, 46).mean(axis=1)
    assert band.max() / band.min() < 1.25                               # flat (the input spans a factor 360 here)
    k = np.arange(10, w.N_out // 2 - 10)
    fr = k * f_in / w.N
    truth = 2.0 / f_in / np.abs(1 - a * np.exp(-2j * np.pi * fr / f_in)) ** 2
    assert abs(np.mean(w.psd[k] / truth) - 1.0) < 0.04


def test_output_lags_the_input_by_half_an_fft_block():
    """the output lags the input by N/2 input samples: the cross-correlation of the band-limited input with
    the output peaks at a lag of N_out / 2 output samples."""
    f_in, f_out = 4096, 1024
    rng = np.random.default_rng(4)
    w = Whitener(f_in, f_out, f_in, f_in // 4)
    x = rng.standard_normal(120 * w.hop)
    o = _run(w, x)
    X = np.fft.rfft(x)
    n_out = len(x) * f_out // f_in
    xd = np.fft.irfft(X[:n_out // 2 + 1], n_out) * n_out / len(x)       # ideal band-limited copy at f_out
    a, b = xd[40 * w.hop_out:100 * w.hop_out], o[40 * w.hop_out:]
    lags = range(w.N_out // 2 - 6, w.N_out // 2 + 7)
    cc = [np.dot(a, b[l:l + len(a)]) for l in lags]
    assert list(lags)[int(np.argmax(cc))] == w.N_out // 2
    assert max(cc) / len(a) > 0.45                                       # sqrt(f_in / f_out) * var(xd) = 0.5: same waveform
