"""TEST INFRASTRUCTURE -- plain float64 oracle of the PSD estimation + whitening front end that precedes the LLOID path
(Sec. II.B.2, lines 63-81, Figs. 2-3).  numpy only; shares no code with the CUDA path.

Algorithm, per detector, one ITERATION per hop = N/2 - Z new input samples at rate f_in:
  1. block = [0]*Z ++ hann(N - 2Z) * (the newest N - 2Z input samples) ++ [0]*Z          (length N; zero history at start)
  2. X = rfft(block)
  3. instantaneous PSD  P[k] = 2 |X[k]|^2 / (f_in * sum(hann^2))                          (one-sided, per Hz)
  4. med[k] = median of the most recent m P[k], m = the largest odd number <= min(count, n_med);  running geometric
     mean of the single-block estimates  g[k] = med[k] exp(-c(m) - gamma):  logG <- ((n - 1) logG + log g) / n,
     n = min(count, n_avg);  PSD S[k] = exp(logG[k] + gamma).  c(m) = E log(median of m unit-mean exponential variates)
     is "the constant factor" that turns a median of chi^2_2-distributed PSD bins into their geometric mean
     (exp(-gamma) times the mean) and exp(gamma) turns that into the arithmetic mean
  5. frequency-domain downsampling: keep bins k <= N_out / 2, N_out = N f_out / f_in      (Fig. 3)
     W[k] = X[k] * sqrt(2 / (f_in * S[k])) * sqrt(f_in / f_out)   (k = 0 and the new Nyquist bin are set to 0;
     the last factor restores unit variance after the band is cut to f_out / f_in of its width)
  6. w = irfft(W, N_out) * N_out / N;  w *= tukey(N_out, taper = Z_out on each side)
  7. overlap-add w into the accumulator; its first hop_out = N_out/2 - Z_out samples are final output; shift.
The output lags the input by N/2 input samples.

Readings (numbers 25-30): the PSD of step 5 is the one already updated with the current block
("the latest PSD", Fig. 3); Hann is the periodic window hann[i] = 0.5 - 0.5 cos(2 pi i / L), L = N - 2Z, whose copies
shifted by L/2 sum to exactly 1; the Tukey window has cosine tapers of Z_out samples at both ends and is 1 between;
the normalisation of step 5 gives unit variance at f_out for a stationary Gaussian input of ANY variance or colour;
during start-up the median runs over an odd number of blocks (1, 1, 3, 3, 5, 5, 7, ...); gaps and gating are not
modelled.
"""
from __future__ import annotations

import functools
import math
from typing import List, Optional

import numpy as np

EULER_GAMMA = 0.5772156649015329


@functools.lru_cache(maxsize=None)
def log_median_mean(m: int) -> float:
    """c(m) = E log X_(k), k = (m + 1) / 2, the median of m (odd) iid unit-mean exponential variates; density of the k-th
    order statistic: m! / ((k-1)! (m-k)!) (1 - e^-x)^(k-1) e^(-x (m-k+1)).  scipy quadrature."""
    from scipy.integrate import quad
    assert m % 2 == 1
    k = (m + 1) // 2
    cst = math.factorial(m) / (math.factorial(k - 1) * math.factorial(m - k))
    f = lambda x: math.log(x) * cst * (1.0 - math.exp(-x)) ** (k - 1) * math.exp(-x * (m - k + 1))
    a, _ = quad(f, 0.0, 1.0, epsabs=1e-13, epsrel=1e-13)
    b, _ = quad(f, 1.0, 60.0, epsabs=1e-13, epsrel=1e-13)
    return a + b


def hann_periodic(L: int) -> np.ndarray:
    return 0.5 - 0.5 * np.cos(2.0 * np.pi * np.arange(L) / L)


def tukey_taper(n: int, taper: int) -> np.ndarray:
    """1 in the middle, half-cosine ramps of `taper` samples at both ends: w[i] = 0.5 (1 - cos(pi (i + 0.5) / taper))."""
    w = np.ones(n)
    if taper > 0:
        ramp = 0.5 * (1.0 - np.cos(np.pi * (np.arange(taper) + 0.5) / taper))
        w[:taper] = ramp
        w[n - taper:] = ramp[::-1]
    return w


class Whitener:
    """One detector.  push(hop_in samples) -> hop_out whitened samples (unit variance at f_out)."""

    def __init__(self, f_in: int, f_out: int, N: int, Z: int, n_med: int = 7, n_avg: int = 64):
        assert f_in % f_out == 0 and N % 2 == 0 and (N - 2 * Z) % 2 == 0 and (N * f_out) % f_in == 0 and (Z * f_out) % f_in == 0
        self.f_in, self.f_out, self.N, self.Z, self.n_med, self.n_avg = f_in, f_out, N, Z, n_med, n_avg
        self.L = N - 2 * Z
        self.hop = N // 2 - Z
        self.N_out, self.Z_out = N * f_out // f_in, Z * f_out // f_in
        self.hop_out = self.N_out // 2 - self.Z_out
        self.hann = hann_periodic(self.L)
        self.tukey = tukey_taper(self.N_out, self.Z_out)
        self.segment = np.zeros(self.L)
        self.acc = np.zeros(self.N_out)
        self.history: List[np.ndarray] = []
        self.logG: Optional[np.ndarray] = None
        self.count = 0
        self.psd = None

    def push(self, x: np.ndarray) -> np.ndarray:
        x = np.asarray(x, dtype=np.float64)
        assert len(x) == self.hop
        self.segment = np.concatenate([self.segment[self.hop:], x])
        block = np.concatenate([np.zeros(self.Z), self.hann * self.segment, np.zeros(self.Z)])
        X = np.fft.rfft(block)
        nb = self.N_out // 2 + 1
        P = 2.0 * np.abs(X[:nb]) ** 2 / (self.f_in * np.sum(self.hann ** 2))
        self.history = (self.history + [P])[-self.n_med:]
        self.count += 1
        m = min(self.count, self.n_med)
        m -= 1 - m % 2                                  # largest odd number <= min(count, n_med)
        med = np.median(np.stack(self.history[-m:]), axis=0)
        with np.errstate(divide="ignore"):
            logg = np.log(med) - log_median_mean(m) - EULER_GAMMA
        n = min(self.count, self.n_avg)
        self.logG = logg if self.logG is None else ((n - 1) * self.logG + logg) / n
        S = np.exp(self.logG + EULER_GAMMA)
        self.psd = S
        W = np.zeros(nb, dtype=np.complex128)
        ok = S > 0
        W[ok] = X[:nb][ok] * np.sqrt(2.0 / (self.f_in * S[ok])) * math.sqrt(self.f_in / self.f_out)
        W[0] = 0.0
        W[-1] = 0.0
        w = np.fft.irfft(W, self.N_out) * (self.N_out / self.N) * self.tukey
        self.acc += w
        out = self.acc[:self.hop_out].copy()
        self.acc = np.concatenate([self.acc[self.hop_out:], np.zeros(self.hop_out)])
        return out
