"""TEST INFRASTRUCTURE -- plain float64 oracle of the event-identification steps that follow the LLOID hot path
(Sec. II.D: 199-221, Fig. 5, Eq. 10).  Like lloid_oracle.py it shares no code with the
CUDA path and only tests/, __graft_entry__.smoke() and bench.py's oracle legs may import it.

    find_peaks_overlap   trigger windows of one buffer plus the overlap that precedes it      (Fig. 5)
    template_acorr       complex template autocorrelation R_j(t), R_j(0) = 1
    xi2                  signal-based consistency statistic of one trigger, Eq. 10
    coincidences         per template: the loudest set of mutually coincident triggers
    cluster              per bank: the one event with the highest network SNR

Readings (numbers 19-24): integrals are sums over integer samples (dt cancels in Eq. 10); the
window of Eq. 10 is t = -delta..delta samples, delta = (autocorrelation length - 1) / 2; z_j(0) is the complex SNR at
the trigger sample; a trigger whose window leaves the available SNR series uses zeros there (stream start) -- the
streaming implementation delays the statistic instead ("contributes to the overall pipeline latency");
coincidence is between triggers of the SAME template, a set of detectors is coincident when EVERY pair is within its
window dt[a][b] (light travel time + 0.005 s, in samples, inclusive); network SNR = sqrt(sum snr^2); ties -> the set
listed first in ascending bit-mask order / the lowest template index.
"""
from __future__ import annotations

import itertools
import math
from typing import List, Optional, Sequence, Tuple

import numpy as np


def find_peaks_overlap(rho: np.ndarray, buffer_len: int, overlap: int):
    """Per trigger window n = 0, 1, ...: window = samples [n*B - overlap, (n+1)*B) (the first one starts at 0; Fig. 5:
    "the first window is shortened").  Returns (snr [n][M], sample [n][M] RELATIVE to n*B -- negative inside the
    overlap --, phase [n][M]); first maximum of |z|^2."""
    rho = np.asarray(rho, dtype=np.float64)
    z = rho[0::2] + 1j * rho[1::2]
    M, n = z.shape
    nwin = n // buffer_len
    snr = np.zeros((nwin, M)); idx = np.zeros((nwin, M), dtype=np.int64); ph = np.zeros((nwin, M))
    for w in range(nwin):
        lo = max(0, w * buffer_len - overlap)
        p = np.abs(z[:, lo:(w + 1) * buffer_len]) ** 2
        k = np.argmax(p, axis=1)                      # numpy argmax returns the first maximum
        zz = z[np.arange(M), lo + k]
        snr[w] = np.sqrt(p[np.arange(M), k]); idx[w] = lo + k - w * buffer_len; ph[w] = np.angle(zz)
    return snr, idx, ph


def template_acorr(h_cos: np.ndarray, h_sin: np.ndarray, delta: int) -> np.ndarray:
    """R[t + delta] = sum_m g[m] conj(g[m + t]) / sum_m |g[m]|^2 for t = -delta..delta, g = h_cos + i h_sin: what the
    complex matched filter z[k] = sum_m g[m] d[k - N + 1 + m] returns t samples after the peak for its own template
    (d = Re(conj(a) g) gives z[k0 + t] = a R[t] up to the template's negative-frequency content), normalised so that
    R(0) = 1 exactly."""
    g = np.asarray(h_cos, dtype=np.float64) + 1j * np.asarray(h_sin, dtype=np.float64)
    N = len(g)
    norm = np.sum(np.abs(g) ** 2)
    R = np.zeros(2 * delta + 1, dtype=np.complex128)
    for t in range(-delta, delta + 1):
        if t >= 0:
            R[t + delta] = np.sum(g[:N - t] * np.conj(g[t:])) if t < N else 0.0
        else:
            R[t + delta] = np.sum(g[-t:] * np.conj(g[:N + t])) if -t < N else 0.0
    return R / norm


def xi2(z: np.ndarray, k0: int, acorr: np.ndarray) -> float:
    """Eq. 10 with sums for integrals: sum_t |z[k0 + t] - z[k0] R[t]|^2 / sum_t (2 - 2 |R[t]|^2), t = -delta..delta.
    z: complex SNR series of one template; samples outside [0, len(z)) count as zero."""
    acorr = np.asarray(acorr, dtype=np.complex128)
    delta = (len(acorr) - 1) // 2
    seg = np.zeros(2 * delta + 1, dtype=np.complex128)
    lo, hi = k0 - delta, k0 + delta + 1
    a, b = max(lo, 0), min(hi, len(z))
    if b > a:
        seg[a - lo:b - lo] = z[a:b]
    num = np.sum(np.abs(seg - z[k0] * acorr) ** 2)
    den = np.sum(2.0 - 2.0 * np.abs(acorr) ** 2)
    return float(num / den)


def coincidences(snr: np.ndarray, sample: np.ndarray, dt: np.ndarray, threshold: float):
    """Coincidence formation for ONE trigger window.

    snr, sample: [n_det][M] single-detector triggers of the window (sample = integer trigger time in f0 samples on a
    clock common to all detectors); dt: [n_det][n_det] symmetric coincidence windows in samples (light travel time +
    0.005 s, rounded up); a trigger exists where snr >= threshold.
    Per template: among all detector sets S with |S| >= 2 in which EVERY pair (a, b) has |sample_a - sample_b| <= dt[a][b],
    the one with the largest network SNR^2 = sum_{a in S} snr_a^2 (ties: the smaller bit mask).  Returns
    (mask [M] int -- bit a set for a participating detector, 0 = no coincidence --, net_snr [M])."""
    snr = np.asarray(snr, dtype=np.float64)
    sample = np.asarray(sample, dtype=np.int64)
    n_det, M = snr.shape
    mask = np.zeros(M, dtype=np.int64)
    net = np.zeros(M)
    subsets = [s for r in range(2, n_det + 1) for s in itertools.combinations(range(n_det), r)]
    subsets.sort(key=lambda s: sum(1 << a for a in s))
    for j in range(M):
        best, best_mask = 0.0, 0
        for s in subsets:
            if any(snr[a, j] < threshold for a in s):
                continue
            if any(abs(int(sample[a, j]) - int(sample[b, j])) > dt[a][b] for a, b in itertools.combinations(s, 2)):
                continue
            v = sum(snr[a, j] ** 2 for a in s)
            if v > best:
                best, best_mask = v, sum(1 << a for a in s)
        mask[j], net[j] = best_mask, math.sqrt(best)
    return mask, net


def cluster(mask: np.ndarray, net: np.ndarray, bank_off: Sequence[int]):
    """Clustering: within each bank keep only the coincident event with the highest network SNR of the
    window (ties: the lowest template index).  bank_off: [n_banks + 1] template offsets.  Returns per bank
    (template index within the stream or -1, mask, net_snr)."""
    out = []
    for b in range(len(bank_off) - 1):
        lo, hi = bank_off[b], bank_off[b + 1]
        best, arg = 0.0, -1
        for j in range(lo, hi):
            if mask[j] != 0 and net[j] > best:
                best, arg = net[j], j
        out.append((arg, int(mask[arg]) if arg >= 0 else 0, float(best)))
    return out
