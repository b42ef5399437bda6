"""Float64 CPU oracle for the LLOID hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this
module.  It shares no code with paper_2511_04730_b200/ (the CUDA path) and never imports it.

LLOID is an approximation of the time-domain matched filter (Eq. 1), so this oracle is
the ALGORITHM of PAPER.md Sec. II.C.2-3 (lines 121-193) followed step by step in float64, in the
paper's order and notation, with the readings of DESIGN.md "Readings of the paper".  `brute_force` is
Eq. 1 written out directly and is the exact oracle for the special case where the two coincide (all
slices at full rate, every singular value kept).

Parity pins (tests/test_oracle_*.py): every function below is pinned by something other
than itself -- hand-evaluated Eq. 4 values, zero-stuff+convolve (the textbook definition the polyphase
form replaces), closed-form tone gains, brute force on tiny inputs, the closed-form
injection inner product, causality, linearity, impulse response.  What is UNPINNED: absolute SNR values
against the paper -- the paper prints no numerical worked example of LLOID (Table I needs the O3 data).

Index conventions (all integer sample indices at the named rate; stream sample 0 is the first strain
sample; d[j] = 0 for j < 0; SNR sample k is the "coalescence at sample k" statistic and reads d[<=k]).
"""
from __future__ import annotations

import math
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

N_DOWN = 32   # PAPER.md:132 "typically set to 32 samples"
N_UP = 8      # PAPER.md:148 "set to 8 samples"


# --------------------------------------------------------------------------------------------------
# Eq. 4 -- sinc-windowed sinc kernel
# --------------------------------------------------------------------------------------------------
def resample_kernel(f: int, half_len: int) -> np.ndarray:
    """g[k] = sinc((k-c)/f) * sinc((k-c)/c), k = 0..2c, c = f*half_len, sinc(x) = sin(pi x)/(pi x); g[c] = 1."""
    c = f * half_len
    g = np.empty(2 * c + 1)
    for k in range(2 * c + 1):
        x = k - c
        if x == 0:
            g[k] = 1.0
        else:
            a = math.pi * x / f
            b = math.pi * x / c
            g[k] = (math.sin(a) / a) * (math.sin(b) / b)
    return g


# --------------------------------------------------------------------------------------------------
# O3 -- decimation to rate f0/D (readings 6, 8)
# --------------------------------------------------------------------------------------------------
class Series:
    """A sampled series x[j] for j in [j0, j0+len(v)); zero outside."""

    def __init__(self, v: np.ndarray, j0: int):
        self.v = np.asarray(v, dtype=np.float64)
        self.j0 = int(j0)

    def window(self, lo: int, hi: int) -> np.ndarray:
        """x[lo:hi] as a dense array (zero-filled outside the stored support)."""
        out = np.zeros(self.v.shape[:-1] + (hi - lo,))
        a = max(lo, self.j0)
        b = min(hi, self.j0 + self.v.shape[-1])
        if b > a:
            out[..., a - lo:b - lo] = self.v[..., a - self.j0:b - self.j0]
        return out


def decimate(d: np.ndarray, D: int, n_down: int = N_DOWN) -> Series:
    """d_r[j] = sqrt(D) * sum_k ghat[k] d[j D + c - k],  ghat = g/sum(g),  c = n_down*D  (zero phase).

    One filter per rate applied directly to the f0 stream (not cascaded).  Sample j of the output sits
    at f0-sample j*D and needs c future f0 samples; d is zero outside [0, len(d)).  Returned for
    j in [-n_down, ceil(len(d)/D) + n_down): everything that can be non-zero.
    """
    d = np.asarray(d, dtype=np.float64)
    if D == 1:
        return Series(d.copy(), 0)
    c = n_down * D
    g = resample_kernel(D, n_down)
    ghat = g / g.sum()
    j_lo = -n_down
    j_hi = -(-len(d) // D) + n_down
    pad = np.concatenate([np.zeros(2 * c), d, np.zeros(2 * c + D)])   # pad[i + 2c] = d[i]
    grev = ghat[::-1]          # sum_k ghat[k] d[jD + c - k] = sum_m ghat[2c - m] d[jD - c + m]
    # window j starts at f0-sample j*D - c, i.e. at pad index j*D + c; j_lo*D + c = 0
    W = np.lib.stride_tricks.sliding_window_view(pad, 2 * c + 1)[::D]
    out = np.empty(j_hi - j_lo)
    step = max(1, (1 << 24) // (2 * c + 1))          # rows per matmul: bounds the temporary copy
    for a in range(0, j_hi - j_lo, step):
        b = min(a + step, j_hi - j_lo)
        out[a:b] = math.sqrt(D) * (W[a:b] @ grev)
    return Series(out, j_lo)


# --------------------------------------------------------------------------------------------------
# O5 -- polyphase upsampler, zero-phase form (Eqs. 7-8; readings 9-11)
# --------------------------------------------------------------------------------------------------
def upsample_input_range(lo: int, hi: int, f: int, n_up: int = N_UP) -> Tuple[int, int]:
    """Input index range [lo', hi') needed to produce outputs [lo, hi) of `upsample`."""
    return lo // f - n_up, (hi - 1) // f + n_up + 1


def upsample(x: np.ndarray, x_lo: int, f: int, lo: int, hi: int, n_up: int = N_UP) -> np.ndarray:
    """(Up x)[i] = sum_{k=0}^{2 n_up} x[floor(i/f) + n_up - k] * g[k f + (i mod f)], g[. > 2c] = 0, c = n_up f.

    x[..., m] holds input sample x_lo + m along the last axis; outputs i in [lo, hi).  Phase 0
    (i mod f = 0) is the copy of Eq. 8 case 1 (g[k f] = delta_{k, n_up} analytically; floating-point
    sin(pi n) is ~1e-17, not 0, so the copy is written out).  The kernel is Eq. 4 with c = n_up*f and
    is NOT normalised.
    """
    g = resample_kernel(f, n_up)
    c = n_up * f
    out = np.zeros(x.shape[:-1] + (hi - lo,))
    i = np.arange(lo, hi)
    q = np.floor_divide(i, f)              # floor division, also for i < 0
    for j in range(f):                     # phase j: sub-kernel z_j[k] = g[k f + j]   (Eq. 7)
        sel = np.nonzero(i - q * f == j)[0]
        if sel.size == 0:
            continue
        if j == 0:                         # Eq. 8 case 1: y[i] = x[i/f] (g[k f] = delta_{k,n_up} analytically)
            m = q[sel] - x_lo
            assert m.min() >= 0 and m.max() < x.shape[-1], "upsample: input range too short"
            out[..., sel] = x[..., m]
            continue
        for k in range(2 * n_up + 1):
            t = k * f + j
            if t > 2 * c:
                continue
            m = q[sel] + n_up - k - x_lo
            assert m.min() >= 0 and m.max() < x.shape[-1], "upsample: input range too short"
            out[..., sel] += x[..., m] * g[t]
    return out


# --------------------------------------------------------------------------------------------------
# O4 -- basis correlation (Eq. 5) and reconstruction (Eq. 6) with the slice delay of Eq. 9
# --------------------------------------------------------------------------------------------------
def basis_correlate(U: np.ndarray, d_r: Series, delay: int, lo: int, hi: int, chunk: int = 4096) -> np.ndarray:
    """Y[l, j] = sum_{n<N} U[l, n] * d_r[j - delay - N + 1 + n]  for j in [lo, hi)   (Eq. 5,
    end-aligned and delayed by the slice delay t^s f^s).

    Columns are evaluated `chunk` at a time only to bound memory; every output is the plain sum.
    """
    L, N = U.shape
    Y = np.empty((L, hi - lo))
    for c0 in range(lo, hi, chunk):
        c1 = min(c0 + chunk, hi)
        seg = d_r.window(c0 - delay - N + 1, c1 - delay)          # length (c1-c0) + N - 1
        X = np.lib.stride_tricks.sliding_window_view(seg, N).T     # X[n, j-c0] = seg[(j-c0) + n]
        Y[:, c0 - lo:c1 - lo] = U @ X
    return Y


def reconstruct(R: np.ndarray, Y: np.ndarray) -> np.ndarray:
    """own[i, j] = sum_l R[i, l] Y[l, j],  R = V diag(sigma)   (Eq. 6)."""
    return R @ Y


# --------------------------------------------------------------------------------------------------
# the whole path: O3 -> O4 -> O5 for output samples [k_lo, k_hi) at f0
# --------------------------------------------------------------------------------------------------
def rate_groups(bank) -> List[Tuple[int, List[int]]]:
    """[(rate, [slice indices])] by decreasing rate; slices at one rate are summed before that rate's
    upsample stage (reading 12)."""
    groups: List[Tuple[int, List[int]]] = []
    for s, sl in enumerate(bank.slices):
        if groups and groups[-1][0] == sl.rate:
            groups[-1][1].append(s)
        else:
            assert not groups or sl.rate < groups[-1][0], "rates must not increase with s"
            groups.append((sl.rate, [s]))
    return groups


def lloid_snr(bank, strain: np.ndarray, k_lo: int = 0, k_hi: Optional[int] = None,
              rows: Optional[Sequence[int]] = None, n_down: int = N_DOWN, n_up: int = N_UP,
              decimated: Optional[Dict[int, Series]] = None) -> np.ndarray:
    """rho^0[rows, k_lo:k_hi]: the 2M real SNR series at f0 (Eq. 9, Fig. 4).

    From the lowest rate up: rho^g = sum_{s in group g} R^s Y^s  +  Up_f(rho^{g+1}), f = rate_g/rate_{g+1}
    (one stage to the next rate PRESENT in the bank, reading 10).  Each lower-rate stream is
    evaluated over exactly the index range the stage above needs (n_up extra samples on both sides),
    which is possible ahead of time because slice s is delayed by t^s.
    """
    strain = np.asarray(strain, dtype=np.float64)
    k_hi = len(strain) if k_hi is None else k_hi
    groups = rate_groups(bank)
    f0 = bank.f0
    assert groups[0][0] == f0, "slice 0 must run at the strain rate"
    # index range needed at every group
    ranges = [(k_lo, k_hi)]
    for g in range(1, len(groups)):
        f = groups[g - 1][0] // groups[g][0]
        ranges.append(upsample_input_range(ranges[-1][0], ranges[-1][1], f, n_up))
    if decimated is None:
        decimated = {}
    rho = None
    for g in range(len(groups) - 1, -1, -1):
        rate, members = groups[g]
        lo, hi = ranges[g]
        D = f0 // rate
        if D not in decimated:
            decimated[D] = decimate(strain, D, n_down)
        acc = None
        for s in members:
            sl = bank.slices[s]
            R = sl.R if rows is None else sl.R[list(rows)]
            own = reconstruct(R, basis_correlate(sl.U, decimated[D], sl.delay, lo, hi))
            acc = own if acc is None else acc + own
        if rho is not None:
            f = rate // groups[g + 1][0]
            acc = acc + upsample(rho, ranges[g + 1][0], f, lo, hi, n_up)
        rho = acc
    return rho


# --------------------------------------------------------------------------------------------------
# Eq. 1 written out (exact oracle for the no-downsampling, full-rank special case)
# --------------------------------------------------------------------------------------------------
def brute_force(H: np.ndarray, strain: np.ndarray, k_lo: int = 0, k_hi: Optional[int] = None) -> np.ndarray:
    """x_i[k] = sum_m h_i[m] d[k - (N-1) + m]   (Eq. 1; discrete, no factor 2, reading 1)."""
    strain = np.asarray(strain, dtype=np.float64)
    k_hi = len(strain) if k_hi is None else k_hi
    N = H.shape[1]
    seg = Series(strain, 0).window(k_lo - (N - 1), k_hi)
    out = np.empty((H.shape[0], k_hi - k_lo))
    for i in range(H.shape[0]):
        out[i] = np.correlate(seg, H[i], mode="valid")    # [k] = sum_m seg[k+m] h[m]
    return out


# --------------------------------------------------------------------------------------------------
# O6 -- per-buffer peaks (integer sample, no interpolation: PAPER.md:307)
# --------------------------------------------------------------------------------------------------
def find_peaks(rho: np.ndarray, buffer_len: int):
    """For every complex template j (rows 2j, 2j+1) and every buffer of `buffer_len` samples:
    first k maximising rho_2j^2 + rho_2j+1^2; returns (snr [n_buf][M], sample [n_buf][M] within the
    buffer, phase [n_buf][M] = atan2(rho_2j+1, rho_2j) at the maximum)."""
    M = rho.shape[0] // 2
    n_buf = rho.shape[1] // buffer_len
    snr = np.empty((n_buf, M))
    idx = np.empty((n_buf, M), dtype=np.int64)
    ph = np.empty((n_buf, M))
    for b in range(n_buf):
        blk = rho[:, b * buffer_len:(b + 1) * buffer_len]
        re, im = blk[0::2], blk[1::2]
        p = re * re + im * im
        k = np.argmax(p, axis=1)             # numpy: "the first occurrence is returned" -> lowest index
        j = np.arange(M)
        snr[b] = np.sqrt(p[j, k])
        idx[b] = k
        ph[b] = np.arctan2(im[j, k], re[j, k])
    return snr, idx, ph
