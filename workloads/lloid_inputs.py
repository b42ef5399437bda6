"""Seeded synthetic LLOID workloads: chirp templates, slice layouts, SVD banks, strain, injections.

Everything here produces INPUTS of the hot path; nothing here resamples,
filters, reconstructs or searches peaks.  The SVD bank is the "pregenerated SVD bank" the paper's
filtering stage consumes (Fig. 1 caption, Sec. II.C.1, Eq. 3) and is the
argument of ``lloid_bank_create``; building it is an offline, untimed step.

Conventions:
  * strain rate f0 = 2048 Hz; a template has N = T*f0 real samples h[m], m = 0..N-1, the LAST sample
    is the merger; ``a = N-1-m`` counts f0-samples before the merger, tau = a/f0.
  * real rows are interleaved: row 2j = cosine quadrature, row 2j+1 = sine quadrature.
  * slice s covers a in [B_s, E_s), B_0 = 0, B_{s+1} = E_s; rate f^s = f0/D_s; its low-rate template is
    the analytic chirp sampled every D_s-th f0 sample, times sqrt(D_s) (keeps unit variance per rate).
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional, Sequence, Tuple

import numpy as np

MTSUN_S = 4.925490947e-6  # G*Msun/c^3 in seconds
F0_HZ = 2048


# --------------------------------------------------------------------------------------------------
# containers
# --------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Slice:
    rate: int          # f^s in Hz (power of two, divides f0)
    n_taps: int        # N^s, samples at `rate`
    delay: int         # t^s * rate: samples (at `rate`) between the merger and this slice's newest tap
    U: np.ndarray      # [L^s][N^s] orthonormal rows, oldest tap first        (Eq. 3 u_l^s[k])
    R: np.ndarray      # [2M][L^s]  = V diag(sigma)                           (Eq. 6 sigma_l nu_il)
    kept_energy: float = 1.0   # sum_{l<L} sigma_l^2 / sum sigma_l^2

    @property
    def n_basis(self) -> int:
        return int(self.U.shape[0])


@dataclasses.dataclass
class Bank:
    f0: int
    M: int                     # complex templates; 2M real rows
    slices: List[Slice]
    mchirp: Optional[np.ndarray] = None   # [M] chirp masses (Msun) when the bank is a chirp bank
    T: Optional[float] = None             # template length in seconds

    def as_f32(self) -> "Bank":
        """Same bank with U and R rounded to float32 (what the C ABI takes), held as float64."""
        sl = [dataclasses.replace(s, U=s.U.astype(np.float32).astype(np.float64),
                                  R=s.R.astype(np.float32).astype(np.float64)) for s in self.slices]
        return dataclasses.replace(self, slices=sl)

    def describe(self) -> str:
        return " ".join(f"{s.rate}x{s.n_taps}(L{s.n_basis})" for s in self.slices)


@dataclasses.dataclass
class Injection:
    bank: int
    template: int      # complex template index j in the bank
    det: int
    k0: int            # stream sample (at f0) of the template's last sample = coalescence sample
    amp: float         # A
    phase: float       # phi


# --------------------------------------------------------------------------------------------------
# Newtonian chirps (BASELINE.json configs: f(t) ~ (tc-t)^(-3/8), Tukey taper, unit norm, flat PSD)
# --------------------------------------------------------------------------------------------------
def chirp_frequency(tau, mc):
    """GW frequency (Hz) at time `tau` (s) before merger for chirp mass `mc` (Msun)."""
    tau = np.asarray(tau, dtype=np.float64)
    with np.errstate(divide="ignore"):
        return (1.0 / math.pi) * (5.0 / (256.0 * tau)) ** 0.375 * (mc * MTSUN_S) ** (-0.625)


def chirp_time_to_merger(f, mc):
    """Inverse of chirp_frequency: tau (s) at which the chirp passes frequency f (Hz)."""
    return (5.0 / 256.0) * (math.pi * f) ** (-8.0 / 3.0) * (mc * MTSUN_S) ** (-5.0 / 3.0)


def _tukey(p, n, alpha=1.0 / 16.0):
    """Tukey window value at positions p (0..n-1) of an n-point window."""
    p = np.asarray(p, dtype=np.float64)
    if n < 2:
        return np.ones_like(p)
    x = p / (n - 1.0)
    w = np.ones_like(x)
    lo = x < alpha / 2
    hi = x > 1 - alpha / 2
    w[lo] = 0.5 * (1 + np.cos(math.pi * (2 * x[lo] / alpha - 1)))
    w[hi] = 0.5 * (1 + np.cos(math.pi * (2 * x[hi] / alpha - 2 / alpha + 1)))
    return w


def _chirp_quadratures(mc, a, N, f0, f_max):
    """Unnormalised windowed (cos, sin) chirp values at samples-before-merger `a` (array, 0 <= a < N)."""
    a = np.asarray(a, dtype=np.float64)
    a0 = int(math.floor(chirp_time_to_merger(f_max, mc) * f0)) + 1   # first a with f(tau) <= f_max
    a0 = max(a0, 1)
    n_sup = N - a0
    c = np.zeros(a.shape)
    s = np.zeros(a.shape)
    ok = (a >= a0) & (a <= N - 1)
    if n_sup < 2 or not ok.any():
        return c, s
    tau = a[ok] / f0
    ph = -2.0 * (tau / (5.0 * mc * MTSUN_S)) ** 0.625
    amp = tau ** (-0.25) * _tukey(a[ok] - a0, n_sup)
    c[ok] = amp * np.cos(ph)
    s[ok] = amp * np.sin(ph)
    return c, s


def _chirp_norms(mc, N, f0, f_max):
    c, s = _chirp_quadratures(mc, np.arange(N), N, f0, f_max)
    return math.sqrt(float(c @ c)), math.sqrt(float(s @ s))


def chirp_templates(mchirp: Sequence[float], T: float, f0: int = F0_HZ, f_max: float = 1024.0) -> np.ndarray:
    """Full-rate real template rows H[2M][N], N = T*f0, unit norm, last sample = merger."""
    N = int(round(T * f0))
    a = np.arange(N)[::-1]
    H = np.zeros((2 * len(mchirp), N))
    for j, mc in enumerate(mchirp):
        c, s = _chirp_quadratures(mc, a, N, f0, f_max)
        H[2 * j] = c / math.sqrt(float(c @ c))
        H[2 * j + 1] = s / math.sqrt(float(s @ s))
    return H


# --------------------------------------------------------------------------------------------------
# slice layout
# --------------------------------------------------------------------------------------------------
def slice_layout(mc_min: float, T: float, f0: int = F0_HZ, r_min: int = 32, min_taps: int = 1024,
                 max_taps: int = 4096, guard: float = 3.0) -> List[Tuple[int, int, int]]:
    """Generator's slice rule (the paper gives none).

    Returns [(rate, B_s, E_s)] with B/E in f0-samples before merger.  Rate r is allowed once every
    template's frequency is <= r/guard (lowest chirp mass = highest frequency at a given tau); walking
    outward from the merger each rate keeps >= min_taps samples, boundaries land on the next coarser
    grid, spans longer than max_taps are split equally, the lowest allowed rate runs to T.
    """
    Nf0 = int(round(T * f0))
    out: List[Tuple[int, int, int]] = []
    pos, rate = 0, f0
    while pos < Nf0:
        D = f0 // rate
        nxt = rate // 2
        if nxt >= r_min:
            tau_sw = chirp_time_to_merger(nxt / guard, mc_min)
            a_sw = int(math.ceil(tau_sw * f0))
        else:
            a_sw = Nf0
        end = max(a_sw, pos + min_taps * D)
        g = 2 * D if nxt >= r_min else D
        end = -(-end // g) * g
        # do not leave a stub shorter than min_taps at the next rate
        if end >= Nf0 or Nf0 - end < min_taps * (2 * D):
            end = Nf0
        span = (end - pos) // D
        parts = -(-span // max_taps)
        edges = [pos + D * ((span * p) // parts) for p in range(parts)] + [end]
        for p in range(parts):
            out.append((rate, edges[p], edges[p + 1]))
        pos = end
        if nxt >= r_min:
            rate = nxt
    return out


# --------------------------------------------------------------------------------------------------
# SVD bank (Eq. 3) -- offline, untimed
# --------------------------------------------------------------------------------------------------
def _truncate(sig: np.ndarray, energy: Optional[float]) -> Tuple[int, float]:
    e = sig ** 2
    tot = float(e.sum())
    if energy is None:
        return len(sig), 1.0
    cum = np.cumsum(e) / tot
    L = int(np.searchsorted(cum, energy - 1e-15) + 1)
    L = min(max(L, 1), len(sig))
    return L, float(cum[L - 1])


def decompose_slice(Hs: np.ndarray, energy: Optional[float] = 0.9999, method: str = "svd"):
    """H^s (2M x N^s) -> (U [L][N^s] orthonormal rows, R [2M][L] = V diag(sigma), kept energy)."""
    if method == "svd":
        V, sig, Ut = np.linalg.svd(Hs, full_matrices=False)
        L, kept = _truncate(sig, energy)
        return Ut[:L].copy(), V[:, :L] * sig[:L], kept
    if method == "gram":
        # eigen-decomposition of the smaller Gram matrix, then re-orthonormalise the kept rows by QR;
        # R is the projection H U^T, which is V diag(sigma) for exact singular vectors.
        small_rows = Hs.shape[0] <= Hs.shape[1]
        G = Hs @ Hs.T if small_rows else Hs.T @ Hs
        w, Q = np.linalg.eigh(G)
        w, Q = w[::-1].clip(min=0), Q[:, ::-1]
        L, kept = _truncate(np.sqrt(w), energy)
        Ut = (Q[:, :L].T @ Hs) if small_rows else Q[:, :L].T
        Qr, _ = np.linalg.qr(Ut.T)
        U = Qr.T.copy()
        return U, Hs @ U.T, kept
    raise ValueError(method)


def slice_template_matrices(mchirp: Sequence[float], T: float, layout: Sequence[Tuple[int, int, int]],
                            f0: int = F0_HZ, f_max: float = 1024.0) -> List[np.ndarray]:
    """Per slice the template matrix H^s [2M][N^s] (float64) that the SVD of PAPER.md:112-119 decomposes: the analytic chirps
    evaluated on the slice's coarse grid, oldest tap first, rows scaled by sqrt(D) / (full-rate norm)."""
    mchirp = np.asarray(mchirp, dtype=np.float64)
    M = len(mchirp)
    N = int(round(T * f0))
    norms = [_chirp_norms(mc, N, f0, f_max) for mc in mchirp]
    out = []
    for rate, Bs, Es in layout:
        D = f0 // rate
        assert Bs % D == 0 and Es % D == 0 and Es > Bs
        Ns = (Es - Bs) // D
        # n = 0 is the oldest tap: a = E_s - D, ..., B_s
        a = Es - D * (1 + np.arange(Ns))
        Hs = np.empty((2 * M, Ns))
        for j, mc in enumerate(mchirp):
            c, s = _chirp_quadratures(mc, a, N, f0, f_max)
            Hs[2 * j] = c * (math.sqrt(D) / norms[j][0])
            Hs[2 * j + 1] = s * (math.sqrt(D) / norms[j][1])
        out.append(Hs)
    return out


def bank_from_layout(mchirp: Sequence[float], T: float, layout: Sequence[Tuple[int, int, int]],
                     f0: int = F0_HZ, energy: Optional[float] = 0.9999, f_max: float = 1024.0,
                     method: str = "svd") -> Bank:
    mchirp = np.asarray(mchirp, dtype=np.float64)
    slices = []
    for (rate, Bs, Es), Hs in zip(layout, slice_template_matrices(mchirp, T, layout, f0, f_max)):
        D = f0 // rate
        U, R, kept = decompose_slice(Hs, energy, method)
        slices.append(Slice(rate=rate, n_taps=Hs.shape[1], delay=Bs // D, U=U, R=R, kept_energy=kept))
    return Bank(f0=f0, M=len(mchirp), slices=slices, mchirp=mchirp, T=T)


def build_bank(mchirp: Sequence[float], T: float, f0: int = F0_HZ, r_min: int = 32,
               energy: Optional[float] = 0.9999, method: str = "svd", **layout_kw) -> Bank:
    layout = slice_layout(float(np.min(mchirp)), T, f0=f0, r_min=r_min, **layout_kw)
    return bank_from_layout(mchirp, T, layout, f0=f0, energy=energy, method=method)


def random_bank(seed: int, M: int, shape: Sequence[Tuple[int, int, int]], f0: int = F0_HZ) -> Bank:
    """Shape-faithful stand-in bank: seeded random orthonormal U, random R; shape = [(rate, N^s, L^s)].

    Slices abut (delays follow from the tap counts).  R is scaled so each slice contributes variance
    1/S per real row in unit-variance noise, i.e. the summed SNR has unit variance like a chirp bank.
    """
    rng = np.random.default_rng(seed)
    slices, pos = [], 0
    S = len(shape)
    for rate, Ns, L in shape:
        D = f0 // rate
        assert pos % D == 0, "slice boundary must lie on this slice's sample grid"
        Q, _ = np.linalg.qr(rng.standard_normal((Ns, L)))
        R = rng.standard_normal((2 * M, L))
        R *= 1.0 / np.sqrt(S * (R ** 2).sum(axis=1, keepdims=True))
        slices.append(Slice(rate=rate, n_taps=Ns, delay=pos // D, U=Q.T.copy(), R=R))
        pos += Ns * D
    return Bank(f0=f0, M=M, slices=slices, T=pos / f0)


# --------------------------------------------------------------------------------------------------
# strain and injections
# --------------------------------------------------------------------------------------------------
def make_strain(seed: int, n_samples: int) -> np.ndarray:
    """Whitened detector strain stand-in: seeded N(0,1) float32 (PAPER.md:85 'unit variance')."""
    return np.random.default_rng(seed).standard_normal(n_samples).astype(np.float32)


def injection_waveform(mc: float, T: float, amp: float, phase: float, f0: int = F0_HZ,
                       f_max: float = 1024.0) -> np.ndarray:
    """A*(cos(phi) h_2j + sin(phi) h_2j+1), N = T*f0 samples, last sample = merger."""
    H = chirp_templates([mc], T, f0, f_max)
    return amp * (math.cos(phase) * H[0] + math.sin(phase) * H[1])


def inject(strain: np.ndarray, wave: np.ndarray, k0: int) -> None:
    """Add `wave` so that its last sample lands on stream sample k0 (in place, float32 strain)."""
    N = len(wave)
    lo = k0 - (N - 1)
    s0, s1 = max(lo, 0), min(k0 + 1, len(strain))
    if s1 > s0:
        strain[s0:s1] = (strain[s0:s1].astype(np.float64) + wave[s0 - lo:s1 - lo]).astype(np.float32)


# --------------------------------------------------------------------------------------------------
# the five BASELINE.json configs
# --------------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Config:
    number: int
    name: str
    n_banks: int
    M: int
    mc_lo: float
    mc_hi: float
    mc_dist: str            # "uniform" | "loguniform"
    n_det: int
    T_max: float            # longest template (s)
    r_min: int
    seconds: int            # stream length
    buffer_len: int         # samples per push at f0
    n_inj: int
    snr_lo: float
    snr_hi: float
    fixed_layout: Optional[List[Tuple[int, int, int]]] = None
    f0: int = F0_HZ
    seed_base: Optional[int] = None   # config 4 reuses config 3's seeds ("the same setup")

    # ---- deterministic pieces -----------------------------------------------------------------
    def seed(self, idx: int) -> int:
        return (self.number if self.seed_base is None else self.seed_base) * 1000 + idx

    def mchirps(self) -> np.ndarray:
        """All chirp masses, sorted, shape [n_banks][M] (contiguous split = 'similar templates grouped')."""
        rng = np.random.default_rng(self.seed(999))
        n = self.n_banks * self.M
        if self.mc_dist == "uniform":
            mc = rng.uniform(self.mc_lo, self.mc_hi, n)
        else:
            mc = np.exp(rng.uniform(math.log(self.mc_lo), math.log(self.mc_hi), n))
        return np.sort(mc).reshape(self.n_banks, self.M)

    def bank_T(self, mc_min: float) -> float:
        if self.fixed_layout is not None:
            return self.T_max
        tau10 = chirp_time_to_merger(10.0, mc_min)
        return float(min(max(2.0 ** math.ceil(math.log2(tau10)), 8.0), self.T_max))

    def layout(self, b: int, mcs: Optional[np.ndarray] = None):
        mcs = self.mchirps() if mcs is None else mcs
        if self.fixed_layout is not None:
            return self.T_max, list(self.fixed_layout)
        T = self.bank_T(float(mcs[b].min()))
        return T, slice_layout(float(mcs[b].min()), T, f0=self.f0, r_min=self.r_min)

    def bank(self, b: int, method: str = "svd", mcs: Optional[np.ndarray] = None) -> Bank:
        mcs = self.mchirps() if mcs is None else mcs
        T, lay = self.layout(b, mcs)
        return bank_from_layout(mcs[b], T, lay, f0=self.f0, energy=0.9999, method=method)

    def injections(self, seconds: Optional[int] = None) -> List[Injection]:
        """Seeded injections: end sample >= T_b, never two within T_b of each other in one bank."""
        seconds = self.seconds if seconds is None else seconds
        rng = np.random.default_rng(self.seed(998))
        mcs = self.mchirps()
        out: List[Injection] = []
        tries = 0
        while len(out) < self.n_inj and tries < 100 * max(self.n_inj, 1):
            tries += 1
            b = int(rng.integers(self.n_banks))
            j = int(rng.integers(self.M))
            det = int(rng.integers(self.n_det))
            T = self.bank_T(float(mcs[b].min()))
            lo = int(T * self.f0)
            hi = seconds * self.f0 - 64
            amp = float(rng.uniform(self.snr_lo, self.snr_hi))
            ph = float(rng.uniform(0, 2 * math.pi))
            if hi <= lo:
                continue
            k0 = int(rng.integers(lo, hi))
            sep = min(T, seconds / 8.0) * self.f0      # never two within T_b (or 1/8 of a short stream) in one bank+detector
            if any(o.bank == b and o.det == det and abs(o.k0 - k0) < sep for o in out):
                continue
            out.append(Injection(b, j, det, k0, amp, ph))
        return out

    def strain(self, seconds: Optional[int] = None, injections: Optional[List[Injection]] = None) -> np.ndarray:
        """[n_det][seconds*f0] float32 white noise plus the config's injections."""
        seconds = self.seconds if seconds is None else seconds
        n = seconds * self.f0
        d = np.stack([make_strain(self.seed(det), n) for det in range(self.n_det)])
        injections = self.injections(seconds) if injections is None else injections
        mcs = self.mchirps()
        for inj in injections:
            T = self.bank_T(float(mcs[inj.bank].min()))
            w = injection_waveform(float(mcs[inj.bank, inj.template]), T, inj.amp, inj.phase, self.f0)
            inject(d[inj.det], w, inj.k0)
        return d

    @property
    def work_units(self) -> float:
        return float(self.n_banks * self.M * self.n_det * self.seconds)


CONFIGS = {
    1: Config(1, "tiny", 1, 64, 1.0, 1.5, "uniform", 1, 8.0, 512, 16, 2048, 2, 10.0, 10.0,
              fixed_layout=[(2048, 0, 2048), (512, 2048, 16384)]),
    2: Config(2, "small-bank", 4, 500, 1.0, 3.0, "uniform", 2, 64.0, 64, 256, 2048, 20, 8.0, 20.0),
    3: Config(3, "mid-scale", 100, 1000, 0.9, 20.0, "loguniform", 3, 128.0, 32, 600, 2048, 30, 8.0, 20.0),
    4: Config(4, "low-latency", 100, 1000, 0.9, 20.0, "loguniform", 3, 128.0, 32, 600, 128, 30, 8.0, 20.0,
              seed_base=3),
    5: Config(5, "full-scale", 1000, 1000, 0.9, 200.0, "loguniform", 3, 256.0, 32, 3600, 2048, 300, 8.0, 20.0),
}


def make_config(number: int, **overrides) -> Config:
    return dataclasses.replace(CONFIGS[number], **overrides)


def random_triggers(seed: int, n_det: int, M: int, buffer_len: int, p_trigger: float = 0.5, p_coinc: float = 0.3,
                    max_shift: int = 40, overlap: int = 0):
    """Seeded synthetic single-detector triggers [n_det][M] for the coincidence / clustering stage (input generator only):
    structured array (snr float32, sample int32, phase float32); sample = NO_TRIGGER (-2^31) where there is no trigger.
    A fraction p_coinc of the templates gets triggers at nearly equal times in several detectors."""
    rng = np.random.default_rng(seed)
    dt = np.dtype([("snr", np.float32), ("sample", np.int32), ("phase", np.float32)])
    out = np.zeros((n_det, M), dtype=dt)
    out["sample"] = -2147483648
    for j in range(M):
        base = int(rng.integers(-overlap, buffer_len))
        coinc = rng.random() < p_coinc
        for a in range(n_det):
            if rng.random() < p_trigger:
                k = base + int(rng.integers(-max_shift, max_shift + 1)) if coinc else int(rng.integers(-overlap, buffer_len))
                k = min(max(k, -overlap), buffer_len - 1)
                out[a, j] = (np.float32(4.0 + 8.0 * rng.random()), k, np.float32(rng.uniform(-np.pi, np.pi)))
    return out


def template_autocorrelations(H: np.ndarray, delta: int) -> np.ndarray:
    """Input generator for the xi^2 test: [M][2 delta + 1] complex128 autocorrelations of the complex
    templates g_j = H[2j] + i H[2j+1], R_j(t) = sum_m g_j[m] conj(g_j[m + t]) / sum |g_j|^2, t = -delta..delta, through
    numpy's correlate (R_j(0) = 1)."""
    H = np.asarray(H, dtype=np.float64)
    M, N = H.shape[0] // 2, H.shape[1]
    out = np.zeros((M, 2 * delta + 1), dtype=np.complex128)
    for j in range(M):
        g = H[2 * j] + 1j * H[2 * j + 1]
        # np.correlate(a, v, "full")[k] = sum_n a[n + k - (N - 1)] conj(v[n]); lag t = -(k - (N - 1))
        c = np.correlate(g, g, mode="full")
        mid = N - 1
        lags = np.arange(-delta, delta + 1)
        idx = mid - lags
        ok = (idx >= 0) & (idx < len(c))
        out[j, ok] = c[idx[ok]]
        out[j] /= np.sum(np.abs(g) ** 2)
    return out
