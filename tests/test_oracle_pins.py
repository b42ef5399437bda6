"""Pins of the float64 oracle against what the paper and the mathematics fix (no GPU).

Each test names the passage it binds to.  A plausible mistake anywhere in oracle/lloid_oracle.py (dropped
term, wrong sign or index, transposed operand, off-by-one delay) must fail at least one of these.
"""
import math
import os

import numpy as np
import pytest
import scipy.signal

from oracle import (N_DOWN, N_UP, Series, basis_correlate, brute_force, decimate, find_peaks, lloid_snr,
                    rate_groups, reconstruct, resample_kernel, upsample, upsample_input_range)
from workloads import (Bank, Slice, bank_from_layout, chirp_templates, decompose_slice, make_strain,
                       random_bank)

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------- Eq. 4
def test_eq4_hand_values():
    for line in open(os.path.join(GOLDEN, "eq4_kernel_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        f, n, k, val = line.split()
        g = resample_kernel(int(f), int(n))
        assert abs(g[int(k)] - float(val)) < 1e-14, line


@pytest.mark.parametrize("f", [2, 4, 8, 64])
def test_eq4_structure(f):
    gd = resample_kernel(f, N_DOWN)
    gu = resample_kernel(f, N_UP)
    assert len(gd) == 2 * f * N_DOWN + 1 and len(gu) == 2 * f * N_UP + 1   # f=2 -> 129 and 33 taps
    for g, c in ((gd, f * N_DOWN), (gu, f * N_UP)):
        assert g[c] == 1.0
        assert np.array_equal(g, g[::-1])                   # symmetric -> zero phase
        assert abs(g[0]) < 1e-15 and abs(g[-1]) < 1e-15       # window zero at the ends
        # Nyquist-filter property: zero at every multiple of f except the centre (Eq. 8 case 1)
        z = g[c % f::f].copy()
        z[c // f] = 0
        assert np.abs(z).max() < 1e-15


# ---------------------------------------------------------------- decimator
@pytest.mark.parametrize("D,n_down", [(2, N_DOWN), (4, N_DOWN), (16, N_DOWN), (4, 12), (16, 12), (8, 5)])
def test_decimate_equals_textbook_filter_then_pick(D, n_down):
    """Zero-phase decimation = full-rate convolution with sqrt(D)*ghat, centred, then every D-th sample -- also
    for a non-default half length (lloid_options.n_down, PAPER.md:132 'typically set to 32')."""
    rng = np.random.default_rng(D)
    d = rng.standard_normal(2000)
    g = resample_kernel(D, n_down)
    c = n_down * D
    assert len(g) == 2 * c + 1
    full = scipy.signal.convolve(d, math.sqrt(D) * g / g.sum(), mode="full")   # full[i] = sum_k h[k] d[i-k]
    s = decimate(d, D, n_down)
    assert s.j0 == -n_down
    for j in range(-n_down, 2000 // D + n_down):
        i = j * D + c
        want = full[i] if 0 <= i < len(full) else 0.0
        assert abs(s.window(j, j + 1)[0] - want) < 1e-13


@pytest.mark.parametrize("D,frac,gain_tol", [(2, 0.3, 1e-3), (8, 0.5, 1e-3), (4, 0.9, 2e-3)])
def test_decimate_tone_gain_closed_form(D, frac, gain_tol):
    """A tone below the new Nyquist comes out with the same phase and gain G(nu) = sum ghat[k] cos(2 pi nu (k-c))."""
    n = 8192
    nu = frac * 0.5 / D                      # cycles per f0 sample
    t = np.arange(n)
    d = np.cos(2 * math.pi * nu * t + 0.3)
    g = resample_kernel(D, N_DOWN)
    c = N_DOWN * D
    G = float((g / g.sum()) @ np.cos(2 * math.pi * nu * (np.arange(2 * c + 1) - c)))
    assert abs(G - 1) < gain_tol             # flat passband (SURVEY 8c pins)
    s = decimate(d, D)
    j = np.arange(2 * N_DOWN, n // D - 2 * N_DOWN)      # away from the stream edges
    want = math.sqrt(D) * G * np.cos(2 * math.pi * nu * (j * D) + 0.3)
    assert np.abs(s.window(j[0], j[-1] + 1) - want).max() < 1e-12


def test_decimate_unit_variance_convention():
    """DESIGN.md reading 6: DC gain sqrt(D) so white N(0,1) stays (close to) unit variance at every rate."""
    d = make_strain(5, 1 << 18).astype(np.float64)
    for D in (2, 8, 32):
        v = decimate(d, D).window(64, (1 << 18) // D - 64)
        assert abs(v.var() - 1.0) < 0.05


# ---------------------------------------------------------------- upsampler
@pytest.mark.parametrize("f", [2, 4, 8])
def test_upsample_equals_zero_stuff_and_convolve(f):
    """the polyphase form replaces 'insert zeros, convolve with the kernel'."""
    rng = np.random.default_rng(f)
    x = rng.standard_normal((3, 200))
    g = resample_kernel(f, N_UP)
    c = N_UP * f
    stuffed = np.zeros((3, 200 * f))
    stuffed[:, ::f] = x
    lo, hi = 20 * f, 180 * f
    y = upsample(x, 0, f, lo, hi)
    for r in range(3):
        full = np.convolve(stuffed[r], g, mode="full")        # full[i + c] is the zero-phase output i
        assert np.abs(y[r] - full[lo + c:hi + c]).max() < 1e-13
    # Eq. 8 case 1: outputs at i mod f == 0 are the inputs, exactly
    assert np.array_equal(y[:, ::f], x[:, 20:180])


def test_upsample_causal_eq8_plus_advance_is_zero_phase():
    """Eq. 8 case 2 as printed is causal (delay N_up input samples); applied to an input advanced by N_up
    it equals the zero-phase form used by the oracle (reading 9)."""
    f = 2
    rng = np.random.default_rng(0)
    x = rng.standard_normal(300)
    g = resample_kernel(f, N_UP)
    lo, hi = 40, 500
    y = upsample(x[None], 0, f, lo, hi)[0]
    xa = np.concatenate([x[N_UP:], np.zeros(N_UP)])            # advanced input
    for i in range(lo, hi):
        if i % f == 0:
            want = x[i // f]
        else:
            want = sum(xa[i // f - k] * g[k * f + i % f] for k in range(2 * N_UP) if k * f + i % f <= 2 * N_UP * f)
        assert abs(y[i - lo] - want) < 1e-13


def test_upsample_tone_gain():
    f = 2
    q = np.arange(400)
    nu = 0.25 * 0.5                                           # a quarter of the input Nyquist
    x = np.cos(2 * math.pi * nu * q + 0.7)
    y = upsample(x[None], 0, f, 100, 700)[0]
    i = np.arange(100, 700)
    assert np.abs(y - np.cos(2 * math.pi * nu * i / f + 0.7)).max() < 1e-3   # within 1e-3 to 0.5 Nyquist


def test_upsample_input_range_is_sufficient_and_tight():
    """The range the oracle asks of the stage below is exactly what `upsample` reads: it is enough (no assert), every
    input inside it but none outside influences the outputs (checked by perturbing single inputs), and cutting it
    short by two on the left or one on the right makes `upsample` fail."""
    for f in (2, 4):
        for lo, hi in ((0, 64), (-5, 7), (33, 35), (f + 1, 3 * f)):
            a, b = upsample_input_range(lo, hi, f)
            x = np.random.default_rng(1).standard_normal(b - a + 8)        # 4 spare inputs on both sides
            y = upsample(x[None], a - 4, f, lo, hi)[0]                     # must not assert
            used = []
            for m in range(len(x)):
                xp = x.copy()
                xp[m] += 1.0
                used.append(bool(np.abs(upsample(xp[None], a - 4, f, lo, hi)[0] - y).max() > 1e-9))
            idx = np.nonzero(used)[0] + a - 4
            assert a <= idx.min() <= a + 1 and (idx.max() == b - 1 if (hi - 1) % f else b - 3 <= idx.max() <= b - 1)
            with pytest.raises(AssertionError):
                upsample(x[None, 6:], a + 2, f, lo, hi)
            if (hi - 1) % f:
                with pytest.raises(AssertionError):
                    upsample(x[None, 4:b - a + 3], a, f, lo, hi)


# ---------------------------------------------------------------- Eq. 5 / Eq. 6 index conventions
def test_basis_correlate_definition_by_loops():
    rng = np.random.default_rng(3)
    U = rng.standard_normal((3, 7))
    d = rng.standard_normal(50)
    delay = 4
    Y = basis_correlate(U, Series(d, 0), delay, 0, 50, chunk=16)
    for l in range(3):
        for j in range(50):
            acc = 0.0
            for n in range(7):
                idx = j - delay - 7 + 1 + n
                if 0 <= idx < 50:
                    acc += U[l, n] * d[idx]
            assert abs(Y[l, j] - acc) < 1e-13
    R = rng.standard_normal((4, 3))
    own = reconstruct(R, Y)
    assert abs(own[2, 10] - sum(R[2, l] * Y[l, 10] for l in range(3))) < 1e-13


# ---------------------------------------------------------------- Eq. 1 and the exact special case
def _tiny_templates(seed=0, rows=6, N=96):
    rng = np.random.default_rng(seed)
    H = rng.standard_normal((rows, N))
    return H / np.linalg.norm(H, axis=1, keepdims=True)


def _full_rate_bank(H, cuts, energy=None):
    """All slices at f0 (no downsampling), every singular value kept unless `energy` is given."""
    N = H.shape[1]
    sl = []
    edges = [0] + list(cuts) + [N]
    for Bs, Es in zip(edges[:-1], edges[1:]):
        a = Es - 1 - np.arange(Es - Bs)
        Hs = H[:, N - 1 - a]
        U, R, kept = decompose_slice(Hs, energy)
        sl.append(Slice(rate=2048, n_taps=Es - Bs, delay=Bs, U=U, R=R, kept_energy=kept))
    return Bank(f0=2048, M=H.shape[0] // 2, slices=sl)


def test_brute_force_definition_by_loops():
    H = _tiny_templates(rows=2, N=9)
    d = np.random.default_rng(1).standard_normal(30)
    bf = brute_force(H, d)
    for i in range(2):
        for k in range(30):
            acc = sum(H[i, m] * d[k - 8 + m] for m in range(9) if 0 <= k - 8 + m < 30)
            assert abs(bf[i, k] - acc) < 1e-13


def test_lloid_full_rate_full_rank_equals_brute_force_1e10():
    """North star: LLOID with no downsampling and all singular values kept reproduces Eq. 1 to 1e-10 relative."""
    H = _tiny_templates()
    d = np.random.default_rng(2).standard_normal(700)
    bank = _full_rate_bank(H, cuts=(32, 50))
    got = lloid_snr(bank, d)
    want = brute_force(H, d)
    assert np.abs(got - want).max() <= 1e-10 * np.abs(want).max()
    assert np.abs(got - want).max() < 1e-13


def test_lloid_range_and_row_subset_invariance(cfg1):
    """Computing a window / a subset of rows gives the same numbers as the whole (chunk invariance)."""
    bank, d = cfg1["bank32"], cfg1["strain"][0]
    whole = lloid_snr(bank, d, 16384, 16384 + 4096)
    part = lloid_snr(bank, d, 16384 + 1000, 16384 + 1300, rows=[5, 70])
    assert np.abs(part - whole[[5, 70], 1000:1300]).max() < 1e-12


# ---------------------------------------------------------------- SVD bank (Eq. 3)
def test_svd_bank_orthonormal_and_residual(cfg1):
    bank, H = cfg1["bank"], cfg1["H"]
    N = H.shape[1]
    for s in bank.slices:
        D = bank.f0 // s.rate
        assert np.abs(s.U @ s.U.T - np.eye(s.n_basis)).max() < 1e-12
        a = (s.delay + s.n_taps) * D - D * (1 + np.arange(s.n_taps))
        Hs = math.sqrt(D) * H[:, N - 1 - a]
        res = np.linalg.norm(Hs - s.R @ s.U) ** 2 / np.linalg.norm(Hs) ** 2
        assert abs(res - (1 - s.kept_energy)) < 1e-12
        assert 0.9999 <= s.kept_energy and res <= 1e-4
        # smallest L reaching 99.99 %: one basis fewer falls short
        sig = np.linalg.svd(Hs, compute_uv=False)
        e = np.cumsum(sig ** 2) / np.sum(sig ** 2)
        assert e[s.n_basis - 1] >= 0.9999 - 1e-12 and (s.n_basis == 1 or e[s.n_basis - 2] < 0.9999)
    assert 50 <= bank.slices[0].n_basis <= 128 and bank.slices[1].n_basis <= 128   # "two orders" sanity band


def test_gram_bank_matches_svd_bank(cfg1):
    c = cfg1["cfg"]
    b2 = c.bank(0, method="gram")
    d = cfg1["strain"][0]
    a = lloid_snr(cfg1["bank"], d, 20000, 20256)
    b = lloid_snr(b2, d, 20000, 20256)
    assert np.abs(a - b).max() < 1e-9
    for s in b2.slices:
        assert np.abs(s.U @ s.U.T - np.eye(s.n_basis)).max() < 1e-12


# ---------------------------------------------------------------- normalisation: closed-form injection
def test_noiseless_injection_closed_form(cfg1):
    H = cfg1["H"]
    N = H.shape[1]
    j, A, phi, k0 = 11, 7.5, 0.9, N + 333
    inj = A * (math.cos(phi) * H[2 * j] + math.sin(phi) * H[2 * j + 1])
    d = np.zeros(k0 + 50)
    d[k0 - N + 1:k0 + 1] = inj
    bf = brute_force(H[2 * j:2 * j + 2], d, k0, k0 + 1)[:, 0]
    eps = float(H[2 * j] @ H[2 * j + 1])
    assert abs(eps) < 1e-2
    assert abs(bf[0] - A * (math.cos(phi) + eps * math.sin(phi))) < 1e-12
    assert abs(bf[1] - A * (math.sin(phi) + eps * math.cos(phi))) < 1e-12
    # phi = 0 -> Re z = A exactly (unit-norm rows, reading 1)
    d0 = np.zeros(k0 + 1)
    d0[k0 - N + 1:k0 + 1] = A * H[2 * j]
    assert abs(brute_force(H[2 * j:2 * j + 1], d0, k0, k0 + 1)[0, 0] - A) < 1e-12
    # LLOID reaches the same value within its approximation error (~1e-2 A)
    ll = lloid_snr(cfg1["bank"], d, k0, k0 + 1, rows=[2 * j, 2 * j + 1])[:, 0]
    assert np.abs(ll - bf).max() < 3e-2 * A


# ---------------------------------------------------------------- whole multirate path
def test_lloid_causality_bit_identical(cfg1):
    bank, d = cfg1["bank32"], cfg1["strain"][0].astype(np.float64)
    k = 20000
    a = lloid_snr(bank, d, k - 300, k + 1, rows=[0, 1, 64])
    d2 = d.copy()
    d2[k + 1:] = np.random.default_rng(9).standard_normal(len(d) - k - 1) * 50
    b = lloid_snr(bank, d2, k - 300, k + 1, rows=[0, 1, 64])
    assert np.array_equal(a, b)
    # and recent samples do matter (the last ~12 template samples are zero: f > 1024 Hz is cut)
    d2[k - 30] += 1.0
    assert not np.array_equal(a, lloid_snr(bank, d2, k - 300, k + 1, rows=[0, 1, 64]))


def test_lloid_impulse_response_is_time_reversed_template(cfg1):
    bank, H = cfg1["bank"], cfg1["H"]
    N = H.shape[1]
    p = 3000
    d = np.zeros(p + N + 200)
    d[p] = 1.0
    rows = [0, 1, 50, 127]
    out = lloid_snr(bank, d, p, p + N, rows=rows)         # out[i, k-p] = h_eff_i[N-1-(k-p)]
    eff = out[:, ::-1]
    dist = np.linalg.norm(eff - H[rows], axis=1)
    assert dist.max() < 5e-2 and dist.min() > 1e-4           # LLOID approximation error ~1e-2
    # nothing before the impulse (causality) and (almost) nothing after the template has passed
    assert np.abs(lloid_snr(bank, d, p - 100, p, rows=rows)).max() == 0.0


def test_lloid_linearity_and_shift_invariance(cfg1):
    bank = cfg1["bank32"]
    rng = np.random.default_rng(4)
    a = rng.standard_normal(30000)
    b = rng.standard_normal(30000)
    rows = [3, 90]
    k0, k1 = 25000, 25400
    la, lb = lloid_snr(bank, a, k0, k1, rows=rows), lloid_snr(bank, b, k0, k1, rows=rows)
    lab = lloid_snr(bank, 2 * a - 3 * b, k0, k1, rows=rows)
    assert np.abs(lab - (2 * la - 3 * lb)).max() < 1e-11
    shift = 4 * 7                                            # multiple of max D_s = 4
    a_s = np.concatenate([np.zeros(shift), a])
    assert np.abs(lloid_snr(bank, a_s, k0 + shift, k1 + shift, rows=rows) - la).max() < 1e-11


def test_lloid_vs_brute_force_approximation_band(cfg1):
    """Multirate + truncated LLOID differs from Eq. 1 by ~1e-2 RMS (inherent) -- a sanity band
    that catches misaligned slices (a one-sample delay error at 512 Hz gives errors of order 1)."""
    bank, H, d = cfg1["bank"], cfg1["H"], cfg1["strain"][0]
    k0 = 17000
    ll = lloid_snr(bank, d, k0, k0 + 600)
    bf = brute_force(H, d, k0, k0 + 600)
    err = ll - bf
    assert err.std() < 3e-2 and np.abs(err).max() < 0.2


@pytest.mark.parametrize("n_down", [N_DOWN, 12])
def test_multirate_chain_with_skipped_and_repeated_rates(n_down):
    """Random bank, rates 2048/512/512/128 (one x4 stage, two slices at one rate, another x4 stage):
    the oracle must equal an independent composition written with scipy's upfirdn -- with the default decimator
    half length and with n_down = 12 (the lloid_options.n_down path the GPU test test_n_down_option compares against)."""
    N_DOWN = n_down
    bank = random_bank(7, 3, [(2048, 40, 5), (512, 30, 4), (512, 20, 3), (128, 25, 4)])
    d = np.random.default_rng(8).standard_normal(6000)
    k0, k1 = 3000, 3256
    got = lloid_snr(bank, d, k0, k1, n_down=n_down)
    if n_down != 32:
        assert np.abs(got - lloid_snr(bank, d, k0, k1)).max() > 1e-4      # the option does change the result

    def own(s, D):
        sl = bank.slices[s]
        g = resample_kernel(D, N_DOWN)
        if D == 1:
            dr = d
            off = 0
        else:
            # textbook: convolve at full rate, keep every D-th sample, compensate the group delay c
            full = scipy.signal.upfirdn(math.sqrt(D) * g / g.sum(), d, up=1, down=1)
            c = N_DOWN * D
            dr = full[c::D]
            off = 0
        x = np.concatenate([np.zeros(sl.n_taps + sl.delay), dr])
        n_out = len(dr)
        Y = np.stack([np.correlate(x, sl.U[l], mode="valid")[:n_out] for l in range(sl.n_basis)])
        # correlate 'valid' [k] = sum_n x[k+n] U[n]; x index k+n = (j - delay - N + 1 + n) + N + delay -> k = j + 1
        Y = np.concatenate([Y[:, 1:], np.zeros((sl.n_basis, 1))], axis=1)
        return sl.R @ Y

    def up(x, f):
        g = resample_kernel(f, N_UP)
        y = scipy.signal.upfirdn(g, x, up=f, down=1, axis=-1)
        return y[..., N_UP * f:]

    r128 = own(3, 16)
    r512 = own(1, 4) + own(2, 4)
    n = min(r512.shape[1], up(r128, 4).shape[1])
    r512 = r512[:, :n] + up(r128, 4)[:, :n]
    r2048 = own(0, 1)
    n = min(r2048.shape[1], up(r512, 4).shape[1])
    want = r2048[:, :n] + up(r512, 4)[:, :n]
    assert np.abs(got - want[:, k0:k1]).max() < 1e-11


def test_rate_groups():
    bank = random_bank(1, 2, [(2048, 16, 2), (512, 16, 2), (512, 16, 2), (128, 16, 2)])
    assert rate_groups(bank) == [(2048, [0]), (512, [1, 2]), (128, [3])]


# ---------------------------------------------------------------- peaks
def test_find_peaks_brute_force_and_ties():
    rho = np.zeros((4, 16))
    rho[0, 5] = 3.0
    rho[1, 5] = 4.0          # |z| = 5 at k=5
    rho[0, 9] = 5.0          # tie |z| = 5 at k=9 (second buffer) ...
    rho[0, 13] = -5.0        # ... and at k=13: lowest index wins
    rho[2, 2] = -1.0
    snr, idx, ph = find_peaks(rho, 8)
    assert snr.shape == (2, 2)
    assert idx[0, 0] == 5 and snr[0, 0] == 5.0 and abs(ph[0, 0] - math.atan2(4, 3)) < 1e-15
    assert idx[1, 0] == 1 and snr[1, 0] == 5.0 and ph[1, 0] == 0.0
    assert idx[0, 1] == 2 and abs(ph[0, 1] - math.pi) < 1e-15
    assert idx[1, 1] == 0 and snr[1, 1] == 0.0
    # against an explicit loop on random data
    r = np.random.default_rng(0).standard_normal((6, 64))
    snr, idx, ph = find_peaks(r, 32)
    for b in range(2):
        for j in range(3):
            best, kb = -1.0, -1
            for k in range(32):
                v = r[2 * j, 32 * b + k] ** 2 + r[2 * j + 1, 32 * b + k] ** 2
                if v > best:
                    best, kb = v, k
            assert idx[b, j] == kb and abs(snr[b, j] - math.sqrt(best)) < 1e-15


def test_injections_recovered_at_injected_sample(cfg1):
    """SNR >= 8 injections: noiseless, brute force and LLOID both peak exactly at the injected template's
    coalescence sample with |z| = A and phase = phi; in N(0,1) noise the peak stays within +-2 samples."""
    from workloads import injection_waveform, inject
    bank, H, d, B = cfg1["bank32"], cfg1["H"], cfg1["strain"][0], 2048
    for inj in cfg1["inj"]:
        b0 = (inj.k0 // B) * B
        rows = [2 * inj.template, 2 * inj.template + 1]
        clean = np.zeros(len(d), dtype=np.float32)
        inject(clean, injection_waveform(float(bank.mchirp[inj.template]), 8.0, inj.amp, inj.phase), inj.k0)
        for series in (lloid_snr(bank, clean, b0, b0 + B, rows=rows), brute_force(H[rows], clean, b0, b0 + B)):
            snr, idx, ph = find_peaks(series, B)
            assert idx[0, 0] == inj.k0 - b0
            assert abs(snr[0, 0] - inj.amp) < 2e-2 * inj.amp
            dphi = (ph[0, 0] - inj.phase + math.pi) % (2 * math.pi) - math.pi
            assert abs(dphi) < 2e-2
        for series in (lloid_snr(bank, d, b0, b0 + B, rows=rows), brute_force(H[rows], d, b0, b0 + B)):
            snr, idx, ph = find_peaks(series, B)
            assert abs(int(idx[0, 0]) - (inj.k0 - b0)) <= 2
            assert abs(snr[0, 0] - inj.amp) < 3.5            # noise adds ~N(0,1) per quadrature
            dphi = (ph[0, 0] - inj.phase + math.pi) % (2 * math.pi) - math.pi
            # a one-sample time shift trades against ~0.5 rad of phase (2 pi * ~150 Hz / 2048 Hz)
            assert abs(dphi) < (0.35 if idx[0, 0] == inj.k0 - b0 else 1.2)
