"""CPU pins of oracle/events_oracle.py (overlapped trigger windows, template autocorrelation, xi^2 of Eq. 10, coincidence,
clustering) against closed forms, hand-built cases and brute force -- no GPU."""
import itertools
import math

import numpy as np

from oracle import brute_force, cluster, coincidences, find_peaks, find_peaks_overlap, template_acorr, xi2


def test_overlap_zero_equals_plain_peak_search():
    rng = np.random.default_rng(1)
    rho = rng.standard_normal((12, 4 * 256))
    a = find_peaks(rho, 256)
    b = find_peaks_overlap(rho, 256, 0)
    assert np.array_equal(a[1], b[1])
    assert np.allclose(a[0], b[0], rtol=1e-14) and np.allclose(a[2], b[2], rtol=1e-14)


def test_peak_in_the_overlap_is_reported_by_both_windows():
    """Fig. 5: windows overlap, so a trigger just before a buffer boundary belongs to two windows."""
    B, ov = 100, 20
    rho = np.zeros((2, 3 * B))
    rho[0, 2 * B - 7] = 9.0            # 7 samples before the start of window 2
    rho[1, 2 * B - 7] = 1.0
    rho[0, 2 * B - 30] = 5.0           # outside window 2's overlap
    rho[0, 40] = 3.0
    snr, idx, ph = find_peaks_overlap(rho, B, ov)
    assert idx[0, 0] == 40 and math.isclose(snr[0, 0], 3.0)
    assert idx[1, 0] == B - 7 and math.isclose(snr[1, 0], math.hypot(9, 1))
    assert idx[2, 0] == -7 and math.isclose(snr[2, 0], math.hypot(9, 1)) and math.isclose(ph[2, 0], math.atan2(1, 9))
    rho[0, 2 * B - 7] = 0.0; rho[1, 2 * B - 7] = 0.0
    snr, idx, _ = find_peaks_overlap(rho, B, ov)
    assert idx[2, 0] == -ov and snr[2, 0] == 0.0      # all zero in window 2: first sample of the window


def test_first_window_is_shortened_and_ties_take_the_first_sample():
    B, ov = 64, 16
    rho = np.zeros((2, 2 * B))
    rho[0, 5] = 2.0; rho[0, 9] = 2.0
    rho[0, B - 3] = 4.0; rho[0, B + 11] = 4.0          # tie between the overlap and the buffer: the earlier sample wins
    snr, idx, _ = find_peaks_overlap(rho, B, ov)
    assert idx[0, 0] == B - 3                           # window 0 = [0, B)
    assert idx[1, 0] == -3 and snr[1, 0] == 4.0


def test_acorr_closed_form_for_a_complex_exponential():
    """g[m] = exp(i w m), m < N: R(t) = sum_m g[m] conj(g[m + t]) / N = exp(-i w t) (N - |t|) / N."""
    N, w, delta = 200, 0.37, 50
    m = np.arange(N)
    R = template_acorr(np.cos(w * m), np.sin(w * m), delta)
    t = np.arange(-delta, delta + 1)
    assert np.allclose(R, np.exp(-1j * w * t) * (N - np.abs(t)) / N, atol=1e-13)
    assert abs(R[delta] - 1.0) < 1e-15
    assert np.allclose(R[::-1], np.conj(R), atol=1e-15)           # Hermitian: R(-t) = conj R(t)


def test_acorr_is_the_matched_filter_response_to_the_template_itself():
    """Noiseless injection of a chirp through brute-force filtering: z(k0 + t) = z(k0) R(t) up to the templates'
    non-analyticity (R_j is what a perfect signal leaves in the SNR series)."""
    from workloads import chirp_templates
    H = chirp_templates([1.3], 1.0, 2048, 1024.0)
    N, delta = H.shape[1], 175
    R = template_acorr(H[0], H[1], delta)
    A, phi = 11.0, 0.8
    d = np.zeros(N + 2 * delta + 8)
    k0 = N - 1 + delta + 3
    d[k0 - N + 1:k0 + 1] = A * (math.cos(phi) * H[0] + math.sin(phi) * H[1])
    rho = brute_force(H, d)
    z = rho[0] + 1j * rho[1]
    seg = z[k0 - delta:k0 + delta + 1]
    assert abs(abs(z[k0]) - A) < 0.02 * A
    assert np.abs(seg - z[k0] * R).max() < 0.02 * A
    assert xi2(z, k0, R) < 1e-3 * A * A / np.sum(2 - 2 * np.abs(R) ** 2) * len(R)


def test_xi2_closed_forms():
    rng = np.random.default_rng(3)
    delta = 40
    t = np.arange(-delta, delta + 1)
    R = np.exp(-0.5 * (t / 9.0) ** 2) * np.exp(0.3j * t)
    z0 = 7.0 * np.exp(0.4j)
    z = np.zeros(400, dtype=complex); k0 = 200
    z[k0 - delta:k0 + delta + 1] = z0 * R
    assert xi2(z, k0, R) < 1e-28                                   # a perfect signal
    e = rng.standard_normal(2 * delta + 1) + 1j * rng.standard_normal(2 * delta + 1)
    e[delta] = 0.0                                                 # keeps z[k0] = z0
    c = 0.7
    z[k0 - delta:k0 + delta + 1] += c * e
    want = c * c * np.sum(np.abs(e) ** 2) / np.sum(2 - 2 * np.abs(R) ** 2)
    assert math.isclose(xi2(z, k0, R), want, rel_tol=1e-12)
    # window leaving the series: the missing samples count as zeros
    k1 = 10
    seg = np.concatenate([np.zeros(delta - k1, dtype=complex), z[:k1 + delta + 1]])
    want = np.sum(np.abs(seg - z[k1] * R) ** 2) / np.sum(2 - 2 * np.abs(R) ** 2)
    assert math.isclose(xi2(z, k1, R), want, rel_tol=1e-12)


def test_xi2_has_unit_mean_in_gaussian_noise():
    """E |z(t) - z(0) R(t)|^2 = 2 - 2 |R(t)|^2 for the SNR of unit-variance white noise (E|z|^2 = 2, E z(t) z*(0) = 2 R(t)):
    the denominator of Eq. 10 normalises the statistic to mean 1."""
    from workloads import chirp_templates
    H = chirp_templates([2.0], 0.5, 2048, 1024.0)
    delta = 100
    R = template_acorr(H[0], H[1], delta)
    rng = np.random.default_rng(5)
    d = rng.standard_normal(400000)
    rho = brute_force(H, d)
    z = rho[0] + 1j * rho[1]
    ks = np.arange(2000, len(d) - 2000, 450)
    vals = np.array([xi2(z, int(k), R) for k in ks])
    assert abs(vals.mean() - 1.0) < 0.08, vals.mean()


def _coinc_loop(snr, sample, dt, thr):
    """Independent restatement with explicit loops over bit masks."""
    n_det, M = snr.shape
    mask = np.zeros(M, dtype=np.int64); net = np.zeros(M)
    for j in range(M):
        for m in range(1, 1 << n_det):
            dets = [a for a in range(n_det) if (m >> a) & 1]
            if len(dets) < 2 or any(snr[a, j] < thr for a in dets):
                continue
            ok = all(abs(int(sample[a, j]) - int(sample[b, j])) <= dt[a][b] for a in dets for b in dets if a < b)
            v = math.sqrt(sum(float(snr[a, j]) ** 2 for a in dets))
            if ok and v > net[j]:
                mask[j], net[j] = m, v
    return mask, net


def test_coincidence_hand_cases_and_loop_restatement():
    dt = np.array([[0, 31, 56], [31, 0, 55], [56, 55, 0]])          # H-L 0.0150 s, H-V, L-V at 2048 Hz (illustrative)
    #                 tmpl 0: HL within, V far     1: all three     2: only one trigger   3: H-V within, L below threshold
    snr = np.array([[8.0, 6.0, 9.0, 7.0], [5.0, 6.0, 0.0, 3.0], [9.0, 6.0, 0.0, 5.0]])
    smp = np.array([[100, 500, 10, 900], [131, 520, 0, 905], [400, 540, 0, 956]])
    mask, net = coincidences(snr, smp, dt, 4.0)
    assert mask.tolist() == [0b011, 0b111, 0, 0b101]
    assert np.allclose(net, [math.hypot(8, 5), math.sqrt(108), 0.0, math.hypot(7, 5)])
    smp[1, 0] = 132                                                  # one sample outside the H-L window
    assert coincidences(snr, smp, dt, 4.0)[0][0] == 0
    # pairwise, not chained: H-L ok, L-V ok, H-V too far -> the louder pair wins, not the triple
    snr = np.array([[6.0], [6.0], [7.0]]); smp = np.array([[0], [30], [80]])
    mask, net = coincidences(snr, smp, dt, 4.0)
    assert mask[0] == 0b110 and math.isclose(net[0], math.hypot(6, 7))
    from workloads import random_triggers
    tr = random_triggers(11, 3, 400, 2048, overlap=67)
    have = tr["sample"] != -2147483648
    s = np.where(have, tr["snr"], 0.0)
    a = coincidences(s, tr["sample"], dt, 4.0)
    b = _coinc_loop(s.astype(np.float64), tr["sample"], dt, 4.0)
    assert np.array_equal(a[0], b[0]) and np.allclose(a[1], b[1])
    assert (a[0] != 0).sum() > 20


def test_cluster_keeps_one_event_per_bank():
    mask = np.array([0, 3, 5, 0, 0, 0, 7, 3, 3])
    net = np.array([0.0, 9.0, 11.0, 0.0, 0.0, 0.0, 8.0, 12.0, 12.0])
    out = cluster(mask, net, [0, 3, 6, 9])
    assert out == [(2, 5, 11.0), (-1, 0, 0.0), (7, 3, 12.0)]      # tie in the last bank -> the lower template index


def test_generator_autocorrelations_equal_the_oracle_definition():
    """workloads.template_autocorrelations (numpy.correlate, feeds the CUDA side) against oracle.template_acorr."""
    from workloads import chirp_templates, template_autocorrelations
    H = chirp_templates([1.1, 1.7, 2.9], 1.0, 2048, 1024.0)
    A = template_autocorrelations(H, 175)
    for j in range(3):
        assert np.abs(A[j] - template_acorr(H[2 * j], H[2 * j + 1], 175)).max() < 1e-13
