"""CPU tests of the seeded input generators (workloads/): they build INPUTS only, but the parity tests and bench.py lean
on their structure (slice tables that abut, orthonormal bases, reproducible seeds), so that structure is pinned here."""
import math

import numpy as np
import pytest

from workloads import (CONFIGS, bank_from_layout, chirp_frequency, chirp_templates, chirp_time_to_merger, make_strain,
                       random_bank, slice_layout)


def test_chirp_frequency_and_time_are_inverse():
    for mc in (0.9, 1.4, 20.0, 200.0):
        for f in (10.0, 32.0, 512.0):
            assert abs(chirp_frequency(chirp_time_to_merger(f, mc), mc) - f) < 1e-9 * f


def test_chirp_templates_unit_norm_band_limited_and_near_quadrature():
    H = chirp_templates([1.0, 1.3], 8.0)
    assert H.shape == (4, 8 * 2048)
    assert np.allclose((H ** 2).sum(axis=1), 1.0, atol=1e-12)
    for j in range(2):
        assert abs(float(H[2 * j] @ H[2 * j + 1])) < 5e-3          # cosine and sine rows are nearly orthogonal
    # zero above 1024 Hz: the last samples before merger are empty
    assert np.all(H[:, -2:] == 0.0)


@pytest.mark.parametrize("cfg,bank", [(2, 0), (2, 3), (3, 0), (3, 50), (3, 99), (5, 0), (5, 999)])
def test_slice_layouts_abut_and_respect_the_rule(cfg, bank):
    c = CONFIGS[cfg]
    mcs = c.mchirps()
    T, lay = c.layout(bank, mcs)
    assert lay[0][0] == c.f0 and lay[0][1] == 0 and lay[-1][2] == int(round(T * c.f0))
    for (r0, b0, e0), (r1, b1, e1) in zip(lay[:-1], lay[1:]):
        assert e0 == b1 and r1 <= r0                                # contiguous, rates never increase
    mc_min = float(mcs[bank].min())
    for rate, b0, e0 in lay:
        D = c.f0 // rate
        assert b0 % D == 0 and e0 % D == 0 and rate >= c.r_min
        assert 1 <= (e0 - b0) // D <= 4096                          # taps per slice
        if rate < c.f0:                                             # every template is below rate/3 inside the slice
            assert chirp_frequency(b0 / c.f0, mc_min) <= rate / 3.0 * (1 + 1e-9)


def test_config1_fixed_layout_matches_baseline_json():
    """BASELINE.json configs[0]: last 1 s at 2048 Hz, 1-8 s at 512 Hz."""
    T, lay = CONFIGS[1].layout(0)
    assert T == 8.0 and lay == [(2048, 0, 2048), (512, 2048, 16384)]
    bank = CONFIGS[1].bank(0)
    assert [(s.rate, s.n_taps, s.delay) for s in bank.slices] == [(2048, 2048, 0), (512, 3584, 512)]


def test_random_bank_is_orthonormal_abutting_and_seeded():
    shape = [(2048, 512, 24), (1024, 768, 40), (256, 512, 33)]
    a, b = random_bank(7, 40, shape), random_bank(7, 40, shape)
    pos = 0
    for s, (rate, n, L), s2 in zip(a.slices, shape, b.slices):
        assert np.allclose(s.U @ s.U.T, np.eye(L), atol=1e-12)
        assert s.delay * (2048 // rate) == pos and s.R.shape == (80, L)
        assert np.array_equal(s.U, s2.U) and np.array_equal(s.R, s2.R)
        pos += n * (2048 // rate)
    assert np.allclose(sum((s.R ** 2).sum(axis=1) for s in a.slices), 1.0)          # unit SNR variance per row


def test_bank_truncation_keeps_requested_energy():
    mc = np.linspace(1.2, 1.3, 12)
    lay = [(2048, 0, 1024), (1024, 1024, 4096)]
    bank = bank_from_layout(mc, 2.0, lay, energy=0.9999)
    full = bank_from_layout(mc, 2.0, lay, energy=None)
    for s, f in zip(bank.slices, full.slices):
        assert s.kept_energy >= 0.9999 - 1e-12 and s.n_basis <= f.n_basis == min(24, s.n_taps)
        assert np.allclose(s.U @ s.U.T, np.eye(s.n_basis), atol=1e-12)


def test_injections_and_strain_are_reproducible_and_separated():
    c = CONFIGS[2]
    inj = c.injections()
    assert len(inj) == c.n_inj and all(8.0 <= i.amp <= 20.0 for i in inj)
    assert [(i.bank, i.template, i.det, i.k0) for i in inj] == [(i.bank, i.template, i.det, i.k0) for i in c.injections()]
    for a in inj:
        assert a.k0 >= 64 * c.f0                                    # the whole template fits before the merger
        for b in inj:
            if a is not b and a.bank == b.bank and a.det == b.det:
                assert abs(a.k0 - b.k0) >= min(64.0, c.seconds / 8.0) * c.f0
    x = make_strain(5, 4096)
    assert x.dtype == np.float32 and np.array_equal(x, make_strain(5, 4096)) and abs(float(x.std()) - 1.0) < 0.05
    assert CONFIGS[4].mchirps().tobytes() == CONFIGS[3].mchirps().tobytes()        # config 4 = "the same setup" as config 3
