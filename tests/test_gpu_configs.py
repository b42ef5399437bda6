"""GPU parity on the shapes of BASELINE.json configs 2-5 (-m gpu): long multirate chirp banks streamed through the
C ABI for longer than their template length, compared with the float64 oracle on the buffers that hold an
injection (full SNR of every template through snr_debug, then peaks).  Banks are the configs' own seeded chirp
masses and slice layouts with a reduced number of templates so the CPU side stays within seconds-to-a-minute;
the full-size configs are exercised by bench.py."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from parity_util import TOL, check_peaks, snr_errors


def _cuda():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def _bank(cfg_no, b, n_templates):
    """Bank b of a config with its real slice layout, thinned to n_templates evenly spaced chirp masses."""
    from workloads import CONFIGS, bank_from_layout
    c = CONFIGS[cfg_no]
    mcs = c.mchirps()
    T, lay = c.layout(b, mcs)
    sel = np.linspace(0, c.M - 1, n_templates).round().astype(int)
    mc = mcs[b][sel]
    return c, bank_from_layout(mc, T, lay, f0=c.f0, energy=0.9999, method="gram").as_f32(), mc, T


def _stream_and_check(banks, strain, B, precision, check, must):
    """Push all of `strain` in buffers of B; `check` = {push index: bank index} whose SNR is dumped and compared."""
    import paper_2511_04730_b200 as lib
    from oracle import find_peaks, lloid_snr
    n_det, n = strain.shape
    st = lib.LloidStream(banks, n_det, B, precision=precision)
    off = np.concatenate([[0], np.cumsum([b.M for b in banks])])
    worst = 0.0
    for p in range(n // B):
        bi = check.get(p)
        out = st.push(strain[:, p * B:(p + 1) * B], want_snr_bank=bi)
        if bi is None:
            continue
        peaks, rho = out
        bank = banks[bi]
        for det in range(n_det):
            ref = lloid_snr(bank, strain[det][:(p + 1) * B], p * B, (p + 1) * B)
            err, _ = snr_errors(rho[det], ref)
            worst = max(worst, err)
            assert err <= TOL[precision], f"push {p} bank {bi} det {det}: max err {err:.3e} of SNR rms"
            snr_o, idx_o, ph_o = find_peaks(ref, B)
            pk = peaks[det, off[bi]:off[bi + 1]]
            mm = [(0, j) for (pp, bb, dd, j) in must if (pp, bb, dd) == (p, bi, det)]      # bit-exact for loud injections
            check_peaks(pk[None], ref, B, TOL[precision], mm)                 # every GPU peak is an oracle maximum
            for (_, j) in mm:
                assert snr_o[0, j] >= 8.0 * 0.8
    st.close()
    return worst


def _inject(strain, det, mc, T, k0, amp, phase):
    from workloads import inject, injection_waveform
    inject(strain[det], injection_waveform(float(mc), T, amp, phase), k0)


@pytest.mark.parametrize("precision", [2, 0])
def test_config2_bank_with_injection(precision):
    """Config 2 bank 0 (64 s, 2048..128 Hz, 7 slices, two pairs at one rate), 2 detectors, 1 s buffers, 67 s."""
    _cuda()
    from workloads import make_strain
    c, bank, mc, T = _bank(2, 0, 96)
    B, secs = 2048, 67
    strain = np.stack([make_strain(2100 + d, secs * 2048) for d in range(2)])
    k0 = 65 * 2048 + 777
    _inject(strain, 1, mc[40], T, k0, 14.0, 1.1)
    worst = _stream_and_check([bank], strain, B, precision, {64: 0, 65: 0, 66: 0}, [(65, 0, 1, 40)])
    print(f"config2 bank0 precision {precision}: worst err {worst:.2e}")


def test_config3_subset_three_banks():
    """Config 3: lightest (128 s, 8 slices down to 128 Hz), middle (128 s, down to 64 Hz) and heaviest (16 s) banks in
    ONE stream (cross-bank stacking of equal-geometry slices), 2 detectors, injections at SNR 9 and 18."""
    _cuda()
    from workloads import make_strain
    sel = [(0, 64), (50, 48), (99, 40)]
    made = [_bank(3, b, m) for b, m in sel]
    banks = [x[1] for x in made]
    B, secs = 2048, 131
    strain = np.stack([make_strain(3100 + d, secs * 2048) for d in range(2)])
    k_a, k_b, k_c = 129 * 2048 + 100, 130 * 2048 + 2047, 129 * 2048 + 1500
    _inject(strain, 0, made[0][2][10], made[0][3], k_a, 18.0, 0.3)
    _inject(strain, 1, made[1][2][30], made[1][3], k_b, 9.0, 4.0)
    _inject(strain, 0, made[2][2][5], made[2][3], k_c, 12.0, 2.0)
    must = [(129, 0, 0, 10), (130, 1, 1, 30), (129, 2, 0, 5)]
    worst = _stream_and_check(banks, strain, B, 2, {128: 1, 129: 0, 130: 1}, must)
    # the heaviest bank shares push 129 with bank 0: second pass for its dump
    worst = max(worst, _stream_and_check(banks, strain[:, :130 * 2048], B, 2, {129: 2}, must))
    print(f"config3 subset: worst err {worst:.2e}")


def test_config4_low_latency_buffers():
    """Config 4: the same banks pushed in 128-sample buffers (1/16 s); 2 new samples per push at 64 Hz.
    The last second (16 pushes) of every template is compared with the oracle."""
    _cuda()
    from workloads import make_strain
    c, bank, mc, T = _bank(3, 99, 64)          # 16 s bank, 2048..128 Hz
    B, secs = 128, 18
    strain = np.stack([make_strain(4100 + d, secs * 2048) for d in range(3)])
    _inject(strain, 2, mc[20], T, 17 * 2048 + 1000, 11.0, 5.0)
    p_inj = (17 * 2048 + 1000) // B
    check = {p: 0 for p in range(17 * 16, 18 * 16)}
    worst = _stream_and_check([bank], strain, B, 2, check, [(p_inj, 0, 2, 20)])
    print(f"config4 buffers of 128: worst err {worst:.2e}")


def test_config5_extreme_banks():
    """Config 5: the 256 s bank (12 slices, six of them at 128 Hz, lowest rate 64 Hz) and the heaviest 8 s bank."""
    _cuda()
    from workloads import make_strain
    made = [_bank(5, 0, 32), _bank(5, 999, 48)]
    banks = [x[1] for x in made]
    B, secs = 2048, 259
    strain = np.stack([make_strain(5100, secs * 2048)])
    _inject(strain, 0, made[0][2][7], made[0][3], 257 * 2048 + 300, 10.0, 0.7)
    _inject(strain, 0, made[1][2][11], made[1][3], 258 * 2048 + 1200, 20.0, 3.0)
    worst = _stream_and_check(banks, strain, B, 2, {257: 0, 258: 1}, [(257, 0, 0, 7), (258, 1, 0, 11)])
    print(f"config5 extremes: worst err {worst:.2e}")


def test_config2_full_size_bench_configuration_sampled():
    """BASELINE.json configs[1] at FULL size, exactly the stream bench.py times (4 SVD banks x 500 templates, 2 detectors,
    2048-sample buffers, split precision): 3 pushes; a sample of templates of every bank is compared with the oracle over
    every sample of the last push (the oracle evaluates just those rows), and for ALL templates the reported peak must be
    the first maximum of the SNR block the same push dumped (internal consistency at full size)."""
    _cuda()
    import paper_2511_04730_b200 as lib
    from oracle import lloid_snr
    from workloads import CONFIGS, make_strain
    c = CONFIGS[2]
    mcs = c.mchirps()
    banks = [c.bank(b, mcs=mcs).as_f32() for b in range(c.n_banks)]
    B, n_push = c.buffer_len, 3
    strain = np.stack([make_strain(c.seed(det), n_push * B) for det in range(c.n_det)])
    off = np.concatenate([[0], np.cumsum([b.M for b in banks])])
    rng = np.random.default_rng(2222)
    for bi, bank in enumerate(banks):
        st = lib.LloidStream(banks, c.n_det, B, precision=lib.LLOID_PREC_F16_SPLIT)
        for p in range(n_push):
            peaks, rho = st.push(strain[:, p * B:(p + 1) * B], want_snr_bank=bi)
        st.close()
        tmpl = np.sort(rng.choice(bank.M, 12, replace=False))
        rows = np.stack([2 * tmpl, 2 * tmpl + 1], axis=1).ravel()
        for det in range(c.n_det):
            ref = lloid_snr(bank, strain[det], (n_push - 1) * B, n_push * B, rows=list(rows))
            z_ref = ref[0::2] + 1j * ref[1::2]
            z = rho[det][2 * tmpl] + 1j * rho[det][2 * tmpl + 1]
            rms = math.sqrt(np.mean(np.abs(z_ref) ** 2))
            err = np.abs(z - z_ref).max() / rms
            assert err <= TOL[2], f"bank {bi} det {det}: max err {err:.3e} of SNR rms"
            # all templates: peak == first maximum of the dumped block, computed the way the kernel does (fp32 |z|^2)
            re, im = rho[det][0::2], rho[det][1::2]
            p32 = re * re + im * im
            k = np.argmax(p32, axis=1)
            pk = peaks[det, off[bi]:off[bi + 1]]
            same = pk["sample"] == k
            # the kernel compares unscaled accumulators; after the power-of-two rescale ties can only differ where two
            # samples round to the same fp32 |z|^2 -- require the value to match there
            assert np.all(same | (np.abs(p32[np.arange(bank.M), pk["sample"]] - p32[np.arange(bank.M), k]) <= 1e-6 * p32.max()))
            assert np.abs(pk["snr"] - np.sqrt(p32[np.arange(bank.M), pk["sample"]])).max() <= 1e-5 * np.sqrt(p32.max())
        print(f"full config 2 bank {bi}: sampled max err {err:.2e}, peak/sample agreement {np.mean(same):.4f}")


def test_config3_twelve_banks_merged_classes_sampled():
    """The first 12 banks of config 3 with their REAL slice layouts (rates, taps, delays from each bank's own chirp masses,
    as bench.py's stand-ins) and 1000 templates each, 3 detectors: many slices of different banks share merged geometry
    classes with per-member column offsets.  Basis counts are those bench.py measured for bank 0 (10, 12, 22, 44, 34, 52,
    45, 39); U is random orthonormal, R random (generation stays within seconds).  Sampled templates of three banks vs
    the oracle."""
    _cuda()
    import paper_2511_04730_b200 as lib
    from oracle import lloid_snr
    from workloads import CONFIGS, make_strain, random_bank
    c = CONFIGS[3]
    mcs = c.mchirps()
    Ls = [10, 12, 22, 44, 34, 52, 45, 39]
    banks = []
    for b in range(12):
        T, lay = c.layout(b, mcs)
        shape = [(rate, (e - s0) // (c.f0 // rate), Ls[min(i, len(Ls) - 1)]) for i, (rate, s0, e) in enumerate(lay)]
        banks.append(random_bank(c.seed(b), c.M, shape, f0=c.f0).as_f32())
    assert len({(s.rate, s.n_taps, s.delay) for bk in banks for s in bk.slices}) > 20      # the layouts do differ
    B, n_push = c.buffer_len, 3
    strain = np.stack([make_strain(c.seed(det) + 7, n_push * B) for det in range(c.n_det)])
    rng = np.random.default_rng(3333)
    for bi in (0, 5, 11):
        bank = banks[bi]
        st = lib.LloidStream(banks, c.n_det, B, precision=lib.LLOID_PREC_F16_SPLIT)
        for p in range(n_push):
            peaks, rho = st.push(strain[:, p * B:(p + 1) * B], want_snr_bank=bi)
        st.close()
        tmpl = np.sort(rng.choice(bank.M, 8, replace=False))
        rows = np.stack([2 * tmpl, 2 * tmpl + 1], axis=1).ravel()
        worst = 0.0
        for det in range(c.n_det):
            ref = lloid_snr(bank, strain[det], (n_push - 1) * B, n_push * B, rows=list(rows))
            z_ref = ref[0::2] + 1j * ref[1::2]
            z = rho[det][2 * tmpl] + 1j * rho[det][2 * tmpl + 1]
            rms = math.sqrt(np.mean(np.abs(z_ref) ** 2))
            worst = max(worst, np.abs(z - z_ref).max() / rms)
        print(f"config 3 (12 banks) bank {bi} [{bank.describe()[:48]}...]: sampled max err {worst:.2e}")
        assert worst <= TOL[2]
