"""GPU parity of the event-identification stage (-m gpu): overlapped trigger windows (Fig. 5), coincidence
formation and clustering through the C ABI against oracle/events_oracle.py."""
import math

import numpy as np
import pytest

from parity_util import TOL, zc

pytestmark = pytest.mark.gpu

NO_TRIGGER = -2147483648
DT3 = np.array([[0, 31, 56], [31, 0, 55], [56, 55, 0]], dtype=np.int32)   # illustrative H/L/V windows at 2048 Hz


def _cuda():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def test_overlapped_trigger_windows_against_the_oracle():
    """Windows [n0 - 67, n0 + B): every reported peak is a maximum of the oracle SNR over ITS window; a loud signal that
    ends 9 samples before a buffer boundary is reported by both windows, bit-exactly at the oracle's sample."""
    _cuda()
    import paper_2511_04730_b200 as lib
    from oracle import find_peaks_overlap, lloid_snr
    from workloads import bank_from_layout, inject, injection_waveform, make_strain
    f0, B, ov = 2048, 1024, 67
    mc = np.linspace(1.2, 1.4, 37)
    lay = [(2048, 0, 1024), (1024, 1024, 3072), (512, 3072, 8192), (256, 8192, 16384)]
    bank = bank_from_layout(mc, 8.0, lay, f0=f0).as_f32()
    n_push = 20
    strain = np.stack([make_strain(31, n_push * B), make_strain(32, n_push * B)])
    k_inj = 18 * B - 9
    inject(strain[0], injection_waveform(float(mc[11]), 8.0, 15.0, 0.6, f0), k_inj)
    st = lib.LloidStream([bank], 2, B, precision=lib.LLOID_PREC_F16_SPLIT, trigger_overlap=ov)
    pk = np.stack([st.push(strain[:, p * B:(p + 1) * B]).copy() for p in range(n_push)])       # [push][det][M]
    st.reset()
    pk2 = st.push(strain[:, :B]).copy()
    assert np.array_equal(pk2, pk[0])                                   # reset clears the carried tail peak
    st.close()
    for det in range(2):
        ref = lloid_snr(bank, strain[det])
        z = zc(ref)
        gate = TOL[2] * math.sqrt(np.mean(np.abs(z) ** 2))
        snr_o, idx_o, ph_o = find_peaks_overlap(ref, B, ov)
        for p in range(n_push):
            k = pk["sample"][p, det].astype(np.int64)
            lo = -ov if p > 0 else 0
            assert (k >= lo).all() and (k < B).all()
            at = z[np.arange(bank.M), p * B + k]
            assert (snr_o[p] - np.abs(at) <= 2 * gate).all()
            assert np.abs(pk["snr"][p, det] - np.abs(at)).max() <= gate
        agree = np.mean(pk["sample"][:, det] == idx_o)
        assert agree > 0.98, agree
        assert (idx_o[1:] < 0).mean() > 0.01                             # the overlap is exercised
    assert pk["sample"][17, 0, 11] == B - 9 or abs(int(pk["sample"][17, 0, 11]) - (B - 9)) <= 2
    s17, s18 = int(pk["sample"][17, 0, 11]), int(pk["sample"][18, 0, 11])
    assert s18 == s17 - B and s18 < 0 and pk["snr"][18, 0, 11] == pk["snr"][17, 0, 11] and pk["snr"][18, 0, 11] > 11


def test_threshold_marks_missing_triggers():
    _cuda()
    import paper_2511_04730_b200 as lib
    from workloads import make_strain, random_bank
    bank = random_bank(5, 90, [(2048, 512, 12), (1024, 512, 20)]).as_f32()
    st = lib.LloidStream([bank], 1, 512, threshold=3.0, trigger_overlap=40)
    for p in range(3):
        pk = st.push(make_strain(50 + p, 512)[None])
    st.close()
    below = pk["snr"][0] == 0
    assert below.any() and (~below).any()
    assert (pk["sample"][0][below] == NO_TRIGGER).all() and (pk["sample"][0][~below] >= -40).all()


@pytest.mark.parametrize("n_det", [2, 3, 4])
def test_coincidence_and_clustering_on_seeded_triggers(n_det):
    """The coincidence / clustering kernel alone, on seeded synthetic triggers (no CUDA path upstream of it)."""
    torch = _cuda()
    import paper_2511_04730_b200 as lib
    from oracle import cluster, coincidences
    from workloads import random_bank, random_triggers
    Ms = [70, 1, 130, 257]
    banks = [random_bank(60 + i, M, [(2048, 64, 2)]).as_f32() for i, M in enumerate(Ms)]
    st = lib.LloidStream(banks, n_det, 256, trigger_overlap=67)
    off = np.concatenate([[0], np.cumsum(Ms)])
    dt = np.array([[0, 31, 56, 20], [31, 0, 55, 40], [56, 55, 0, 9], [20, 40, 9, 0]], dtype=np.int32)[:n_det, :n_det]
    for seed in (1, 2, 3):
        tr = random_triggers(seed, n_det, int(off[-1]), 256, overlap=67)
        if seed == 3:
            tr["sample"][:, off[1]:off[2]] = NO_TRIGGER                  # a bank without any trigger
        dev = torch.from_numpy(tr.view(np.int32).reshape(n_det, -1, 3).copy()).cuda()
        ev = st.events(dt, peaks_dev=dev)
        have = tr["sample"] != NO_TRIGGER
        mask, net = coincidences(np.where(have, tr["snr"], 0.0), tr["sample"], dt, 1.0)
        want = cluster(mask, net, off)
        assert any(w[0] >= 0 for w in want)
        for b, (j, m, v) in enumerate(want):
            assert ev["template_index"][b] == j and ev["det_mask"][b] == m, (b, ev[b], want[b])
            assert abs(ev["net_snr"][b] - v) <= 1e-6 * max(v, 1.0)
            for a in range(lib.binding.LLOID_MAX_DET):
                if (m >> a) & 1:
                    assert ev["sample"][b][a] == tr["sample"][a, j] and ev["snr"][b][a] == tr["snr"][a, j]
                else:
                    assert ev["sample"][b][a] == NO_TRIGGER
    st.close()


def test_end_to_end_three_detector_event():
    """The same chirp injected into three detectors with arrival-time shifts inside the coincidence windows: the event of
    its bank is that template with all three detectors; the oracle chain (LLOID SNR -> overlapped peaks -> coincidence ->
    clustering) gives the same event."""
    _cuda()
    import paper_2511_04730_b200 as lib
    from oracle import cluster, coincidences, find_peaks_overlap, lloid_snr
    from workloads import bank_from_layout, inject, injection_waveform, make_strain
    f0, B, ov, thr = 2048, 2048, 67, 4.0
    lay = [(2048, 0, 2048), (512, 2048, 8192)]
    mcs = [np.linspace(1.0, 1.2, 24), np.linspace(1.3, 1.5, 30)]
    banks = [bank_from_layout(mc, 4.0, lay, f0=f0).as_f32() for mc in mcs]
    n_push = 7
    strain = np.stack([make_strain(70 + d, n_push * B) for d in range(3)])
    k0 = 5 * B + 20                                                       # near a boundary: detector 1 peaks in the overlap
    for d, (shift, amp) in enumerate([(0, 9.0), (-28, 8.0), (25, 7.0)]):
        inject(strain[d], injection_waveform(float(mcs[1][17]), 4.0, amp, 0.3 + d, f0), k0 + shift)
    st = lib.LloidStream(banks, 3, B, threshold=thr, trigger_overlap=ov)
    evs = []
    for p in range(n_push):
        st.push(strain[:, p * B:(p + 1) * B])
        evs.append(st.events(DT3).copy())
    st.close()
    refs = [[lloid_snr(bk, strain[d]) for d in range(3)] for bk in banks]
    off = [0, 24, 54]
    for p in range(n_push):
        snr = np.zeros((3, 54)); smp = np.zeros((3, 54), dtype=np.int64)
        for b in range(2):
            for d in range(3):
                s, i, _ = find_peaks_overlap(refs[b][d], B, ov)
                snr[d, off[b]:off[b + 1]] = np.where(s[p] >= thr, s[p], 0.0)
                smp[d, off[b]:off[b + 1]] = i[p]
        mask, net = coincidences(snr, smp, DT3, thr)
        want = cluster(mask, net, off)
        for b in range(2):
            g = evs[p][b]
            if want[b][0] >= 0 and want[b][2] > 7.0:                      # a clear event: template, detectors and SNR agree
                assert g["template_index"] == want[b][0] and g["det_mask"] == want[b][1], (p, b, g, want[b])
                assert abs(g["net_snr"] - want[b][2]) < 0.01
    e = evs[5][1]
    assert e["template_index"] == 24 + 17 and e["det_mask"] == 7 and e["net_snr"] > 11
    assert e["sample"][1] < 0 <= e["sample"][0]


def test_xi2_from_the_materialised_snr_against_the_oracle():
    """Eq. 10 on the GPU SNR series (snr_debug dumps of consecutive buffers side by side) for the triggers of every middle
    buffer, against oracle.xi2 on the float64 LLOID SNR at the oracle's own trigger samples."""
    torch = _cuda()
    import paper_2511_04730_b200 as lib
    from oracle import find_peaks, lloid_snr, xi2
    from workloads import bank_from_layout, chirp_templates, inject, injection_waveform, make_strain, template_autocorrelations
    f0, B, delta = 2048, 1024, 175
    mc = np.linspace(1.2, 1.4, 21)
    lay = [(2048, 0, 1024), (1024, 1024, 3072), (512, 3072, 8192), (256, 8192, 16384)]
    bank = bank_from_layout(mc, 8.0, lay, f0=f0).as_f32()
    n_push = 20
    strain = make_strain(91, n_push * B)[None].copy()
    inject(strain[0], injection_waveform(float(mc[7]), 8.0, 14.0, 1.1, f0), 18 * B + 300)
    acorr = template_autocorrelations(chirp_templates(mc, 8.0, f0, 1024.0), delta)
    st = lib.LloidStream([bank], 1, B)
    snr_all = torch.zeros((2 * bank.M, n_push * B), dtype=torch.float32, device="cuda")
    pks = []
    for p in range(n_push):
        pk, snr = st.push(strain[:, p * B:(p + 1) * B], want_snr_bank=0)
        snr_all[:, p * B:(p + 1) * B] = torch.from_numpy(snr[0]).cuda()
        pks.append(pk[0].copy())
    st.close()
    ac_dev = torch.from_numpy(np.stack([acorr.real, acorr.imag], axis=-1).astype(np.float32)).cuda().contiguous()
    ref = lloid_snr(bank, strain[0])
    z = ref[0::2] + 1j * ref[1::2]
    _, idx_o, _ = find_peaks(ref, B)
    worst, n_cmp = 0.0, 0
    for p in (1, 9, 17, 18):
        k0 = (pks[p]["sample"].astype(np.int64) + p * B).astype(np.int32)
        got = lib.binding.lloid_xi2_series(snr_all, torch.from_numpy(k0).cuda(), ac_dev, delta).cpu().numpy()
        for j in range(bank.M):
            if pks[p]["sample"][j] != idx_o[p, j]:
                continue                                    # a near-tie resolved differently: another trigger, not comparable
            want = xi2(z[j], int(idx_o[p, j]) + p * B, acorr[j])
            worst = max(worst, abs(got[j] - want) / want)
            n_cmp += 1
    print(f"xi2: {n_cmp} triggers compared, worst relative error {worst:.2e}")
    assert n_cmp > 70 and worst < 2e-3
    # the injected template's trigger is consistent with its autocorrelation; all values are O(1) in noise
    got18 = lib.binding.lloid_xi2_series(snr_all, torch.from_numpy((pks[18]["sample"].astype(np.int64) + 18 * B).astype(np.int32)).cuda(),
                                         ac_dev, delta).cpu().numpy()
    assert pks[18]["snr"][7] > 11 and 0.3 < got18[7] < 2.5
    none = torch.full((bank.M,), NO_TRIGGER, dtype=torch.int32, device="cuda")
    assert (lib.binding.lloid_xi2_series(snr_all, none, ac_dev, delta).cpu().numpy() == -1).all()


@pytest.mark.parametrize("delta", [175, 350])
def test_xi2_in_the_stream_against_the_oracle(delta):
    """lloid_stream_xi2: the second reconstruction pass one buffer later (SNR never materialised), 2 detectors x 2 banks,
    against oracle.xi2 on the float64 LLOID SNR -- for every buffer, including the first (zeros before the stream start)."""
    _cuda()
    import paper_2511_04730_b200 as lib
    from oracle import find_peaks, lloid_snr, xi2
    from workloads import bank_from_layout, chirp_templates, inject, injection_waveform, make_strain, template_autocorrelations
    f0, B = 2048, 1024
    lay = [(2048, 0, 1024), (1024, 1024, 3072), (512, 3072, 8192), (256, 8192, 16384)]
    mcs = [np.linspace(1.2, 1.4, 21), np.linspace(1.5, 1.8, 150)]           # the second bank has two template tiles
    banks = [bank_from_layout(mc, 8.0, lay, f0=f0).as_f32() for mc in mcs]
    acorr = [template_autocorrelations(chirp_templates(mc, 8.0, f0, 1024.0), delta) for mc in mcs]
    n_push = 20
    strain = np.stack([make_strain(93 + d, n_push * B) for d in range(2)])
    inject(strain[1], injection_waveform(float(mcs[1][140]), 8.0, 13.0, 2.1, f0), 17 * B + 1000)   # window crosses a buffer edge
    st = lib.LloidStream(banks, 2, B, acorr=acorr)
    with pytest.raises(lib.LloidError):
        st.xi2()                                                          # needs two pushes
    pks, xis = [], {}
    for p in range(n_push):
        pks.append(st.push(strain[:, p * B:(p + 1) * B]).copy())
        if p >= 1:
            xis[p - 1] = st.xi2()
    st.close()
    off = [0, 21, 171]
    worst, n_cmp = 0.0, 0
    for det in range(2):
        for b, bank in enumerate(banks):
            ref = lloid_snr(bank, strain[det])
            z = ref[0::2] + 1j * ref[1::2]
            _, idx_o, _ = find_peaks(ref, B)
            for p in (0, 1, 8, 16, 17, 18):
                got = xis[p][det, off[b]:off[b + 1]]
                for j in range(0, bank.M, 3 if bank.M > 50 else 1):
                    if pks[p]["sample"][det, off[b] + j] != idx_o[p, j]:
                        continue
                    want = xi2(z[j], int(idx_o[p, j]) + p * B, acorr[b][j])
                    worst = max(worst, abs(got[j] - want) / want)
                    n_cmp += 1
    print(f"stream xi2 (delta {delta}): {n_cmp} triggers compared, worst relative error {worst:.2e}")
    assert n_cmp > 250 and worst < 2e-3
    assert pks[17]["snr"][1, 21 + 140] > 10 and 0.3 < xis[17][1, 21 + 140] < 2.5


def test_xi2_is_off_without_autocorrelations():
    _cuda()
    import paper_2511_04730_b200 as lib
    from workloads import make_strain, random_bank
    st = lib.LloidStream([random_bank(5, 40, [(2048, 256, 8)]).as_f32()], 1, 256)
    st.push(make_strain(1, 256)[None]); st.push(make_strain(2, 256)[None])
    with pytest.raises(lib.LloidError) as e:
        st.xi2()
    assert e.value.code == lib.binding.LLOID_ESTATE
    st.close()
