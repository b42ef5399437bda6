"""Full-size, live-history GPU parity on BASELINE.json configs 2-5 (-m gpu) -- VERDICT r1 row g.

Each test creates THE stream bench.py times for that config (bench.bank_plan / bench.iter_banks: every bank of the config
with its real slice layout; the chirp-SVD banks of bench.real_bank_ids -- among them the banks hit by the first seeded
injections -- and shape-faithful stand-ins for the rest), pushes parity_seconds(c) = T_max + 2 s of the config's own seeded
strain carrying the config's own seeded injections (those that fall in a chirp-SVD bank: a stand-in bank has no chirp to
match), so that EVERY slice of every bank reads live data, and compares with the float64 oracle:

  * banks checked: every injected chirp-SVD bank, the lightest and the heaviest bank, and one stand-in (>= 5 banks);
  * pushes checked: for an injected bank the pushes that hold its injections, for the others the last push(es);
  * on each: sampled template rows (the injected ones among them) of the dumped SNR element by element against
    lloid_snr(rows=...), gate 2e-3 of the SNR rms; ALL templates' reported peaks validated as maxima of the oracle SNR
    (tests/parity_util.py peak rule), the injected templates' samples bit-exact.

One lloid_stream_push dumps one bank, so the stream is replayed once per checked bank (lloid_state_reset between).
"""
import math

import numpy as np
import pytest

from parity_util import TOL, check_peaks, snr_errors

pytestmark = pytest.mark.gpu

_REAL = {}      # (seed-equivalent config, bank) -> chirp-SVD bank, shared by config 3 and config 4 (same banks)


def _cuda():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _real_banks(cfg_no, ids):
    import bench
    key = 3 if cfg_no == 4 else cfg_no                       # config 4 is config 3's bank set
    miss = [b for b in ids if (key, b) not in _REAL]
    if miss:
        for b, bank in bench.real_banks(key, miss).items():
            _REAL[(key, b)] = bank
    return {b: _REAL[(key, b)] for b in ids}


def _fullsize(cfg_no, n_rows=6, tail_pushes=1):
    torch = _cuda()
    import bench
    import paper_2511_04730_b200 as lib
    from oracle import decimate, find_peaks, lloid_snr
    c, plan = bench.bank_plan(cfg_no)
    B, f0, n_det = c.buffer_len, c.f0, c.n_det
    S = bench.parity_seconds(c)
    real_ids = [p[1] for p in plan if p[0] == "real"]
    real = _real_banks(cfg_no, real_ids)
    injs = [i for i in c.injections(S) if i.bank in real]
    strain = c.strain(S, injections=injs)                                          # [n_det][S*f0] noise + injections
    n_push = S * f0 // B
    # ---- banks to check: injected chirp-SVD banks, lightest, heaviest, one stand-in
    standins = [p[1] for p in plan if p[0] == "standin"]
    check_banks = sorted({i.bank for i in injs} | {real_ids[0], real_ids[-1]})
    if len(check_banks) < 4:
        check_banks = sorted(set(check_banks) | set(real_ids[:4]))
    if standins:
        check_banks.append(standins[len(standins) // 2])
    keep = {}

    def gen():
        for b, bank in enumerate(bench.iter_banks(cfg_no, plan, real=real)):
            if b in check_banks:
                keep[b] = bank
            yield bank
    st = lib.LloidStream(gen(), n_det, B, precision=lib.LLOID_PREC_F16_SPLIT)
    assert st.Mtot == c.n_banks * c.M
    off = np.concatenate([[0], np.cumsum(st.Ms)])
    dev_strain = torch.from_numpy(np.ascontiguousarray(strain.reshape(n_det, n_push, B).transpose(1, 0, 2))).cuda()
    dec = [{D: decimate(strain[det], D) for D in sorted({f0 // s.rate for b in keep.values() for s in b.slices})}
           for det in range(n_det)]
    rng = np.random.default_rng(1000 * cfg_no + 7)
    per_s = f0 // B                                                                # pushes per second
    worst, n_checked, agree = 0.0, 0, []
    for bi in check_banks:
        bank = keep[bi]
        mine = [i for i in injs if i.bank == bi]
        # seconds to check: those holding an injection of this bank; else the last `tail_pushes` seconds
        secs = sorted({i.k0 // f0 for i in mine}) or list(range(S - tail_pushes, S))
        want = {p for s in secs for p in range(s * per_s, (s + 1) * per_s)}
        snr_dev = torch.zeros((len(want), n_det, 2 * bank.M, B), dtype=torch.float32, device="cuda")
        pk_dev = torch.zeros((len(want),) + tuple(st.peaks_dev.shape), dtype=torch.int32, device="cuda")
        st.reset()
        slot = {}
        for p in range(n_push):
            if p in want:
                slot[p] = len(slot)
                lib.lloid_stream_push(st.handle, dev_strain[p].data_ptr(), pk_dev[slot[p]].data_ptr(), snr_dev[slot[p]].data_ptr(), bi)
            else:
                st.push_device(dev_strain[p])
        torch.cuda.synchronize()
        rho_all = snr_dev.cpu().numpy()
        pk_all = pk_dev.cpu().numpy().view(lib.PEAK_DTYPE).reshape(len(want), n_det, st.Mtot)[:, :, off[bi]:off[bi + 1]]
        del snr_dev, pk_dev
        for s in secs:
            k_lo, k_hi = s * f0, (s + 1) * f0
            sl = [slot[p] for p in range(s * per_s, (s + 1) * per_s)]
            for det in range(n_det):
                rho_gpu = np.concatenate([rho_all[i, det] for i in sl], axis=1)   # [2M][f0]
                ref = lloid_snr(bank, strain[det], k_lo, k_hi, decimated=dec[det])
                # sampled rows element by element (the whole block is available: also gate the full block)
                inj_here = [i for i in mine if i.det == det and i.k0 // f0 == s]
                tmpl = sorted({i.template for i in inj_here} | set(rng.choice(bank.M, n_rows, replace=False).tolist()))
                rows = [r for j in tmpl for r in (2 * j, 2 * j + 1)]
                e_rows, _ = snr_errors(rho_gpu[rows], ref[rows])
                e_all, e_rms = snr_errors(rho_gpu, ref)
                worst = max(worst, e_rows, e_all)
                assert e_rows <= TOL[2] and e_all <= TOL[2], f"config {cfg_no} bank {bi} det {det} second {s}: {e_rows:.3e} / {e_all:.3e}"
                # all templates' peaks, per pushed buffer of this second
                must = [((i.k0 % f0) // B, i.template) for i in inj_here if i.amp >= 8.0]
                pk = np.stack([pk_all[i, det] for i in sl])                         # [per_s][M]
                agree.append(check_peaks(pk, ref, B, TOL[2], must))
                snr_o, idx_o, _ = find_peaks(ref, B)
                for i in inj_here:                                                  # and the oracle does see the injection:
                    # loud within a few ms of the injected sample (heavy, narrow-band templates peak several samples off
                    # it in N(0,1) noise, possibly in the neighbouring buffer -- the bit-exact check above is GPU vs oracle)
                    a, b = max(i.k0 % f0 - 16, 0), min(i.k0 % f0 + 17, f0)
                    z = ref[2 * i.template, a:b] + 1j * ref[2 * i.template + 1, a:b]
                    assert np.abs(z).max() > 0.75 * i.amp - 2.0, (bi, det, i.template, i.amp, float(np.abs(z).max()))
                n_checked += 1
    st.close()
    kinds = {b: ("standin" if b in standins else ("injected" if any(i.bank == b for i in injs) else "real")) for b in check_banks}
    print(f"config {cfg_no}: {c.n_banks} banks x {c.M} templates x {n_det} det, {n_push} pushes of {B}; checked banks {kinds}; "
          f"{n_checked} (bank, det, second) blocks; worst err {worst:.2e} of SNR rms (gate {TOL[2]}); "
          f"peak sample agreement {np.mean(agree):.4f}; injections checked {len(injs)}")
    assert len(check_banks) >= (5 if c.n_banks > 8 else c.n_banks)


def test_config2_full_size_live_history():
    _fullsize(2)


def test_config3_full_size_live_history():
    _fullsize(3)


def test_config4_full_size_live_history():
    _fullsize(4)


def test_config5_full_size_live_history():
    _fullsize(5)
