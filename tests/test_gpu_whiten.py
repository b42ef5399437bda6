"""GPU parity of the PSD estimation + whitening front end (lloid_whitener_*) against oracle/whiten_oracle.py
(-m gpu): the paper's configuration (16384 -> 2048 Hz, 4 s FFT blocks, 1 s padding, 7-block median)."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _cuda():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _coloured(seed, n, sig):
    from scipy.signal import lfilter
    x = lfilter([1.0, 0.4], [1.0, -0.85], np.random.default_rng(seed).standard_normal(n)) * sig
    return x.astype(np.float32)


@pytest.mark.parametrize("cfg", [(16384, 2048, 65536, 16384, 7, 64, 24), (4096, 1024, 4096, 512, 5, 8, 40)])
def test_whitened_output_and_psd_against_the_oracle(cfg):
    torch = _cuda()
    import paper_2511_04730_b200 as lib
    from oracle import Whitener
    f_in, f_out, N, Z, n_med, n_avg, n_push = cfg
    n_det = 2
    ws = lib.Whitener(n_det, f_in, f_out, N, Z, n_med, n_avg)
    refs = [Whitener(f_in, f_out, N, Z, n_med, n_avg) for _ in range(n_det)]
    assert ws.hop_in == refs[0].hop and ws.hop_out == refs[0].hop_out and ws.psd_bins == refs[0].N_out // 2 + 1
    x = np.stack([_coloured(100 + d, n_push * ws.hop_in, 10.0 ** (d - 1) * 3) for d in range(n_det)])
    worst, worst_psd = 0.0, 0.0
    for p in range(n_push):
        seg = x[:, p * ws.hop_in:(p + 1) * ws.hop_in]
        out, psd = ws.push(torch.from_numpy(np.ascontiguousarray(seg)).cuda(), want_psd=True)
        out, psd = out.cpu().numpy(), psd.cpu().numpy()
        for d in range(n_det):
            want = refs[d].push(seg[d])
            rms = max(math.sqrt(np.mean(want ** 2)), 1e-3)
            worst = max(worst, np.abs(out[d] - want).max() / max(rms, 0.5))
            k = slice(1, ws.psd_bins - 1)
            worst_psd = max(worst_psd, np.abs(psd[d][k] / refs[d].psd[k] - 1).max())
    print(f"whitening {cfg[:4]}: worst output error {worst:.2e} (of the rms), worst relative PSD error {worst_psd:.2e}")
    assert worst < 2e-4 and worst_psd < 2e-4
    # unit variance once the PSD has settled; reset restores the zero-history start
    assert abs(out.var() - 1.0) < 0.3
    ws.reset()
    first = ws.push(torch.from_numpy(np.ascontiguousarray(x[:, :ws.hop_in])).cuda()).cpu().numpy()
    want0 = Whitener(f_in, f_out, N, Z, n_med, n_avg).push(x[0, :ws.hop_in])
    assert np.abs(first[0] - want0).max() < 2e-4 * max(1.0, np.abs(want0).max())
    ws.close()


def test_whitened_strain_feeds_the_filter():
    """Front end + path: coloured detector noise with a chirp -> whitener -> LLOID stream; the SNR series has unit variance
    per quadrature (what Eq. 1's normalisation assumes)."""
    torch = _cuda()
    import paper_2511_04730_b200 as lib
    from workloads import random_bank
    f_in, f_out = 16384, 2048
    ws = lib.Whitener(1, f_in, f_out, 65536, 16384)
    bank = random_bank(9, 32, [(2048, 1024, 16), (512, 512, 12)]).as_f32()
    st = lib.LloidStream([bank], 1, ws.hop_out)
    x = _coloured(7, 40 * ws.hop_in, 5.0)
    vals = []
    for p in range(40):
        wout = ws.push(torch.from_numpy(x[None, p * ws.hop_in:(p + 1) * ws.hop_in].copy()).cuda())
        _, snr = st.push(wout.cpu().numpy(), want_snr_bank=0)
        if p >= 20:
            vals.append(snr[0])
    v = np.concatenate(vals, axis=1).var(axis=1)
    assert abs(v.mean() - 1.0) < 0.1, v.mean()
    ws.close(); st.close()
