"""Shared helpers of the GPU parity tests: ONE statement of the tolerances (readings 15 and 18).

SNR gate (north star):  max_k |z_gpu[k] - z_oracle[k]|  <=  tol * rms(|z_oracle|)  over the compared block,
tol = 1e-4 (LLOID_PREC_FP32_FFMA), 2e-3 (LLOID_PREC_F16_SPLIT), 1e-2 (single-plane fp16: not a north-star mode).

Peak rule: the GPU takes the first maximum of ITS |z|^2, every sample of which may be off by the SNR gate, so the
oracle's |z| at the GPU's sample can fall short of the oracle's maximum by at most 2 * gate (one gate per sample
compared), and the reported snr / phase are within one gate of the oracle's values AT THAT SAMPLE (phase error times |z|
is an arc length: allowed 2 * gate to cover the chord-to-arc slack).  Injected templates at SNR >= 8: sample bit-exact.
"""
import math

import numpy as np

TOL = {0: 1e-4, 1: 1e-2, 2: 2e-3}


def zc(rho):
    """[2M][n] real rows (2j = Re, 2j+1 = Im) -> complex [M][n]."""
    return rho[0::2] + 1j * rho[1::2]


def snr_errors(rho_gpu, rho_ref):
    """(max, rms) of |z_gpu - z_oracle| in units of rms(|z_oracle|)."""
    z_ref, z_gpu = zc(rho_ref), zc(rho_gpu)
    rms = math.sqrt(np.mean(np.abs(z_ref) ** 2))
    err = np.abs(z_gpu - z_ref)
    return float(err.max() / rms), float(math.sqrt(np.mean(err ** 2)) / rms)


def check_peaks(pk, rho_ref, B, tol, must_match=()):
    """pk: [n_push][M] structured GPU peaks of one bank + detector; rho_ref [2M][n_push*B] float64 oracle SNR.
    Applies the peak rule above with gate = tol * rms(|z_oracle|) of the block.  Returns the fraction of peaks whose
    sample equals the oracle's first maximum."""
    from oracle import find_peaks
    snr, idx, _ = find_peaks(rho_ref, B)
    n_push, M = snr.shape
    z = zc(rho_ref)
    gate = tol * math.sqrt(np.mean(np.abs(z) ** 2))
    for (p, j) in must_match:
        assert pk["sample"][p, j] == idx[p, j], (p, j, int(pk["sample"][p, j]), int(idx[p, j]))
    for p in range(n_push):
        k = pk["sample"][p].astype(np.int64)
        assert (k >= 0).all() and (k < B).all()
        at = z[np.arange(M), p * B + k]
        assert (snr[p] - np.abs(at) <= 2 * gate).all(), f"push {p}: a GPU peak sample is not a maximum of the oracle SNR"
        assert np.abs(pk["snr"][p] - np.abs(at)).max() <= gate, f"push {p}: peak snr"
        dphi = np.angle(np.exp(1j * (pk["phase"][p] - np.angle(at))))
        assert np.abs(dphi * np.abs(at)).max() <= 2 * gate, f"push {p}: peak phase"
    return float(np.mean(pk["sample"] == idx))
