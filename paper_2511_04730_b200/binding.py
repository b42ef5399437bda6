"""Thin ctypes binding of liblloid.so (include/lloid.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; PyTorch is used here for device memory and
streams.  There is no CPU fallback: importing this module without the built library raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblloid.so")

LLOID_OK, LLOID_EINVAL, LLOID_ELATENCY, LLOID_ENOMEM, LLOID_ECUDA, LLOID_ESTATE = 0, -1, -2, -3, -4, -5
LLOID_PREC_FP32_FFMA, LLOID_PREC_F16, LLOID_PREC_F16_SPLIT = 0, 1, 2

PEAK_DTYPE = np.dtype([("snr", np.float32), ("sample", np.int32), ("phase", np.float32)])
LLOID_MAX_DET = 4
LLOID_NO_TRIGGER = -2147483648
EVENT_DTYPE = np.dtype([("template_index", np.int32), ("det_mask", np.int32), ("net_snr", np.float32), ("reserved", np.int32),
                        ("snr", np.float32, (LLOID_MAX_DET,)), ("sample", np.int32, (LLOID_MAX_DET,)), ("phase", np.float32, (LLOID_MAX_DET,))])


class lloid_slice(C.Structure):
    _fields_ = [("rate_hz", C.c_int32), ("n_taps", C.c_int32), ("n_basis", C.c_int32), ("delay", C.c_int64),
                ("basis", C.c_void_p), ("recon", C.c_void_p)]


class lloid_options(C.Structure):
    _fields_ = [("n_down", C.c_int32), ("n_up", C.c_int32), ("precision", C.c_int32), ("threshold", C.c_float),
                ("trigger_overlap", C.c_int32)]


class LloidError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"lloid error {code}: {msg}")
        self.code = code


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python paper_2511_04730_b200/build.py` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    sig = {
        "lloid_options_default": (None, [C.POINTER(lloid_options)]),
        "lloid_bank_create": (C.c_int, [C.POINTER(vp), i32, i32, i32, C.POINTER(lloid_slice), C.POINTER(lloid_options)]),
        "lloid_bank_destroy": (None, [vp]),
        "lloid_stream_create": (C.c_int, [C.POINTER(vp), C.POINTER(vp), i32, i32, i32, vp]),
        "lloid_stream_destroy": (None, [vp]),
        "lloid_stream_push": (C.c_int, [vp, vp, vp, vp, i32]),
        "lloid_stream_push_host": (C.c_int, [vp, vp, vp]),
        "lloid_stream_events": (C.c_int, [vp, vp, C.POINTER(i32), vp]),
        "lloid_whitener_create": (C.c_int, [C.POINTER(vp), i32, i32, i32, i32, i32, i32, i32, vp]),
        "lloid_whitener_push": (C.c_int, [vp, vp, vp, vp]),
        "lloid_whitener_reset": (C.c_int, [vp]),
        "lloid_whitener_destroy": (None, [vp]),
        "lloid_whitener_hop_in": (i32, [vp]),
        "lloid_whitener_hop_out": (i32, [vp]),
        "lloid_whitener_psd_bins": (i32, [vp]),
        "lloid_bank_set_autocorrelation": (C.c_int, [vp, vp, i32]),
        "lloid_stream_xi2": (C.c_int, [vp, vp]),
        "lloid_svd_slice": (C.c_int, [vp, i32, i32, C.c_double, i32, C.POINTER(i32), vp, vp, C.POINTER(C.c_double), C.POINTER(C.c_double), vp]),
        "lloid_svd_slice_noalloc": (C.c_int, [vp, i32, i32, C.c_double, i32, C.POINTER(i32), vp, vp, C.POINTER(C.c_double), C.POINTER(C.c_double), vp]),
        "lloid_xi2_series": (C.c_int, [vp, i32, i64, vp, vp, i32, vp, vp]),
        "lloid_stream_push_host_async": (C.c_int, [vp, vp, vp]),
        "lloid_stream_host_sync": (C.c_int, [vp]),
        "lloid_state_reset": (C.c_int, [vp]),
        "lloid_stream_samples_pushed": (i64, [vp]),
        "lloid_stream_total_templates": (i32, [vp]),
        "lloid_stream_launches_per_push": (i32, [vp]),
        "lloid_stream_work_per_push": (C.c_int, [vp, C.POINTER(C.c_double)]),
        "lloid_stream_set_stage_timing": (C.c_int, [vp, i32]),
        "lloid_stream_stage_times": (C.c_int, [vp, C.POINTER(C.c_float)]),
        "lloid_stage_name": (C.c_char_p, [i32]),
        "lloid_last_error": (C.c_char_p, []),
        "lloid_version": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    return lib


_lib = _load()
EXPORTS = ["lloid_options_default", "lloid_bank_create", "lloid_bank_destroy", "lloid_stream_create",
           "lloid_stream_destroy", "lloid_stream_push", "lloid_stream_push_host", "lloid_stream_push_host_async", "lloid_stream_host_sync", "lloid_stream_events", "lloid_xi2_series", "lloid_svd_slice", "lloid_svd_slice_noalloc", "lloid_bank_set_autocorrelation", "lloid_stream_xi2", "lloid_whitener_create", "lloid_whitener_push", "lloid_whitener_reset",
           "lloid_whitener_destroy", "lloid_whitener_hop_in", "lloid_whitener_hop_out", "lloid_whitener_psd_bins", "lloid_state_reset",
           "lloid_stream_samples_pushed", "lloid_stream_total_templates", "lloid_stream_launches_per_push",
           "lloid_stream_work_per_push", "lloid_stream_set_stage_timing", "lloid_stream_stage_times",
           "lloid_stage_name", "lloid_last_error", "lloid_version"]


def lloid_last_error() -> str:
    return _lib.lloid_last_error().decode()


def lloid_version() -> str:
    return _lib.lloid_version().decode()


def _check(rc: int):
    if rc != LLOID_OK:
        raise LloidError(rc, lloid_last_error())


def lloid_options_default() -> lloid_options:
    o = lloid_options()
    _lib.lloid_options_default(C.byref(o))
    return o


def lloid_bank_create(strain_rate_hz: int, n_templates: int, slices: Sequence[dict], precision: Optional[int] = None,
                      threshold: float = 0.0, n_down: int = 32, trigger_overlap: int = 0) -> int:
    """slices: dicts with rate_hz, n_taps, n_basis, delay, basis (float32 [L][N]), recon (float32 [2M][L]);
    arrays are contiguous numpy arrays (host) or torch CUDA tensors (device).  Returns the bank handle."""
    arr = (lloid_slice * len(slices))()
    keep = []
    for i, s in enumerate(slices):
        ptrs = []
        for key in ("basis", "recon"):
            a = s[key]
            if isinstance(a, np.ndarray):
                a = np.ascontiguousarray(a, dtype=np.float32)
                ptrs.append(a.ctypes.data)
            else:   # torch tensor
                a = a.contiguous().float()
                ptrs.append(a.data_ptr())
            keep.append(a)
        arr[i] = lloid_slice(int(s["rate_hz"]), int(s["n_taps"]), int(s["n_basis"]), int(s["delay"]), ptrs[0], ptrs[1])
    opt = lloid_options_default()
    opt.n_down = n_down
    opt.threshold = threshold
    opt.trigger_overlap = trigger_overlap
    if precision is not None:
        opt.precision = precision
    h = C.c_void_p()
    _check(_lib.lloid_bank_create(C.byref(h), strain_rate_hz, n_templates, len(slices), arr, C.byref(opt)))
    return h.value


def lloid_bank_destroy(bank: int):
    _lib.lloid_bank_destroy(bank)


def lloid_stream_create(banks: Sequence[int], n_detectors: int, buffer_len: int, cuda_stream: int = 0) -> int:
    arr = (C.c_void_p * len(banks))(*banks)
    h = C.c_void_p()
    _check(_lib.lloid_stream_create(C.byref(h), arr, len(banks), n_detectors, buffer_len, cuda_stream))
    return h.value


def lloid_stream_destroy(stream: int):
    _lib.lloid_stream_destroy(stream)


def lloid_stream_push(stream: int, strain_ptr: int, peaks_ptr: int, snr_debug_ptr: int = 0, debug_bank: int = 0):
    """Raw device pointers (torch tensors' data_ptr())."""
    _check(_lib.lloid_stream_push(stream, strain_ptr, peaks_ptr, snr_debug_ptr or None, debug_bank))


def lloid_stream_events(stream: int, peaks_ptr: int, dt_samples, events_ptr: int):
    dt = np.ascontiguousarray(dt_samples, dtype=np.int32)
    _check(_lib.lloid_stream_events(stream, peaks_ptr, dt.ctypes.data_as(C.POINTER(C.c_int32)), events_ptr))


def lloid_xi2_series(snr_dev, trigger_sample_dev, acorr_dev, delta: int, cuda_stream: int = 0):
    """torch CUDA tensors: snr float32 [2M][n], trigger_sample int32 [M], acorr float32 [M][2 delta + 1][2] -> xi2 float32 [M]."""
    import torch
    M, n = snr_dev.shape[0] // 2, snr_dev.shape[1]
    assert snr_dev.is_contiguous() and acorr_dev.is_contiguous() and tuple(acorr_dev.shape) == (M, 2 * delta + 1, 2)
    out = torch.empty(M, dtype=torch.float32, device=snr_dev.device)
    _check(_lib.lloid_xi2_series(snr_dev.data_ptr(), M, n, trigger_sample_dev.data_ptr(), acorr_dev.data_ptr(), delta, out.data_ptr(),
                                 cuda_stream))
    return out


def lloid_svd_slice(H: np.ndarray, energy: float = 0.9999, max_basis: Optional[int] = None, device: str = "cuda:0"):
    """Truncated SVD of a slice's template matrix on the GPU: H float64 [2M][N] (host) -> (U float32 [L][N], R float32 [2M][L],
    sigma float64 [L], kept energy)."""
    import torch
    H = np.ascontiguousarray(H, dtype=np.float64)
    n, N = H.shape
    mb = min(n, N) if max_basis is None else max_basis
    dev = torch.device(device)
    torch.cuda.set_device(dev)
    U = torch.empty((mb, N), dtype=torch.float32, device=dev)
    R = torch.empty((n, mb), dtype=torch.float32, device=dev)
    L, kept = C.c_int32(), C.c_double()
    sig = np.zeros(mb)
    _check(_lib.lloid_svd_slice(H.ctypes.data, n, N, energy, mb, C.byref(L), U.data_ptr(), R.data_ptr(),
                                sig.ctypes.data_as(C.POINTER(C.c_double)), C.byref(kept), torch.cuda.current_stream(dev).cuda_stream))
    L = L.value
    return (U.flatten()[:L * N].reshape(L, N).cpu().numpy(), R.flatten()[:n * L].reshape(n, L).cpu().numpy(), sig[:L].copy(), kept.value)


def lloid_svd_slice_noalloc(H_dev, energy: float, U_dev, R_dev, stream: int = 0):
    """lloid_svd_slice without device allocations inside the library: H_dev float64 [n][N], U_dev float32 [max_basis][N] and
    R_dev float32 [n][max_basis] are torch CUDA tensors the CALLER owns (n <= 128, N <= 2048).  Returns (L, sigma [L], kept
    energy); U_dev / R_dev hold U [L][N] and R [n][L] compactly."""
    n, N = H_dev.shape
    mb = U_dev.shape[0]
    L, kept = C.c_int32(), C.c_double()
    sig = np.zeros(mb)
    _check(_lib.lloid_svd_slice_noalloc(H_dev.data_ptr(), n, N, energy, mb, C.byref(L), U_dev.data_ptr(), R_dev.data_ptr(),
                                        sig.ctypes.data_as(C.POINTER(C.c_double)), C.byref(kept), stream))
    return L.value, sig[:L.value].copy(), kept.value


def lloid_stream_push_host_async(stream: int, strain_host_ptr: int, peaks_host_ptr: int):
    _check(_lib.lloid_stream_push_host_async(stream, strain_host_ptr, peaks_host_ptr))


def lloid_stream_host_sync(stream: int):
    _check(_lib.lloid_stream_host_sync(stream))


def lloid_stream_push_host(stream: int, strain_host_ptr: int, peaks_host_ptr: int):
    _check(_lib.lloid_stream_push_host(stream, strain_host_ptr, peaks_host_ptr))


def lloid_state_reset(stream: int):
    _check(_lib.lloid_state_reset(stream))


def lloid_stream_samples_pushed(stream: int) -> int:
    return _lib.lloid_stream_samples_pushed(stream)


def lloid_stream_total_templates(stream: int) -> int:
    return _lib.lloid_stream_total_templates(stream)


def lloid_stream_launches_per_push(stream: int) -> int:
    return _lib.lloid_stream_launches_per_push(stream)


def lloid_stream_work_per_push(stream: int) -> List[float]:
    out = (C.c_double * 8)()
    _check(_lib.lloid_stream_work_per_push(stream, out))
    return list(out)


LLOID_N_STAGES = 5


def lloid_stream_set_stage_timing(stream: int, enable: bool):
    _check(_lib.lloid_stream_set_stage_timing(stream, 1 if enable else 0))


def lloid_stream_stage_times(stream: int):
    """(pushes covered, {stage name: accumulated ms}); synchronises the stream."""
    ms = (C.c_float * LLOID_N_STAGES)()
    n = _lib.lloid_stream_stage_times(stream, ms)
    if n < 0:
        _check(n)
    return n, {_lib.lloid_stage_name(i).decode(): float(ms[i]) for i in range(LLOID_N_STAGES)}


# ---------------------------------------------------------------------------------------------------
# convenience wrappers (still marshalling only)
# ---------------------------------------------------------------------------------------------------
def bank_slices(bank) -> List[dict]:
    """Slice table of a workloads.Bank-like object (attributes f0, M, slices[*].rate/n_taps/delay/U/R)."""
    return [dict(rate_hz=s.rate, n_taps=s.n_taps, n_basis=s.U.shape[0], delay=s.delay,
                 basis=np.ascontiguousarray(s.U, dtype=np.float32), recon=np.ascontiguousarray(s.R, dtype=np.float32))
            for s in bank.slices]


class Whitener:
    """PSD estimation + whitening front end (lloid_whitener_*): torch CUDA tensors in and out."""

    def __init__(self, n_detectors: int, rate_in: int, rate_out: int, fft_len: int, zero_pad: int, n_median: int = 7,
                 n_average: int = 64, device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("Whitener needs a CUDA device (no CPU fallback)")
        self.torch, self.device = torch, torch.device(device)
        torch.cuda.set_device(self.device)
        h = C.c_void_p()
        _check(_lib.lloid_whitener_create(C.byref(h), n_detectors, rate_in, rate_out, fft_len, zero_pad, n_median, n_average,
                                          torch.cuda.current_stream(self.device).cuda_stream))
        self.handle, self.n_det = h.value, n_detectors
        self.hop_in, self.hop_out = _lib.lloid_whitener_hop_in(h), _lib.lloid_whitener_hop_out(h)
        self.psd_bins = _lib.lloid_whitener_psd_bins(h)

    def push(self, strain_dev, want_psd: bool = False):
        t = self.torch
        assert strain_dev.is_cuda and strain_dev.dtype == t.float32 and strain_dev.is_contiguous()
        assert tuple(strain_dev.shape) == (self.n_det, self.hop_in)
        out = t.empty((self.n_det, self.hop_out), dtype=t.float32, device=self.device)
        psd = t.empty((self.n_det, self.psd_bins), dtype=t.float32, device=self.device) if want_psd else None
        _check(_lib.lloid_whitener_push(self.handle, strain_dev.data_ptr(), out.data_ptr(), psd.data_ptr() if want_psd else None))
        return (out, psd) if want_psd else out

    def reset(self):
        _check(_lib.lloid_whitener_reset(self.handle))

    def close(self):
        if self.handle:
            _lib.lloid_whitener_destroy(self.handle)
            self.handle = None


class LloidStream:
    """Owns bank and stream handles plus the torch device buffers a push needs."""

    def __init__(self, banks, n_detectors: int, buffer_len: int, precision: int = LLOID_PREC_F16_SPLIT,
                 threshold: float = 0.0, device: str = "cuda:0", n_down: int = 32, bank_handles=None, Ms=None,
                 trigger_overlap: int = 0, acorr=None):
        """banks: iterable of Bank-like objects (uploaded here, owned by this object), or None with `bank_handles`
        (+ their template counts `Ms`): existing lloid_bank handles owned by the caller (several streams can share them)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("LloidStream needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.n_det, self.B = n_detectors, buffer_len
        self.Ms, self.bank_handles = [], []
        self.owns_banks = bank_handles is None
        if bank_handles is not None:
            self.bank_handles, self.Ms = list(bank_handles), list(Ms)
        else:
            for b in banks:                  # any iterable: a generator lets the caller build banks one at a time
                self.Ms.append(b.M)
                self.bank_handles.append(lloid_bank_create(b.f0, b.M, bank_slices(b), precision, threshold, n_down, trigger_overlap))
                if acorr is not None:       # list of complex [M][2 delta + 1] arrays, one per bank (xi^2 of Eq. 10)
                    a = np.asarray(acorr[len(self.bank_handles) - 1])
                    a32 = np.ascontiguousarray(np.stack([a.real, a.imag], axis=-1), dtype=np.float32)
                    _check(_lib.lloid_bank_set_autocorrelation(self.bank_handles[-1], a32.ctypes.data, (a.shape[1] - 1) // 2))
        self.cuda_stream = torch.cuda.current_stream(self.device)
        self.handle = lloid_stream_create(self.bank_handles, n_detectors, buffer_len, self.cuda_stream.cuda_stream)
        self.Mtot = lloid_stream_total_templates(self.handle)
        self.peaks_dev = torch.zeros((n_detectors, self.Mtot, 3), dtype=torch.int32, device=self.device)
        self.strain_dev = torch.zeros((n_detectors, buffer_len), dtype=torch.float32, device=self.device)
        self.peaks_host = torch.zeros((n_detectors, self.Mtot, 3), dtype=torch.int32).pin_memory()
        self.strain_host = torch.zeros((n_detectors, buffer_len), dtype=torch.float32).pin_memory()

    def push_device(self, strain_dev, snr_debug=None, debug_bank: int = 0):
        """strain_dev: CUDA float32 [n_det][B]; asynchronous.  Returns the device peaks tensor (int32 view)."""
        assert strain_dev.is_cuda and strain_dev.dtype == self.torch.float32 and strain_dev.is_contiguous()
        assert tuple(strain_dev.shape) == (self.n_det, self.B)
        lloid_stream_push(self.handle, strain_dev.data_ptr(), self.peaks_dev.data_ptr(),
                          0 if snr_debug is None else snr_debug.data_ptr(), debug_bank)
        return self.peaks_dev

    def push(self, strain: np.ndarray, want_snr_bank: Optional[int] = None):
        """Host numpy [n_det][B] in, structured peaks [n_det][Mtot] out (and SNR [n_det][2M][B] if asked)."""
        t = self.torch
        self.strain_dev.copy_(t.from_numpy(np.ascontiguousarray(strain, dtype=np.float32)))
        snr = None
        if want_snr_bank is not None:
            snr = t.zeros((self.n_det, 2 * self.Ms[want_snr_bank], self.B), dtype=t.float32, device=self.device)
        self.push_device(self.strain_dev, snr, want_snr_bank or 0)
        t.cuda.synchronize(self.device)
        peaks = self.peaks_dev.cpu().numpy().view(PEAK_DTYPE).reshape(self.n_det, self.Mtot)
        return (peaks, snr.cpu().numpy()) if snr is not None else peaks

    def xi2(self):
        """xi^2 of the triggers of the push before the last one: float32 [n_det][Mtot] (-1 = no trigger)."""
        t = self.torch
        out = t.empty((self.n_det, self.Mtot), dtype=t.float32, device=self.device)
        _check(_lib.lloid_stream_xi2(self.handle, out.data_ptr()))
        t.cuda.synchronize(self.device)
        return out.cpu().numpy()

    def events(self, dt_samples, peaks_dev=None):
        """Coincidence + clustering on the peaks of the last push (device): structured array [n_banks] (EVENT_DTYPE)."""
        t = self.torch
        if not hasattr(self, "events_dev"):
            self.events_dev = t.zeros((len(self.bank_handles), EVENT_DTYPE.itemsize // 4), dtype=t.int32, device=self.device)
        pk = self.peaks_dev if peaks_dev is None else peaks_dev
        lloid_stream_events(self.handle, pk.data_ptr(), dt_samples, self.events_dev.data_ptr())
        t.cuda.synchronize(self.device)
        return self.events_dev.cpu().numpy().view(EVENT_DTYPE).reshape(len(self.bank_handles))

    def push_host(self):
        """End-to-end call on the pinned host buffers self.strain_host -> self.peaks_host (synchronous)."""
        lloid_stream_push_host(self.handle, self.strain_host.data_ptr(), self.peaks_host.data_ptr())
        return self.peaks_host.numpy().view(PEAK_DTYPE).reshape(self.n_det, self.Mtot)

    def push_host_async(self, strain_host, peaks_host):
        """Pipelined end-to-end call: strain_host / peaks_host are PINNED torch tensors the caller keeps alive and does not
        touch until the call after next has returned (or host_sync())."""
        lloid_stream_push_host_async(self.handle, strain_host.data_ptr(), peaks_host.data_ptr())

    def host_sync(self):
        lloid_stream_host_sync(self.handle)

    def reset(self):
        lloid_state_reset(self.handle)

    def work_per_push(self):
        return lloid_stream_work_per_push(self.handle)

    def set_stage_timing(self, enable: bool):
        lloid_stream_set_stage_timing(self.handle, enable)

    def stage_times(self):
        return lloid_stream_stage_times(self.handle)

    @property
    def launches_per_push(self) -> int:
        return lloid_stream_launches_per_push(self.handle)

    def release_banks(self):
        """Hand the bank handles to the caller (who must lloid_bank_destroy them after every stream using them is closed)."""
        self.owns_banks = False
        return list(self.bank_handles), list(self.Ms)

    def close(self):
        if getattr(self, "handle", None):
            lloid_stream_destroy(self.handle)
            self.handle = None
        if getattr(self, "owns_banks", False):
            for b in getattr(self, "bank_handles", []):
                lloid_bank_destroy(b)
        self.bank_handles = []

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
