"""ctypes binding of the C ABI in include/lloid.h — argument marshalling only.

Every function here has the name and meaning of its C counterpart; all arithmetic of the hot path
runs in liblloid.so's CUDA kernels.  There is no CPU fallback: if the shared library is missing
the import of this module's ``lib()`` raises, and on a box without an sm_100 GPU
``lloid_bank_create`` fails with LLOID_ECUDA.

``Bank`` is a small convenience wrapper (create/upload/finalize from a ``workloads.Workload``)
used by the tests and bench.py; it calls only the functions below.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblloid.so")

LLOID_F32, LLOID_F16, LLOID_BF16 = 0, 1, 2
LLOID_OK, LLOID_EINVAL, LLOID_ENOMEM, LLOID_ECUDA, LLOID_ESTATE, LLOID_EOVERFLOW = 0, -1, -2, -3, -4, -5


class lloid_bank_config_t(C.Structure):
    _fields_ = [("n_bins", C.c_int32), ("n_detectors", C.c_int32), ("full_rate_hz", C.c_int32),
                ("peak_window", C.c_int32), ("snr_threshold", C.c_float), ("k_down", C.c_int32),
                ("k_up", C.c_int32), ("precision", C.c_int32), ("device", C.c_int32),
                ("max_chunk", C.c_int32)]


class lloid_bin_desc_t(C.Structure):
    _fields_ = [("n_templates", C.c_int32), ("n_slices", C.c_int32), ("template_len", C.c_int64)]


class lloid_slice_desc_t(C.Structure):
    _fields_ = [("rate_hz", C.c_int32), ("n_taps", C.c_int32), ("n_basis", C.c_int32),
                ("reserved", C.c_int32), ("end_delay", C.c_int64)]


class lloid_trigger_t(C.Structure):
    _fields_ = [("bin", C.c_int32), ("detector", C.c_int32), ("template_idx", C.c_int32),
                ("reserved", C.c_int32), ("sample", C.c_int64), ("snr_re", C.c_float),
                ("snr_im", C.c_float)]


TRIGGER_DTYPE = np.dtype([("bin", "<i4"), ("detector", "<i4"), ("template_idx", "<i4"), ("reserved", "<i4"),
                          ("sample", "<i8"), ("snr_re", "<f4"), ("snr_im", "<f4")])
assert TRIGGER_DTYPE.itemsize == C.sizeof(lloid_trigger_t) == 32

EXPORTS = {
    "lloid_bank_create": (C.c_int, [C.POINTER(C.c_void_p), C.POINTER(lloid_bank_config_t),
                                    C.POINTER(lloid_bin_desc_t), C.POINTER(C.POINTER(lloid_slice_desc_t))]),
    "lloid_bank_upload_slice": (C.c_int, [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]),
    "lloid_bank_upload_slice_shared": (C.c_int, [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]),
    "lloid_bank_alias_bin": (C.c_int, [C.c_void_p, C.c_int32, C.c_int32]),
    "lloid_bank_finalize": (C.c_int, [C.c_void_p]),
    "lloid_filter": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]),
    "lloid_filter_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]),
    "lloid_check_count": (C.c_int, [C.c_int64, C.c_int64]),
    "lloid_reset": (C.c_int, [C.c_void_p, C.c_void_p]),
    "lloid_debug_capture": (C.c_int, [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_int64, C.c_void_p]),
    "lloid_samples_consumed": (C.c_int64, [C.c_void_p]),
    "lloid_chunk_samples": (C.c_int64, [C.c_void_p]),
    "lloid_last_launch_count": (C.c_int64, [C.c_void_p]),
    "lloid_device_bytes": (C.c_int64, [C.c_void_p]),
    "lloid_path_info": (C.c_int, [C.c_void_p, C.POINTER(C.c_int32)]),
    "lloid_graph_safe": (C.c_int, [C.c_void_p, C.c_int64]),
    "lloid_graph_advance": (C.c_int, [C.c_void_p, C.c_int64]),
    "lloid_set_profiling": (C.c_int, [C.c_void_p, C.c_int32]),
    "lloid_last_stage_ms": (C.c_int, [C.c_void_p, C.POINTER(C.c_float)]),
    "lloid_coincidence_scratch_bytes": (C.c_int64, [C.c_void_p, C.c_int64, C.c_int64]),
    "lloid_coincidence": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_int64,
                                    C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]),
    "lloid_noalloc_max_records": (C.c_int64, []),
    "lloid_noalloc_setup": (C.c_int, []),
    "lloid_window_peaks_noalloc": (C.c_int, [C.c_void_p, C.c_int32, C.c_int64, C.c_int64, C.c_int64, C.c_int32, C.c_float, C.c_int32,
                                             C.c_int32, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]),
    "lloid_destroy": (None, [C.c_void_p]),
    "lloid_last_error": (C.c_char_p, []),
    "lloid_version": (C.c_char_p, []),
}

_lib = None


def lib() -> C.CDLL:
    """Load liblloid.so (built in-tree by ``python -m paper_2410_16416_b200.build``)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2410_16416_b200.build` "
                               "(there is no CPU fallback)")
        h = C.CDLL(LIB_PATH)
        for name, (res, args) in EXPORTS.items():
            fn = getattr(h, name)
            fn.restype, fn.argtypes = res, args
        _lib = h
    return _lib


class LloidError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"lloid error {code}: {msg}")
        self.code = code


def _check(code: int) -> None:
    if code != LLOID_OK:
        raise LloidError(code, lib().lloid_last_error().decode())


def lloid_last_error() -> str:
    return lib().lloid_last_error().decode()


def lloid_version() -> str:
    return lib().lloid_version().decode()


def lloid_bank_create(cfg: lloid_bank_config_t, bins: Sequence[lloid_bin_desc_t],
                      slices: Sequence[Sequence[lloid_slice_desc_t]]) -> C.c_void_p:
    nb = len(bins)
    bins_arr = (lloid_bin_desc_t * nb)(*bins)
    keep = [(lloid_slice_desc_t * len(s))(*s) for s in slices]
    ptrs = (C.POINTER(lloid_slice_desc_t) * nb)(*[C.cast(k, C.POINTER(lloid_slice_desc_t)) for k in keep])
    out = C.c_void_p()
    _check(lib().lloid_bank_create(C.byref(out), C.byref(cfg), bins_arr, ptrs))
    return out


def _f64(a: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def lloid_bank_upload_slice(bank, bin_: int, detector: int, slice_: int, basis: np.ndarray, recon: np.ndarray) -> None:
    b, r = _f64(basis), _f64(recon)
    _check(lib().lloid_bank_upload_slice(bank, bin_, detector, slice_, b.ctypes.data, r.ctypes.data))


def lloid_bank_upload_slice_shared(bank, bin_: int, slice_: int, basis: np.ndarray, recon: np.ndarray) -> None:
    b, r = _f64(basis), _f64(recon)
    _check(lib().lloid_bank_upload_slice_shared(bank, bin_, slice_, b.ctypes.data, r.ctypes.data))


def lloid_bank_alias_bin(bank, dst_bin: int, src_bin: int) -> None:
    _check(lib().lloid_bank_alias_bin(bank, dst_bin, src_bin))


def lloid_bank_finalize(bank) -> None:
    _check(lib().lloid_bank_finalize(bank))


def lloid_filter(bank, strain_dev_ptr: int, n_samples: int, triggers_dev_ptr: int, capacity: int,
                 n_triggers_dev_ptr: int, cuda_stream: int = 0) -> None:
    _check(lib().lloid_filter(bank, strain_dev_ptr, n_samples, triggers_dev_ptr, capacity,
                              n_triggers_dev_ptr, cuda_stream))


def lloid_filter_host(bank, strain_host_ptr: int, n_samples: int, triggers_host_ptr: int, capacity: int,
                      n_triggers_host_ptr: int, cuda_stream: int = 0) -> int:
    """Returns the status code (LLOID_OK or LLOID_EOVERFLOW); raises on any other error."""
    rc = lib().lloid_filter_host(bank, strain_host_ptr, n_samples, triggers_host_ptr, capacity,
                                 n_triggers_host_ptr, cuda_stream)
    if rc not in (LLOID_OK, LLOID_EOVERFLOW):
        _check(rc)
    return rc


def lloid_check_count(count: int, capacity: int) -> int:
    return lib().lloid_check_count(count, capacity)


def lloid_reset(bank, cuda_stream: int = 0) -> None:
    _check(lib().lloid_reset(bank, cuda_stream))


def lloid_debug_capture(bank, bin_: int, detector: int, k_begin: int, n: int, snr_dev_ptr: Optional[int]) -> None:
    _check(lib().lloid_debug_capture(bank, bin_, detector, k_begin, n, snr_dev_ptr or None))


def lloid_samples_consumed(bank) -> int:
    return lib().lloid_samples_consumed(bank)


def lloid_chunk_samples(bank) -> int:
    return lib().lloid_chunk_samples(bank)


def lloid_last_launch_count(bank) -> int:
    return lib().lloid_last_launch_count(bank)


def lloid_device_bytes(bank) -> int:
    return lib().lloid_device_bytes(bank)


def lloid_graph_safe(bank, n_samples: int) -> bool:
    return bool(lib().lloid_graph_safe(bank, n_samples))


def lloid_graph_advance(bank, n_samples: int) -> None:
    _check(lib().lloid_graph_advance(bank, n_samples))


def lloid_path_info(bank) -> dict:
    out = (C.c_int32 * 4)()
    _check(lib().lloid_path_info(bank, out))
    return dict(tensor_recon=bool(out[0]), r_in_tmem=bool(out[1]), cuda_core_bds=int(out[2]), folded_slices=int(out[3]))


COINC_DTYPE = np.dtype([("a", "<i8"), ("b", "<i8")])


def lloid_coincidence_scratch_bytes(bank, k_begin: int, n_samples: int) -> int:
    return lib().lloid_coincidence_scratch_bytes(bank, k_begin, n_samples)


def lloid_coincidence(bank, triggers_dev_ptr: int, n_triggers: int, k_begin: int, n_samples: int, max_dt: np.ndarray,
                      scratch_dev_ptr: int, scratch_bytes: int, pairs_dev_ptr: int, capacity: int, n_pairs_dev_ptr: int,
                      cuda_stream: int = 0) -> None:
    dt = np.ascontiguousarray(max_dt, dtype=np.int32)
    _check(lib().lloid_coincidence(bank, triggers_dev_ptr, n_triggers, k_begin, n_samples, dt.ctypes.data, scratch_dev_ptr,
                                   scratch_bytes, pairs_dev_ptr, capacity, n_pairs_dev_ptr, cuda_stream))


def lloid_noalloc_max_records() -> int:
    return lib().lloid_noalloc_max_records()


def lloid_noalloc_setup() -> None:
    _check(lib().lloid_noalloc_setup())


def lloid_window_peaks_noalloc(snr_dev_ptr: int, n_templates: int, n_samples: int, row_stride: int, k_begin: int,
                               peak_window: int, snr_threshold: float, bin_: int, detector: int, triggers_dev_ptr: int,
                               capacity: int, n_triggers_dev_ptr: int, cuda_stream: int = 0) -> None:
    _check(lib().lloid_window_peaks_noalloc(snr_dev_ptr, n_templates, n_samples, row_stride, k_begin, peak_window,
                                            snr_threshold, bin_, detector, triggers_dev_ptr, capacity,
                                            n_triggers_dev_ptr, cuda_stream))


def lloid_set_profiling(bank, enable: bool) -> None:
    _check(lib().lloid_set_profiling(bank, 1 if enable else 0))


def lloid_last_stage_ms(bank) -> np.ndarray:
    out = (C.c_float * 6)()
    _check(lib().lloid_last_stage_ms(bank, out))
    return np.array(list(out), dtype=np.float64)


def lloid_destroy(bank) -> None:
    lib().lloid_destroy(bank)


# --------------------------------------------------------------------------------------------------
# convenience wrapper: marshals a workloads.Workload into the calls above (no arithmetic)
# --------------------------------------------------------------------------------------------------
class Bank:
    def __init__(self, workload, precision: int = LLOID_F32, device: int = 0, max_chunk: int = 0,
                 bins: Optional[Sequence[int]] = None):
        """``bins``: optional subset of workload.bins (bin shard of this rank); indices are local."""
        w = workload
        self.workload = w
        self.bin_ids = list(range(len(w.bins))) if bins is None else list(bins)
        cfg = lloid_bank_config_t(len(self.bin_ids), w.n_detectors, w.f0, w.peak_window, w.threshold,
                                  w.k_down, w.k_up, precision, device, max_chunk)
        descs, sl = [], []
        for gb in self.bin_ids:
            b = w.bins[gb]
            descs.append(lloid_bin_desc_t(b.n_templates, len(b.slices), b.template_len))
            sl.append([lloid_slice_desc_t(s.rate, s.n_taps, s.n_basis, 0, s.end_delay) for s in b.slices])
        self.handle = lloid_bank_create(cfg, descs, sl)
        first_of = {}
        for lb, gb in enumerate(self.bin_ids):
            b = w.bins[gb]
            if id(b) in first_of:                     # replicated bin object: share device arrays
                lloid_bank_alias_bin(self.handle, lb, first_of[id(b)])
                continue
            first_of[id(b)] = lb
            for s in range(len(b.slices)):
                lloid_bank_upload_slice_shared(self.handle, lb, s, b.basis[s], b.recon[s])
        lloid_bank_finalize(self.handle)
        self.n_detectors = w.n_detectors

    def close(self):
        if self.handle is not None:
            lloid_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def filter(self, strain_dev, triggers_dev, count_dev, stream: int = 0) -> None:
        """strain_dev: torch float32 CUDA tensor [D, n]; triggers_dev: uint8 CUDA tensor of 32*capacity bytes;
        count_dev: int64 CUDA tensor [1].  Asynchronous."""
        assert strain_dev.is_cuda and strain_dev.is_contiguous() and strain_dev.shape[0] == self.n_detectors
        cap = triggers_dev.numel() * triggers_dev.element_size() // 32
        lloid_filter(self.handle, strain_dev.data_ptr(), strain_dev.shape[1], triggers_dev.data_ptr(), cap,
                     count_dev.data_ptr(), stream)

    def filter_host(self, strain_host: np.ndarray, triggers_host: np.ndarray, stream: int = 0):
        """strain_host float32 [D, n] (pinned or pageable), triggers_host: np array of TRIGGER_DTYPE.
        Returns (count, status)."""
        assert strain_host.dtype == np.float32 and strain_host.flags.c_contiguous
        cnt = np.zeros(1, dtype=np.int64)
        rc = lloid_filter_host(self.handle, strain_host.ctypes.data, strain_host.shape[1],
                               triggers_host.ctypes.data, len(triggers_host), cnt.ctypes.data, stream)
        return int(cnt[0]), rc
