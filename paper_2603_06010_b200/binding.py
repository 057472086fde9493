"""Thin Python binding of the C ABI in include/tdlike.h (argument marshalling only).

Every step of the hot path runs in the CUDA library; this module converts torch tensors /
numpy arrays to raw pointers and sizes.  There is no CPU fallback: if libtdlike.so cannot be
loaded (and cannot be built with nvcc), `load()` raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "lib", "libtdlike.so")

TD_OK, TD_EINVAL, TD_ENOTSPD, TD_ENOMEM, TD_ECUDA, TD_EUNSUPPORTED = range(6)
TD_PATH_AUTO, TD_PATH_FFT, TD_PATH_DENSE, TD_PATH_DOT, TD_PATH_CDO = 0, 1, 2, 3, 4
TD_FAMILY_RINGDOWN, TD_FAMILY_SINE_GAUSSIAN, TD_FAMILY_CHIRP = 0, 1, 2
TD_PREC_F64, TD_PREC_F32 = 0, 1

# every symbol include/tdlike.h declares: name -> (restype, argtypes)
_VP, _I64, _INT, _DP = C.c_void_p, C.c_int64, C.c_int, C.POINTER(C.c_double)
SYMBOLS = {
    "td_create": (_INT, [_DP, C.POINTER(C.c_int64), _INT, _INT, C.POINTER(_VP)]),
    "td_destroy": (_INT, [_VP]),
    "td_loglike_batch": (_INT, [_VP, _VP, _VP, _I64, _I64, _VP, _VP]),
    "td_inner_batch": (_INT, [_VP, _VP, _VP, _I64, _I64, _VP, _VP, _VP]),
    "td_loglike_batch_host": (_INT, [_VP, _VP, _VP, _I64, _I64, _VP, _VP]),
    "td_loglike_family_batch": (_INT, [_VP, _VP, _INT, _VP, _I64, C.c_double, _VP, _VP]),
    "td_loglike_family_batch_host": (_INT, [_VP, _VP, _INT, _VP, _I64, C.c_double, _VP, _VP]),
    "td_reserve": (_INT, [_VP, _I64]),
    "td_set_path": (_INT, [_VP, _INT]),
    "td_set_fft_variant": (_INT, [_VP, _INT]),
    "td_set_precision": (_INT, [_VP, _INT]),
    "td_get_info": (_INT, [_VP, C.POINTER(C.c_int64), C.POINTER(_INT), _DP, _DP, C.POINTER(_INT)]),
    "td_get_generator": (_INT, [_VP, _INT, _DP]),
    "td_last_launches": (_INT, [_VP]),
    "td_strerror": (C.c_char_p, [_INT]),
    "td_loglike_batch_static": (_INT, [_VP, _VP, _VP, _I64, _I64, _VP, _VP]),
    "td_static_setup": (_INT, [_INT]),
    "td_static_scratch_bytes": (C.c_size_t, []),
    "td_static_last_error": (C.c_char_p, []),
}

_lib = None


class TDError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        super().__init__(f"{what}: {strerror(status)} (status {status})")


def load(build_if_missing: bool = True) -> C.CDLL:
    """Load libtdlike.so (building it with nvcc first if it is absent).  Raises on failure."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        if not build_if_missing:
            raise RuntimeError(f"CUDA library missing: {LIB_PATH} (run python -m paper_2603_06010_b200.build)")
        from . import build as _build
        _build.build()
    lib = C.CDLL(LIB_PATH)
    for name, (res, args) in SYMBOLS.items():
        fn = getattr(lib, name)          # AttributeError if the symbol is not exported
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def strerror(status: int) -> str:
    return load().td_strerror(int(status)).decode()


def static_setup(device: int = 0):
    """td_static_setup: resolve the static scratch array's device address on `device` (optional, see include/tdlike.h)."""
    lib = load()
    st = lib.td_static_setup(int(device))
    if st != TD_OK:
        raise TDError(st, "td_static_setup [" + lib.td_static_last_error().decode() + "]")


def static_scratch_bytes() -> int:
    return int(load().td_static_scratch_bytes())


def _check(status: int, what: str):
    if status != TD_OK:
        raise TDError(status, what)


def _ptr(t, name: str, device_index: Optional[int] = None) -> int:
    """Raw device pointer of a float64 torch CUDA tensor."""
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64:
        raise TypeError(f"{name} must be a float64 CUDA tensor")
    if device_index is not None and t.device.index != device_index:
        raise ValueError(f"{name} lives on cuda:{t.device.index}, handle on cuda:{device_index}")
    return t.data_ptr()


def _stream_ptr(stream, device) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream(device)
    return int(stream.cuda_stream)


class TDLikelihood:
    """Handle owner: td_create on construction, td_destroy on close()/GC."""

    def __init__(self, acf, seg_lengths: Sequence[int], device: int = 0):
        lib = load()
        acf = np.ascontiguousarray(np.asarray(acf, dtype=np.float64))
        seg = np.ascontiguousarray(np.asarray(seg_lengths, dtype=np.int64))
        if acf.ndim != 1 or seg.ndim != 1 or (seg.size and int(seg.sum()) != acf.size):
            raise ValueError("acf must be the concatenation of the per-segment ACFs")
        h = _VP()
        st = lib.td_create(acf.ctypes.data_as(_DP), seg.ctypes.data_as(C.POINTER(C.c_int64)), int(seg.size),
                           int(device), C.byref(h))
        _check(st, "td_create")
        self._h = h
        self._lib = lib
        self.device = int(device)
        self.seg_lengths = seg.copy()
        self.n_tot = int(seg.sum())

    # -- lifetime -------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.td_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- hot path -------------------------------------------------------------------------
    def loglike_batch(self, d, H, out=None, stream=None):
        """out[b] = -1/2 sum_s (d_s-h_bs)^T C_s^-1 (d_s-h_bs); d [N_tot], H [B, ldh>=N_tot] CUDA float64."""
        import torch
        if H.dim() != 2 or H.stride(1) != 1:
            raise ValueError("H must be 2-D with unit stride along samples")
        B, ldh = int(H.shape[0]), int(H.stride(0)) if H.shape[0] > 1 else max(int(H.stride(0)), int(H.shape[1]))
        if H.shape[1] < self.n_tot or d.numel() < self.n_tot or not d.is_contiguous():
            raise ValueError("d / H shorter than N_tot")
        if out is None:
            out = torch.empty(B, dtype=torch.float64, device=H.device)
        st = self._lib.td_loglike_batch(self._h, _ptr(d, "d", self.device), _ptr(H, "H", self.device), ldh, B,
                                        _ptr(out, "out", self.device), _stream_ptr(stream, H.device))
        _check(st, "td_loglike_batch")
        return out

    def loglike_batch_static(self, d, H, out, stream=None):
        """td_loglike_batch_static: the same values as loglike_batch, computed without any device allocation - the
        staged kernels with their workspace in the library's 16 MiB static device array (include/tdlike.h: limits,
        calls that overlap on the GPU race).  `out` is the caller's: this wrapper allocates nothing either."""
        if H.dim() != 2 or H.stride(1) != 1:
            raise ValueError("H must be 2-D with unit stride along samples")
        B, ldh = int(H.shape[0]), int(H.stride(0)) if H.shape[0] > 1 else max(int(H.stride(0)), int(H.shape[1]))
        if H.shape[1] < self.n_tot or d.numel() < self.n_tot or not d.is_contiguous() or out.numel() < B:
            raise ValueError("d / H shorter than N_tot, or out shorter than B")
        st = self._lib.td_loglike_batch_static(self._h, _ptr(d, "d", self.device), _ptr(H, "H", self.device), ldh, B,
                                               _ptr(out, "out", self.device), _stream_ptr(stream, H.device))
        if st != TD_OK:
            why = self._lib.td_static_last_error().decode()
            raise TDError(st, "td_loglike_batch_static" + (f" [{why}]" if why else ""))
        return out

    def inner_batch(self, d, H, want_dh: bool = True, want_hh: bool = True, stream=None, out_dh=None):
        """(<d,h_b>, <h_b,h_b>) summed over segments (Eq. 13 terms).  want_hh=False: only the cross term, which
        under TD_PATH_AUTO is one streaming pass over H (u . h_b, u = C^-1 d)."""
        import torch
        B, ldh = int(H.shape[0]), int(H.stride(0)) if H.shape[0] > 1 else max(int(H.stride(0)), int(H.shape[1]))
        dh = (out_dh if out_dh is not None else torch.empty(B, dtype=torch.float64, device=H.device)) if want_dh else None
        hh = torch.empty(B, dtype=torch.float64, device=H.device) if want_hh else None
        st = self._lib.td_inner_batch(self._h, _ptr(d, "d", self.device), _ptr(H, "H", self.device), ldh, B,
                                      _ptr(dh, "dh") if want_dh else None, _ptr(hh, "hh") if want_hh else None,
                                      _stream_ptr(stream, H.device))
        _check(st, "td_inner_batch")
        return dh, hh

    def loglike_batch_host(self, d_host: np.ndarray, H_host, out_host: Optional[np.ndarray] = None, stream=None):
        """Same result from HOST buffers (d, H, out all host memory; H ideally pinned): the library
        streams H to the device in chunks overlapped with the kernels and copies out back."""
        import torch
        if isinstance(H_host, torch.Tensor):
            Hp, B, ldh = H_host.data_ptr(), int(H_host.shape[0]), int(H_host.stride(0))
        else:
            H_host = np.ascontiguousarray(H_host, dtype=np.float64)
            Hp, B, ldh = H_host.ctypes.data, H_host.shape[0], H_host.shape[1]
        d_host = np.ascontiguousarray(d_host, dtype=np.float64)
        if out_host is None:
            out_host = np.empty(B, dtype=np.float64)
        st = self._lib.td_loglike_batch_host(self._h, d_host.ctypes.data, Hp, ldh, B, out_host.ctypes.data,
                                             _stream_ptr(stream, torch.device("cuda", self.device)))
        _check(st, "td_loglike_batch_host")
        return out_host

    def loglike_family_batch(self, d, family: int, params, fs: float, out=None, stream=None):
        """logL of templates of an analytic family (TD_FAMILY_*) given as rows of 5 parameters: CUDA float64 [B, 5]
        (one segment) or [B, n_seg, 5] (one row per template and segment / detector)."""
        import torch
        n_seg = len(self.seg_lengths)
        ok = (params.dim() == 3 and params.shape[1] == n_seg) or (params.dim() == 2 and n_seg == 1)
        if not ok or params.shape[-1] != 5 or not params.is_contiguous():
            raise ValueError(f"params must be a contiguous [B, {n_seg}, 5] tensor")
        B = int(params.shape[0])
        if out is None:
            out = torch.empty(B, dtype=torch.float64, device=params.device)
        st = self._lib.td_loglike_family_batch(self._h, _ptr(d, "d", self.device), int(family),
                                               _ptr(params, "params", self.device), B, float(fs),
                                               _ptr(out, "out", self.device), _stream_ptr(stream, params.device))
        _check(st, "td_loglike_family_batch")
        return out

    def loglike_family_batch_host(self, d_host: np.ndarray, family: int, params_host: np.ndarray, fs: float,
                                  out_host: Optional[np.ndarray] = None, stream=None):
        """Same from HOST arrays: 5 doubles per template cross the bus instead of N."""
        import torch
        params_host = np.ascontiguousarray(params_host, dtype=np.float64)
        d_host = np.ascontiguousarray(d_host, dtype=np.float64)
        if params_host.shape[-1] != 5 or params_host.size != params_host.shape[0] * len(self.seg_lengths) * 5:
            raise ValueError("params must have shape [B, n_seg, 5]")
        B = int(params_host.shape[0])
        if out_host is None:
            out_host = np.empty(B, dtype=np.float64)
        st = self._lib.td_loglike_family_batch_host(self._h, d_host.ctypes.data, int(family), params_host.ctypes.data, B,
                                                    float(fs), out_host.ctypes.data,
                                                    _stream_ptr(stream, torch.device("cuda", self.device)))
        _check(st, "td_loglike_family_batch_host")
        return out_host

    # -- options / queries ---------------------------------------------------------------
    def reserve(self, B_max: int):
        """Size every batch-dependent buffer for calls of up to B_max templates (td_reserve)."""
        _check(self._lib.td_reserve(self._h, int(B_max)), "td_reserve")

    def set_path(self, path: int):
        _check(self._lib.td_set_path(self._h, int(path)), "td_set_path")

    def set_precision(self, precision: int):
        """TD_PREC_F64 (default) or TD_PREC_F32: fp32 evaluation with fp64 setup (td_set_precision)."""
        _check(self._lib.td_set_precision(self._h, int(precision)), "td_set_precision")

    def set_fft_variant(self, variant: int):
        _check(self._lib.td_set_fft_variant(self._h, int(variant)), "td_set_fft_variant")

    def info(self) -> dict:
        n_seg = len(self.seg_lengths)
        n_tot, ns, lp = C.c_int64(), C.c_int(), C.c_int()
        v = np.empty(n_seg)
        ld = np.empty(n_seg)
        _check(self._lib.td_get_info(self._h, C.byref(n_tot), C.byref(ns), v.ctypes.data_as(_DP),
                                     ld.ctypes.data_as(_DP), C.byref(lp)), "td_get_info")
        return {"n_tot": n_tot.value, "n_seg": ns.value, "v": v, "logdet": ld, "last_path": lp.value}

    def generator(self, seg: int) -> np.ndarray:
        a = np.empty(int(self.seg_lengths[seg]))
        _check(self._lib.td_get_generator(self._h, int(seg), a.ctypes.data_as(_DP)), "td_get_generator")
        return a

    def last_launches(self) -> int:
        return int(self._lib.td_last_launches(self._h))


PROBE_LIB_PATH = os.path.join(_HERE, "lib", "libtdprobe.so")
_probe_lib = None


def probe_throughput(kind: int, device: int = 0) -> float:
    """TFLOP/s of a register-resident loop (0 DFMA, 1 DMMA m8n8k4, 2 both, 3 DADD, 4 FFMA), from the bench-only
    library libtdprobe.so (include/tdprobe.h); not part of the product library."""
    global _probe_lib
    if _probe_lib is None:
        lib = C.CDLL(PROBE_LIB_PATH)
        lib.td_probe_throughput.restype = _INT
        lib.td_probe_throughput.argtypes = [_INT, _INT, _DP]
        _probe_lib = lib
    v = C.c_double()
    _check(_probe_lib.td_probe_throughput(int(kind), int(device), C.byref(v)), "td_probe_throughput")
    return float(v.value)


# C-named convenience wrappers -------------------------------------------------------------
def td_create(acf, seg_lengths, device: int = 0) -> TDLikelihood:
    return TDLikelihood(acf, seg_lengths, device)


def td_loglike_batch(handle: TDLikelihood, d, H, out=None, stream=None):
    return handle.loglike_batch(d, H, out=out, stream=stream)


def td_inner_batch(handle: TDLikelihood, d, H, stream=None):
    return handle.inner_batch(d, H, stream=stream)


def td_destroy(handle: TDLikelihood):
    handle.close()
