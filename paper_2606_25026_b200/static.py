"""ctypes binding of include/wdm_static.h: the one entry point of libwdm.so that allocates nothing (the deterministic
particle deposit with its accumulator mesh in a static device array; N <= WDM_STATIC_MAX_N).  Argument marshalling only.
"""
from __future__ import annotations

import ctypes as C

from . import WDM_C64, WDM_C128, WdmError, lib

WDM_STATIC_MAX_N = 64
EXPORTS = ["wdm_deposit_static", "wdm_static_scratch_bytes", "wdm_static_last_error"]
_ready = False


def _lib():
    global _ready
    L = lib()
    if not _ready:
        vp, i, d = C.c_void_p, C.c_int, C.c_double
        L.wdm_deposit_static.argtypes = [vp, vp, d, C.c_longlong, i, d, i, i, d, vp, vp]
        L.wdm_deposit_static.restype = i
        L.wdm_static_scratch_bytes.argtypes = []
        L.wdm_static_scratch_bytes.restype = C.c_size_t
        L.wdm_static_last_error.argtypes = []
        L.wdm_static_last_error.restype = C.c_char_p
        _ready = True
    return L


def wdm_static_scratch_bytes():
    return int(_lib().wdm_static_scratch_bytes())


def wdm_static_last_error():
    return (_lib().wdm_static_last_error() or b"").decode()


def _addr(t):
    """Device address of a torch tensor, a raw integer address, or None."""
    if t is None:
        return None
    if isinstance(t, int):
        return C.c_void_p(t)
    assert t.is_cuda and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def wdm_deposit_static(pos, mass, mass_scalar, n, N, L, dtype, order, total_mass, rho_out, stream=None):
    """rho_out (N^3 reals on the device, overwritten) = density of the n particles `pos` ((n, 3) reals on the device);
    mass: n reals on the device or None (then every particle weighs mass_scalar).  Asynchronous on `stream` (a
    torch.cuda.Stream, a raw cudaStream_t, or None = torch's current stream).  Calls that overlap on the GPU race on
    the shared static scratch."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    elif hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    rc = _lib().wdm_deposit_static(_addr(pos), _addr(mass), float(mass_scalar), int(n), int(N), float(L), int(dtype), int(order),
                                   float(total_mass), _addr(rho_out), C.c_void_p(stream))
    if rc != 0:
        raise WdmError(rc, wdm_static_last_error())


__all__ = ["WDM_C64", "WDM_C128", "WDM_STATIC_MAX_N", "EXPORTS", "wdm_deposit_static", "wdm_static_scratch_bytes",
           "wdm_static_last_error"]
