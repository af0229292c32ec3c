"""Binding of include/sparse_sv_static.h: sv_norm_static, the one entry point that allocates nothing.

Argument marshalling only.  The mass of a device array of complex128 amplitudes (Eq. 4) is computed by two
kernels whose scratch is a static device array inside libsparse_sv.so (8 KiB per GPU, held until exit); the caller
passes the input and the output tensor.  Calls that overlap on the GPU race on that array: keep them on one stream.
"""
import ctypes as C

from .engine import SvError, lib

STATIC_EXPORTS = ["sv_norm_static", "sv_norm_static_init", "sv_static_last_error"]      # include/sparse_sv_static.h
SCRATCH_BYTES = 8192
MAX_TERMS = 1 << 32

lib.sv_norm_static.restype = C.c_int
lib.sv_norm_static.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_void_p]
lib.sv_norm_static_init.restype = C.c_int
lib.sv_norm_static_init.argtypes = []
lib.sv_static_last_error.restype = C.c_char_p
lib.sv_static_last_error.argtypes = []


def _chk(rc):
    if rc != 0:
        raise SvError(rc, lib.sv_static_last_error().decode())


def norm_static_init():
    """Looks up the scratch array's device address for the current device (sv_norm_static does it itself otherwise)."""
    _chk(lib.sv_norm_static_init())


def norm_static_raw(amps_ptr: int, n: int, out_ptr: int, stream_ptr: int = 0):
    """The call itself on raw device addresses; enqueues on `stream_ptr` (a cudaStream_t) and returns."""
    _chk(lib.sv_norm_static(amps_ptr, n, out_ptr, stream_ptr))


def norm_static(amps_t, out_t, stream=None):
    """amps_t: contiguous torch complex128 CUDA tensor; out_t: torch float64 CUDA tensor of one element (written).
    Enqueued on `stream` (default: torch's current stream); no synchronisation."""
    import torch
    assert amps_t.is_cuda and out_t.is_cuda and amps_t.is_contiguous() and out_t.numel() == 1
    assert amps_t.dtype == torch.complex128 and out_t.dtype == torch.float64
    st = stream if stream is not None else torch.cuda.current_stream(amps_t.device)
    with torch.cuda.device(amps_t.device):
        norm_static_raw(amps_t.data_ptr() if amps_t.numel() else 0, int(amps_t.numel()), out_t.data_ptr(), st.cuda_stream)
