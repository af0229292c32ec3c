"""Thin Python binding of the C-ABI library (include/sparse_sv.h).

Argument marshalling only: every step of the path runs in the CUDA kernels of
libsparse_sv.so.  PyTorch is used for device memory (the arena tensor) and the stream.
There is no CPU fallback: importing this module without the built library raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libsparse_sv.so")

SV_OK, SV_ERR_INVALID_ARG, SV_ERR_CAPACITY, SV_ERR_NOMEM, SV_ERR_CUDA = 0, -1, -2, -3, -4
_ERRNAME = {-1: "SV_ERR_INVALID_ARG", -2: "SV_ERR_CAPACITY", -3: "SV_ERR_NOMEM", -4: "SV_ERR_CUDA"}
CLASS_NAMES = {0: "none", 1: "diagonal", 2: "xor", 3: "group"}

EXPORTS = ["sv_arena_bytes", "sv_create", "sv_create_in_arena", "sv_destroy", "sv_apply_gate", "sv_truncate",
           "sv_norm", "sv_top", "sv_num_terms", "sv_load", "sv_load_device", "sv_get_stats",
           "sv_check_invariants", "sv_last_error", "sv_sync", "sv_profile", "sv_profile_get", "sv_set_option",
           "sv_apply_gate_truncate", "sv_fuse_gates", "sv_reorder_gates", "sv_apply_circuit"]
TEST_EXPORTS = ["sv_test_set_pre_slack", "sv_test_definite_qubits"]      # include/sparse_sv_test.h
KERNELS = ["diag", "move", "bitpass", "sel_hist", "compact", "classify", "grouppass", "bitpass_gen"]
OPT_SAMPLE_MIN_TERMS = 0
OPT_SMALL_STATE_PATH = 2
OPT_TWO_BIT_PASS = 3


class SvStats(C.Structure):
    _fields_ = [("gate_class", C.c_int), ("m", C.c_int), ("active_bits", C.c_int), ("passes", C.c_int),
                ("n_in", C.c_uint64), ("n_out", C.c_uint64), ("launches", C.c_uint64), ("fallbacks", C.c_uint64),
                ("n_mid", C.c_uint64), ("pre_dropped", C.c_uint64), ("small_gates", C.c_uint64)]


class SvKernelProf(C.Structure):
    _fields_ = [("ms", C.c_double), ("launches", C.c_uint64), ("alg_bytes", C.c_double)]


class SvError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("%s: %s" % (_ERRNAME.get(code, str(code)), msg))
        self.code = code


def load_library(path: str = _LIBPATH):
    if not os.path.exists(path):
        raise ImportError("CUDA library %s is missing: run `python -m paper_2607_07816_b200.build` "
                          "(there is no CPU fallback)" % path)
    lib = C.CDLL(path)
    vp, u64, i32, dbl = C.c_void_p, C.c_uint64, C.c_int, C.c_double
    lib.sv_arena_bytes.restype = C.c_size_t
    lib.sv_arena_bytes.argtypes = [u64]
    lib.sv_create.restype = i32
    lib.sv_create.argtypes = [i32, u64, C.POINTER(vp)]
    lib.sv_create_in_arena.restype = i32
    lib.sv_create_in_arena.argtypes = [i32, u64, vp, C.c_size_t, vp, C.POINTER(vp)]
    lib.sv_destroy.restype = None
    lib.sv_destroy.argtypes = [vp]
    lib.sv_apply_gate.restype = i32
    lib.sv_apply_gate.argtypes = [vp, vp, i32, vp]
    lib.sv_truncate.restype = i32
    lib.sv_truncate.argtypes = [vp, u64, dbl, C.POINTER(dbl)]
    lib.sv_fuse_gates.restype = i32
    lib.sv_fuse_gates.argtypes = [i32, vp, vp, vp, i32, C.POINTER(i32), vp, vp, vp, C.c_size_t]
    lib.sv_reorder_gates.restype = i32
    lib.sv_reorder_gates.argtypes = [i32, vp, vp, vp, vp, vp]
    lib.sv_apply_gate_truncate.restype = i32
    lib.sv_apply_gate_truncate.argtypes = [vp, vp, i32, vp, u64, dbl, C.POINTER(dbl)]
    lib.sv_apply_circuit.restype = i32
    lib.sv_apply_circuit.argtypes = [vp, i32, vp, vp, vp, u64, dbl, vp, C.POINTER(i32)]
    lib.sv_norm.restype = i32
    lib.sv_norm.argtypes = [vp, C.POINTER(dbl)]
    lib.sv_top.restype = i32
    lib.sv_top.argtypes = [vp, u64, vp, vp, vp, C.POINTER(u64)]
    lib.sv_num_terms.restype = i32
    lib.sv_num_terms.argtypes = [vp, C.POINTER(u64)]
    lib.sv_load.restype = i32
    lib.sv_load.argtypes = [vp, vp, vp, u64]
    lib.sv_load_device.restype = i32
    lib.sv_load_device.argtypes = [vp, vp, vp, u64]
    lib.sv_get_stats.restype = i32
    lib.sv_get_stats.argtypes = [vp, C.POINTER(SvStats)]
    lib.sv_check_invariants.restype = i32
    lib.sv_check_invariants.argtypes = [vp, C.POINTER(i32)]
    lib.sv_last_error.restype = C.c_char_p
    lib.sv_last_error.argtypes = [vp]
    lib.sv_sync.restype = i32
    lib.sv_sync.argtypes = [vp]
    lib.sv_profile.restype = i32
    lib.sv_profile.argtypes = [vp, i32]
    lib.sv_profile_get.restype = i32
    lib.sv_profile_get.argtypes = [vp, i32, C.POINTER(SvKernelProf)]
    lib.sv_set_option.restype = i32
    lib.sv_set_option.argtypes = [vp, i32, u64]
    lib.sv_test_set_pre_slack.restype = i32
    lib.sv_test_set_pre_slack.argtypes = [vp, C.c_longlong]
    lib.sv_test_definite_qubits.restype = i32
    lib.sv_test_definite_qubits.argtypes = [vp, C.POINTER(C.c_uint64)]
    return lib


lib = load_library()


def fuse_gates(gates, max_m: int = 4):
    """sv_fuse_gates: gates = sequence of (qubits, U); returns the fused blocks as a list of
    (qubits, U).  Argument marshalling only; the fusion itself is the library's host code."""
    gates = list(gates)
    if not gates:
        return []
    ms = np.array([len(q) for q, _ in gates], dtype=np.int32)
    qs = np.ascontiguousarray(np.concatenate([np.asarray(q, dtype=np.int32) for q, _ in gates]))
    for (q, U), m in zip(gates, ms):
        if np.shape(U) != (1 << m, 1 << m):
            raise ValueError("U must be 2^m x 2^m")
    us = np.ascontiguousarray(np.concatenate([np.asarray(U, dtype=np.complex128).reshape(-1) for _, U in gates]))
    cap = len(gates) << (2 * max_m)
    nb = C.c_int(0)
    bm = np.zeros(len(gates), dtype=np.int32)
    bq = np.zeros(int(ms.sum()), dtype=np.int32)
    bu = np.zeros(cap, dtype=np.complex128)
    rc = lib.sv_fuse_gates(len(gates), ms.ctypes.data, qs.ctypes.data, us.ctypes.data, int(max_m), C.byref(nb),
                           bm.ctypes.data, bq.ctypes.data, bu.ctypes.data, cap)
    if rc != SV_OK:
        raise SvError(rc, "sv_fuse_gates: invalid gate list")
    out, qo, uo = [], 0, 0
    for i in range(nb.value):
        m = int(bm[i])
        out.append(([int(x) for x in bq[qo:qo + m]], bu[uo:uo + (1 << (2 * m))].reshape(1 << m, 1 << m).copy()))
        qo += m; uo += 1 << (2 * m)
    return out


def reorder_gates(gates, diag=None, return_active: bool = False):
    """sv_reorder_gates: gates = sequence of (qubits, U) (U is not looked at); diag = optional sequence
    of flags, True where a gate's matrix is diagonal.  Returns the order (list of indices into `gates`), and with
    return_active also the number of active qubits after each scheduled gate.  Argument marshalling only."""
    gates = list(gates)
    if not gates:
        return ([], []) if return_active else []
    ms = np.array([len(q) for q, _ in gates], dtype=np.int32)
    qs = np.ascontiguousarray(np.concatenate([np.asarray(q, dtype=np.int32) for q, _ in gates]))
    dg = None if diag is None else np.ascontiguousarray(np.asarray(list(diag), dtype=np.uint8))
    if dg is not None and dg.shape != (len(gates),):
        raise ValueError("diag must have one flag per gate")
    order = np.zeros(len(gates), dtype=np.int32)
    act = np.zeros(len(gates), dtype=np.int32)
    rc = lib.sv_reorder_gates(len(gates), ms.ctypes.data, qs.ctypes.data, None if dg is None else dg.ctypes.data,
                              order.ctypes.data, act.ctypes.data)
    if rc != SV_OK:
        raise SvError(rc, "sv_reorder_gates: invalid gate list")
    return (order.tolist(), act.tolist()) if return_active else order.tolist()


class SparseSV:
    """One sparse, truncated state on one GPU.  Starts in |0...0>."""

    def __init__(self, n_qubits: int, capacity: int, device="cuda:0", torch_arena: bool = True):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2607_07816_b200.engine needs a CUDA device (no CPU fallback)")
        self.n = int(n_qubits)
        self.capacity = int(capacity)
        self.device = torch.device(device)
        self._h = C.c_void_p()
        self._arena = None
        torch.cuda.set_device(self.device)
        if torch_arena:
            nbytes = int(lib.sv_arena_bytes(self.capacity))
            self._arena = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            ptr = (self._arena.data_ptr() + 255) & ~255
            self._stream = torch.cuda.current_stream(self.device)
            rc = lib.sv_create_in_arena(self.n, self.capacity, ptr, nbytes, self._stream.cuda_stream, C.byref(self._h))
        else:
            rc = lib.sv_create(self.n, self.capacity, C.byref(self._h))
        if rc != SV_OK:
            raise SvError(rc, "sv_create failed (n=%d capacity=%d)" % (self.n, self.capacity))

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib.sv_destroy(self._h)
            self._h = C.c_void_p()
        self._arena = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc):
        if rc != SV_OK:
            raise SvError(rc, lib.sv_last_error(self._h).decode())

    def apply_gate(self, qubits, U):
        q = np.ascontiguousarray(qubits, dtype=np.int32)
        U = np.ascontiguousarray(U, dtype=np.complex128)
        if U.shape != (1 << q.size, 1 << q.size):
            raise ValueError("U must be 2^m x 2^m")
        self._chk(lib.sv_apply_gate(self._h, q.ctypes.data, int(q.size), U.ctypes.data))

    def apply_gate_truncate(self, qubits, U, max_terms: int = 0, min_mass: float = 1.0) -> float:
        """apply_gate followed by truncate in one call (same result; the engine may skip writing what the cut drops)."""
        q = np.ascontiguousarray(qubits, dtype=np.int32)
        U = np.ascontiguousarray(U, dtype=np.complex128)
        if U.shape != (1 << q.size, 1 << q.size):
            raise ValueError("U must be 2^m x 2^m")
        kept = C.c_double(1.0)
        self._chk(lib.sv_apply_gate_truncate(self._h, q.ctypes.data, int(q.size), U.ctypes.data, int(max_terms), float(min_mass),
                                             C.byref(kept)))
        return kept.value

    def apply_circuit(self, gates, max_terms: int = 0, min_mass: float = 1.0):
        """sv_apply_circuit: gates = sequence of (qubits, U); every gate is followed by truncate(max_terms, min_mass).
        Returns the kept fraction of every step (numpy array).  Argument marshalling only."""
        gates = list(gates)
        if not gates:
            return np.zeros(0)
        ms = np.array([len(q) for q, _ in gates], dtype=np.int32)
        qs = np.ascontiguousarray(np.concatenate([np.asarray(q, dtype=np.int32) for q, _ in gates]))
        for (q, U), m in zip(gates, ms):
            if np.shape(U) != (1 << m, 1 << m):
                raise ValueError("U must be 2^m x 2^m")
        us = np.ascontiguousarray(np.concatenate([np.asarray(U, dtype=np.complex128).reshape(-1) for _, U in gates]))
        kept = np.ones(len(gates), dtype=np.float64)
        done = C.c_int(0)
        self._chk(lib.sv_apply_circuit(self._h, len(gates), ms.ctypes.data, qs.ctypes.data, us.ctypes.data, int(max_terms),
                                       float(min_mass), kept.ctypes.data, C.byref(done)))
        return kept

    def truncate(self, max_terms: int = 0, min_mass: float = 1.0) -> float:
        kept = C.c_double(1.0)
        self._chk(lib.sv_truncate(self._h, int(max_terms), float(min_mass), C.byref(kept)))
        return kept.value

    def norm(self) -> float:
        m = C.c_double(0.0)
        self._chk(lib.sv_norm(self._h, C.byref(m)))
        return m.value

    def num_terms(self) -> int:
        n = C.c_uint64(0)
        self._chk(lib.sv_num_terms(self._h, C.byref(n)))
        return int(n.value)

    def top(self, k: int):
        k = min(int(k), self.num_terms())
        keys = np.empty(k, dtype=np.uint64)
        amps = np.empty(k, dtype=np.complex128)
        probs = np.empty(k, dtype=np.float64)
        w = C.c_uint64(0)
        self._chk(lib.sv_top(self._h, k, keys.ctypes.data, amps.ctypes.data, probs.ctypes.data, C.byref(w)))
        w = int(w.value)
        return keys[:w], amps[:w], probs[:w]

    def export(self):
        """All terms in (p desc, key asc) order (host arrays)."""
        return self.top(self.num_terms())

    def load(self, keys, amps):
        keys = np.ascontiguousarray(keys, dtype=np.uint64)
        amps = np.ascontiguousarray(amps, dtype=np.complex128)
        if keys.shape != amps.shape:
            raise ValueError("keys / amps shape mismatch")
        self._chk(lib.sv_load(self._h, keys.ctypes.data, amps.ctypes.data, int(keys.size)))

    def load_device(self, keys_t, amps_t):
        """keys_t: torch int64/uint64 CUDA tensor; amps_t: torch complex128 CUDA tensor."""
        n = int(keys_t.numel())
        assert amps_t.numel() == n and keys_t.is_cuda and amps_t.is_cuda
        assert keys_t.is_contiguous() and amps_t.is_contiguous()
        self._chk(lib.sv_load_device(self._h, keys_t.data_ptr(), amps_t.data_ptr(), n))

    def stats(self) -> dict:
        st = SvStats()
        self._chk(lib.sv_get_stats(self._h, C.byref(st)))
        return {"class": CLASS_NAMES.get(st.gate_class, "?"), "m": st.m, "active_bits": st.active_bits,
                "passes": st.passes, "n_in": int(st.n_in), "n_out": int(st.n_out), "launches": int(st.launches),
                "fallbacks": int(st.fallbacks), "n_mid": int(st.n_mid), "pre_dropped": int(st.pre_dropped),
                "small_gates": int(st.small_gates)}

    def set_option(self, option: int, value: int):
        self._chk(lib.sv_set_option(self._h, int(option), int(value)))

    def test_set_pre_slack(self, slack: int):
        """Test hook (include/sparse_sv_test.h)."""
        self._chk(lib.sv_test_set_pre_slack(self._h, int(slack)))

    def test_definite_qubits(self) -> int:
        """Test hook (include/sparse_sv_test.h): bit q set iff qubit q has the same value in every term."""
        m = C.c_uint64(0)
        self._chk(lib.sv_test_definite_qubits(self._h, C.byref(m)))
        return int(m.value)

    def check_invariants(self) -> bool:
        ok = C.c_int(0)
        self._chk(lib.sv_check_invariants(self._h, C.byref(ok)))
        return bool(ok.value)

    def profile(self, enable: bool = True):
        self._chk(lib.sv_profile(self._h, 1 if enable else 0))

    def profile_get(self) -> dict:
        out = {}
        for i, name in enumerate(KERNELS):
            kp = SvKernelProf()
            self._chk(lib.sv_profile_get(self._h, i, C.byref(kp)))
            out[name] = {"ms": kp.ms, "launches": int(kp.launches), "alg_bytes": kp.alg_bytes}
        return out

    def sync(self):
        self._chk(lib.sv_sync(self._h))
