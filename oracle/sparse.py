"""ctypes binding of the CPU oracle (TEST INFRASTRUCTURE ONLY; see sv_oracle.cpp)."""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        lib.orc_create.restype = C.c_void_p
        lib.orc_create.argtypes = [C.c_int]
        lib.orc_destroy.argtypes = [C.c_void_p]
        lib.orc_num_terms.restype = C.c_uint64
        lib.orc_num_terms.argtypes = [C.c_void_p]
        lib.orc_load.restype = C.c_int
        lib.orc_load.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64]
        lib.orc_apply_gate.restype = C.c_int
        lib.orc_apply_gate.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        lib.orc_norm.restype = C.c_double
        lib.orc_norm.argtypes = [C.c_void_p]
        lib.orc_truncate.restype = C.c_int
        lib.orc_truncate.argtypes = [C.c_void_p, C.c_uint64, C.c_double, C.c_void_p]
        lib.orc_top.restype = C.c_uint64
        lib.orc_top.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib = lib
    return _lib


class SparseOracle:
    """unordered_map<uint64, complex128> simulator; starts in |0...0>."""

    def __init__(self, n_qubits: int):
        self._lib = _load()
        self.n = int(n_qubits)
        self._h = self._lib.orc_create(self.n)
        if not self._h:
            raise ValueError("bad n_qubits")

    def __del__(self):
        if getattr(self, "_h", None):
            self._lib.orc_destroy(self._h)
            self._h = None

    def num_terms(self) -> int:
        return int(self._lib.orc_num_terms(self._h))

    def load(self, keys, amps):
        keys = np.ascontiguousarray(keys, dtype=np.uint64)
        amps = np.ascontiguousarray(amps, dtype=np.complex128)
        assert keys.shape == amps.shape
        rc = self._lib.orc_load(self._h, keys.ctypes.data, amps.ctypes.data, keys.size)
        if rc != 0:
            raise ValueError("orc_load: duplicate or out-of-range key")

    def apply_gate(self, qubits, U):
        q = np.ascontiguousarray(qubits, dtype=np.int32)
        U = np.ascontiguousarray(U, dtype=np.complex128)
        assert U.shape == (1 << q.size, 1 << q.size)
        rc = self._lib.orc_apply_gate(self._h, q.ctypes.data, int(q.size), U.ctypes.data)
        if rc != 0:
            raise ValueError("orc_apply_gate: invalid argument")

    def truncate(self, max_terms: int = 0, min_mass: float = 1.0) -> float:
        kept = C.c_double(1.0)
        rc = self._lib.orc_truncate(self._h, int(max_terms), float(min_mass), C.byref(kept))
        if rc != 0:
            raise ValueError("orc_truncate: invalid argument")
        return kept.value

    def norm(self) -> float:
        return float(self._lib.orc_norm(self._h))

    def top(self, k: int):
        k = min(int(k), self.num_terms())
        keys = np.empty(k, dtype=np.uint64)
        amps = np.empty(k, dtype=np.complex128)
        probs = np.empty(k, dtype=np.float64)
        w = self._lib.orc_top(self._h, k, keys.ctypes.data, amps.ctypes.data, probs.ctypes.data)
        return keys[:w], amps[:w], probs[:w]

    def export(self):
        """All terms, (p desc, key asc)."""
        return self.top(self.num_terms())

    def as_dict(self):
        k, a, _ = self.export()
        return {int(x): complex(y) for x, y in zip(k, a)}
