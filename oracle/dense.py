"""Dense 2^n state-vector simulator (TEST INFRASTRUCTURE ONLY).

The textbook update of PAPER.md Eq. 3 (:33-38) applied, as :47-49 says, to every tuple
of 2^m amplitudes whose basis states differ only in the gate's qubits.  It pins the
sparse oracle for n <= 20.  It is written independently of sv_oracle.cpp: the tuples
are enumerated from the full index space and multiplied with a numpy matmul.

Conventions: qubit q = bit q of the index (R1); local index bit j = bit qubits[j] (R2).
"""
import numpy as np


def ground(n: int) -> np.ndarray:
    psi = np.zeros(1 << n, dtype=np.complex128)
    psi[0] = 1.0
    return psi


def apply_gate(psi: np.ndarray, n: int, qubits, U: np.ndarray) -> np.ndarray:
    qubits = [int(q) for q in qubits]
    m = len(qubits)
    d = 1 << m
    mask = 0
    for q in qubits:
        mask |= 1 << q
    idx = np.arange(1 << n, dtype=np.int64)
    bases = idx[(idx & mask) == 0]                       # one representative per tuple
    offs = np.zeros(d, dtype=np.int64)                   # offs[c] = bits of c scattered to the gate's qubits
    for c in range(d):
        for j, q in enumerate(qubits):
            if (c >> j) & 1:
                offs[c] |= 1 << q
    tup = bases[:, None] | offs[None, :]                 # (2^(n-m), 2^m) indices of each tuple
    out = psi.copy()
    out[tup] = psi[tup] @ np.asarray(U, dtype=np.complex128).T   # new[r] = sum_c U[r, c] old[c]
    return out


def run(n: int, gates) -> np.ndarray:
    psi = ground(n)
    for g in gates:
        psi = apply_gate(psi, n, g.qubits, g.U)
    return psi
