"""Gate fusion oracle (TEST INFRASTRUCTURE ONLY).

"For each block of single- and two-qubit gates ... we fuse those gates into a multi-qubit unitary operation":
the fused operation of a block is, by definition, the operator obtained by applying the block's gates one after the
other.  This oracle writes that definition out: the block's matrix is found COLUMN BY COLUMN by pushing each basis
vector of the block's 2^m-dimensional space through the gates with the dense simulator's gate application
(oracle/dense.py, Eq. 3), the block's qubits relabelled 0..m-1 in order of first appearance.  Nothing is
shared with the library's sv_fuse_gates (which multiplies embedded matrices).

Block formation (the reading taken in DESIGN.md R19, the paper shows blocks only in a figure): greedy over consecutive
gates -- a gate joins the running block while the union of qubits has at most max_m members.
"""
import numpy as np

from . import dense


def blocks_of(gates, max_m=4):
    """gates: sequence of (qubits, U).  Returns a list of lists of gate indices."""
    out, cur, qs = [], [], []
    for i, (q, _) in enumerate(gates):
        new = [x for x in q if x not in qs]
        if cur and len(qs) + len(new) > max_m:
            out.append(cur)
            cur, qs, new = [], [], list(q)
        cur.append(i)
        qs.extend(new)
    if cur:
        out.append(cur)
    return out


def fuse(gates, max_m=4):
    """Returns the fused blocks as a list of (qubits, U)."""
    res = []
    for idxs in blocks_of(gates, max_m):
        qs = []
        for i in idxs:
            qs.extend(x for x in gates[i][0] if x not in qs)
        m = len(qs)
        local = {q: j for j, q in enumerate(qs)}
        U = np.zeros((1 << m, 1 << m), dtype=np.complex128)
        for c in range(1 << m):
            psi = np.zeros(1 << m, dtype=np.complex128)
            psi[c] = 1.0
            for i in idxs:
                q, G = gates[i]
                psi = dense.apply_gate(psi, m, [local[x] for x in q], np.asarray(G, dtype=np.complex128))
            U[:, c] = psi
        res.append((list(qs), U))
    return res
