"""Gate reordering oracle (TEST INFRASTRUCTURE ONLY).

"We reorder the gates so that, during simulation, the set of currently active qubits is kept as small as possible,
while the introduction of additional qubits is postponed for as long as the circuit dependencies allow ... we only
reorder commuting gates or dependency-compatible gates."  The paper states the goal and gives no algorithm; the reading
taken (R20) is a greedy list schedule, and this oracle follows its statement literally, step by step, from
the pairwise definition (no dependency lists, no counters -- nothing is shared with the library's sv_reorder_gates):

  conflict(h, g)  : h and g share a qubit, and not (h diagonal and g diagonal)
  ready(g)        : g is unscheduled and no unscheduled h < g has conflict(h, g)
  active          : the union of the qubits of the scheduled gates
  step            : schedule the ready g with the fewest qubits outside `active`; ties -> the lowest g.

Pins (tests/test_reorder.py): every conflicting pair keeps its order (checked pair by pair), so the reordered circuit
is the same operator (dense simulator); two interleaved independent circuits come out de-interleaved; a hand-worked
example; idempotence.
"""
import numpy as np


def conflict_matrix(gates, diag=None):
    """gates: sequence of (qubits, U).  C[h, g] = True when gates h and g conflict."""
    n = len(gates)
    diag = [False] * n if diag is None else [bool(d) for d in diag]
    C = np.zeros((n, n), dtype=bool)
    for h in range(n):
        for g in range(n):
            if h != g and set(gates[h][0]) & set(gates[g][0]) and not (diag[h] and diag[g]):
                C[h, g] = True
    return C


def reorder(gates, diag=None):
    """Returns (order, n_active_after): order[t] = index of the gate scheduled t-th."""
    n = len(gates)
    C = conflict_matrix(gates, diag)
    earlier = np.triu(np.ones((n, n), dtype=bool), 1)          # earlier[h, g]: h < g
    blocks = C & earlier
    scheduled = np.zeros(n, dtype=bool)
    active = set()
    order, nact = [], []
    for _ in range(n):
        ready = ~scheduled & ~np.any(blocks[~scheduled, :], axis=0)
        best, best_new = None, None
        for g in np.flatnonzero(ready):
            new = len(set(gates[g][0]) - active)
            if best is None or new < best_new:
                best, best_new = int(g), new
        scheduled[best] = True
        active |= set(gates[best][0])
        order.append(best)
        nact.append(len(active))
    return order, nact
