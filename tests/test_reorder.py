"""Gate reordering and the ring workload.  CPU: the oracle (oracle/reorder.py)
against what the mathematics fixes -- every conflicting pair keeps its order (pair by pair), the reordered circuit is
the same operator on the dense simulator, two interleaved independent circuits come out one after the other, a
hand-worked example, idempotence -- and the library's host routine sv_reorder_gates against the oracle.  The paper's
claim that reordering + fusion finds the peak with very few terms is checked on the synthetic ring.
GPU: the reordered, fused ring circuit through the fused call against the oracle, step-locked, and free-running."""
import numpy as np
import pytest

from paper_2607_07816_b200 import workloads as W
from oracle import dense, fusion, reorder


def _gates(c):
    return [(list(g.qubits), np.asarray(g.U, dtype=np.complex128)) for g in c.gates]


def _diag(gates):
    return [W.is_diagonal(U) for _, U in gates]


def _assert_valid(gates, dg, order):
    assert sorted(order) == list(range(len(gates)))
    pos = {g: t for t, g in enumerate(order)}
    for h in range(len(gates)):
        for g in range(h + 1, len(gates)):
            if set(gates[h][0]) & set(gates[g][0]) and not (dg[h] and dg[g]):
                assert pos[h] < pos[g], (h, g)


def test_oracle_hand_worked_example():
    """0: H q0   1: H q5   2: CZ(0,1)   3: CZ(1,2)   4: H q1   5: CZ(0,5).
    With diagonal flags: ready {0,1,3}: 0 (1 new, lowest index); ready {1,2,3}: 1 and 2 both add one qubit -> 1;
    ready {2,3,5}: 5 adds none; then 2 (adds q1), 3 (adds q2; 4 waits for 2 and 3), 4.
    Without flags 3 waits for 2 and 5 waits for 2: 0, 1, 2, then 5 (adds none), 3, 4."""
    H, CZ = W.mat_h(), W.mat_diag_minus_last(2)
    gates = [([0], H), ([5], H), ([0, 1], CZ), ([1, 2], CZ), ([1], H), ([0, 5], CZ)]
    order, nact = reorder.reorder(gates, _diag(gates))
    assert order == [0, 1, 5, 2, 3, 4]
    assert nact == [1, 2, 2, 3, 4, 4]
    order, nact = reorder.reorder(gates, None)
    assert order == [0, 1, 2, 5, 3, 4]
    assert nact == [1, 2, 3, 3, 4, 4]


def test_oracle_interleaved_independent_circuits_are_separated():
    rng = np.random.default_rng(0)
    gates = []
    for i in range(12):
        gates.append(([0, 1] if i % 2 == 0 else [1, 2], W.haar_unitary(rng, 4)))     # chain on {0,1,2}: even indices
        gates.append(([3, 4] if i % 2 == 0 else [4, 5], W.haar_unitary(rng, 4)))     # chain on {3,4,5}: odd indices
    order, nact = reorder.reorder(gates)
    assert order == list(range(0, 24, 2)) + list(range(1, 24, 2))
    assert nact == [2] + [3] * 11 + [5] + [6] * 11


@pytest.mark.parametrize("use_diag", [False, True])
def test_oracle_order_is_valid_and_the_same_operator(use_diag):
    c = W.config2(n=10, num_gates=120, seed=11, max_terms=1 << 10)
    gates = _gates(c)
    dg = _diag(gates) if use_diag else [False] * len(gates)
    order, nact = reorder.reorder(gates, dg)
    _assert_valid(gates, dg, order)
    assert order != list(range(len(gates)))
    assert all(a <= b for a, b in zip(nact, nact[1:])) and nact[-1] == len({q for g in gates for q in g[0]})
    psi, phi = dense.ground(10), dense.ground(10)
    for q, U in gates:
        psi = dense.apply_gate(psi, 10, q, U)
    for i in order:
        phi = dense.apply_gate(phi, 10, gates[i][0], gates[i][1])
    assert np.max(np.abs(psi - phi)) <= 1e-13
    # idempotence: the schedule of an already scheduled list is the list
    again, _ = reorder.reorder([gates[i] for i in order], [dg[i] for i in order])
    assert again == list(range(len(gates)))


def test_oracle_postpones_new_qubits():
    """A gate that activates no new qubit is never passed over: whenever a step adds qubits, no ready gate on the
    already active set existed (checked from the definition)."""
    c = W.ring_peaked(n=12, layers=2, seed=3)
    gates = _gates(c)
    dg = _diag(gates)
    order, nact = reorder.reorder(gates, dg)
    _assert_valid(gates, dg, order)
    done, active = set(), set()
    for t, g in enumerate(order):
        new = len(set(gates[g][0]) - active)
        for h in range(len(gates)):
            if h in done:
                continue
            ready = all((e in done) or not (set(gates[e][0]) & set(gates[h][0]) and not (dg[e] and dg[h]))
                        for e in range(h))
            if ready:
                assert len(set(gates[h][0]) - active) >= new
        done.add(g)
        active |= set(gates[g][0])


def test_ring_workload_shape():
    c = W.ring_peaked()
    assert c.n == 44 and len(c.gates) == 4 * 2 * 22 * 3 + 44 + bin(c.secret).count("1")       # 594 with 22 ones
    assert {g.name for g in c.gates} <= {"u3", "cz", "u3_dg", "cz_dg"}
    pairs = {tuple(sorted(g.qubits)) for g in c.gates if g.m == 2}
    assert pairs == {tuple(sorted((a, (a + 1) % 44))) for a in range(44)}                      # the ring, wrap-around included
    X = W.mat_u3(np.pi, 0.0, np.pi)                       # monomial (exact zeros on the diagonal), X up to rounding
    assert X[0, 0] == 0 and X[1, 1] == 0 and np.allclose(X, W.mat_x(), atol=1e-15)
    for g in c.gates:
        assert np.allclose(g.U.conj().T @ g.U, np.eye(1 << g.m), atol=1e-14)
    # small instance on the dense simulator: peaked at the secret
    c = W.ring_peaked(n=10, layers=2, seed=9)
    psi = dense.ground(10)
    for q, U in _gates(c):
        psi = dense.apply_gate(psi, 10, q, U)
    assert int(np.argmax(np.abs(psi) ** 2)) == c.secret


def test_reordering_and_fusion_find_the_peak_with_few_terms():
    """"with this simulation strategy, it is possible to find the correct output bit string ... using a
    very small number of terms (< 2^5)".  On the synthetic ring (n = 44): 64 terms suffice after reordering + fusion,
    while the circuit in file order misses the peak even with 2^10."""
    from oracle.sparse import SparseOracle
    c = W.ring_peaked()
    gates = _gates(c)
    order, _ = reorder.reorder(gates, _diag(gates))

    def run(seq, K):
        o = SparseOracle(c.n)
        for q, U in fusion.fuse(seq, 4):
            o.apply_gate(q, U)
            o.truncate(K, 1.0)
        k, _, p = o.top(1)
        return int(k[0]), float(p[0])

    top, p = run([gates[i] for i in order], 64)
    assert top == c.secret and p > 0.05
    top, _ = run(gates, 1 << 10)
    assert top != c.secret


def test_library_reorder_equals_oracle():
    from paper_2607_07816_b200 import engine
    rng = np.random.default_rng(4)
    for trial in range(6):
        gates = []
        for _ in range(80):
            m = int(rng.integers(1, 4))
            q = [int(x) for x in rng.choice(64 if trial == 0 else 9, size=m, replace=False)]
            U = np.diag(np.exp(1j * rng.uniform(0, 6.28, 1 << m))) if rng.random() < 0.4 else W.haar_unitary(rng, 1 << m)
            gates.append((q, U))
        for dg in (None, _diag(gates)):
            want = reorder.reorder(gates, dg)
            got = engine.reorder_gates(gates, dg, return_active=True)
            assert got[0] == want[0] and got[1] == want[1]
    c = W.ring_peaked()
    gates = _gates(c)
    assert engine.reorder_gates(gates, _diag(gates)) == reorder.reorder(gates, _diag(gates))[0]
    assert engine.reorder_gates([]) == []
    with pytest.raises(engine.SvError):
        engine.reorder_gates([([1, 1], np.eye(4))])
    with pytest.raises(engine.SvError):
        engine.reorder_gates([([64], np.eye(2))])


def _ring_blocks(c):
    from paper_2607_07816_b200 import engine
    gates = _gates(c)
    order = engine.reorder_gates(gates, _diag(gates))
    return engine.fuse_gates([gates[i] for i in order], 4)


@pytest.mark.gpu
def test_gpu_ring_reordered_fused_step_locked():
    """The n = 44 ring, reordered and fused by the library, one fused call per block at K = 2^12, against the oracle
    applying the same block to the same state."""
    from paper_2607_07816_b200 import engine
    from oracle.sparse import SparseOracle
    from util_parity import assert_truncation_parity, MASS_TOL
    K = 1 << 12
    c = W.ring_peaked()
    sv = engine.SparseSV(c.n, 16 * K)
    sv.set_option(engine.OPT_SAMPLE_MIN_TERMS, 512)
    for q, U in _ring_blocks(c):
        k0, a0, _ = sv.export()
        o = SparseOracle(c.n)
        o.load(k0, a0)
        kg = sv.apply_gate_truncate(q, U, K, 1.0)
        o.apply_gate(q, U)
        ko = o.truncate(K, 1.0)
        assert abs(kg - ko) <= MASS_TOL
        assert_truncation_parity(sv.export()[:2], o.export()[:2])
    assert sv.check_invariants()
    keys, _, _ = sv.top(1)
    assert int(keys[0]) == c.secret


@pytest.mark.gpu
@pytest.mark.parametrize("K", [64, 1 << 16])
def test_gpu_ring_free_running_finds_the_secret(K):
    from paper_2607_07816_b200 import engine
    c = W.ring_peaked()
    sv = engine.SparseSV(c.n, 16 * K)
    for q, U in _ring_blocks(c):
        sv.apply_gate_truncate(q, U, K, 1.0)
    keys, _, probs = sv.top(1)
    assert int(keys[0]) == c.secret and float(probs[0]) > 0.05
    assert abs(sv.norm() - 1.0) <= 1e-9
