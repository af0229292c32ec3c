"""Gate fusion.  CPU: the oracle (oracle/fusion.py) against what the
mathematics fixes -- Kronecker products for gates on disjoint qubits, plain matrix products for gates on the same
qubits, unitarity, and the dense simulator run gate by gate -- and the library's host routine sv_fuse_gates against
the oracle.  GPU: fused blocks through the engine against the unfused circuit on the oracle."""
import numpy as np
import pytest

from paper_2607_07816_b200 import workloads as W
from oracle import dense, fusion


def _gates(c):
    return [(list(g.qubits), np.asarray(g.U, dtype=np.complex128)) for g in c.gates]


def test_oracle_disjoint_gates_give_kronecker_product():
    rng = np.random.default_rng(0)
    A, B, Cm = W.haar_unitary(rng, 2), W.haar_unitary(rng, 2), W.haar_unitary(rng, 4)
    (q, U), = fusion.fuse([([5], A), ([9], B)], max_m=4)
    assert q == [5, 9]
    assert np.allclose(U, np.kron(B, A), atol=1e-15)          # local bit 0 = qubit 5 = the LOW factor
    (q, U), = fusion.fuse([([3, 1], Cm), ([7], A)], max_m=3)
    assert q == [3, 1, 7]
    assert np.allclose(U, np.kron(A, Cm), atol=1e-15)


def test_oracle_same_qubits_give_matrix_product_later_gate_on_the_left():
    rng = np.random.default_rng(1)
    A, B = W.haar_unitary(rng, 4), W.haar_unitary(rng, 4)
    (q, U), = fusion.fuse([([2, 6], A), ([2, 6], B)], max_m=2)
    assert q == [2, 6]
    assert np.allclose(U, B @ A, atol=1e-15)
    # the same gate with its qubits listed the other way round: conjugate by the swap of the two local bits
    S = np.eye(4)[[0, 2, 1, 3]]
    (q, U), = fusion.fuse([([2, 6], A), ([6, 2], B)], max_m=2)
    assert np.allclose(U, (S @ B @ S) @ A, atol=1e-15)


def test_oracle_blocks_are_greedy_and_unitary_and_single_gate_blocks_are_the_gate():
    c = W.config2(n=10, num_gates=60, max_terms=1 << 10)
    gates = _gates(c)
    for max_m in (1, 2, 3, 4):
        if max(len(q) for q, _ in gates) > max_m:
            continue
        blocks = fusion.blocks_of(gates, max_m)
        assert [i for b in blocks for i in b] == list(range(len(gates)))       # in order, nothing lost
        for b in blocks:
            assert len({x for i in b for x in gates[i][0]}) <= max_m
        for b, nxt in zip(blocks, blocks[1:]):                                    # greedy: the next gate did not fit
            assert len({x for i in b for x in gates[i][0]} | set(gates[nxt[0]][0])) > max_m
        for (q, U), b in zip(fusion.fuse(gates, max_m), blocks):
            assert np.allclose(U.conj().T @ U, np.eye(U.shape[0]), atol=1e-13)
            if len(b) == 1:
                assert q == gates[b[0]][0] and np.array_equal(U, gates[b[0]][1])


@pytest.mark.parametrize("max_m", [2, 3, 4])
def test_oracle_fused_circuit_equals_gate_by_gate_on_the_dense_simulator(max_m):
    c = W.config1(n=10, layers=4, seed=5)
    gates = [g for g in _gates(c) if len(g[0]) <= max_m]
    psi = dense.ground(10)
    for q, U in gates:
        psi = dense.apply_gate(psi, 10, q, U)
    phi = dense.ground(10)
    blocks = fusion.fuse(gates, max_m)
    assert len(blocks) < len(gates)
    for q, U in blocks:
        phi = dense.apply_gate(phi, 10, q, U)
    assert np.max(np.abs(psi - phi)) <= 1e-13


def test_library_fusion_equals_oracle():
    from paper_2607_07816_b200 import engine
    rng = np.random.default_rng(3)
    for trial, max_m in enumerate((1, 2, 3, 4, 4, 4)):
        gates = []
        for _ in range(40):
            m = int(rng.integers(1, min(max_m, 3) + 1))
            q = [int(x) for x in rng.choice(14 if trial < 5 else 5, size=m, replace=False)]
            gates.append((q, W.haar_unitary(rng, 1 << m)))
        got = engine.fuse_gates(gates, max_m)
        want = fusion.fuse(gates, max_m)
        assert len(got) == len(want)
        for (qa, Ua), (qb, Ub) in zip(got, want):
            assert qa == qb
            assert np.max(np.abs(Ua - Ub)) <= 1e-14
    assert engine.fuse_gates([], 4) == []
    (q, U), = engine.fuse_gates([([3], W.mat_h())], 4)
    assert q == [3] and np.array_equal(U, W.mat_h())           # a block of one gate is that gate, bit for bit
    with pytest.raises(engine.SvError):
        engine.fuse_gates([([1, 1], np.eye(4))], 4)
    with pytest.raises(engine.SvError):
        engine.fuse_gates([([0, 1, 2], np.eye(8))], 2)


@pytest.mark.gpu
def test_gpu_fused_blocks_equal_the_unfused_circuit():
    """Config 1 (n = 12, no truncation): the engine runs the fused blocks, the oracle runs the gates one by one."""
    from paper_2607_07816_b200 import engine
    from oracle.sparse import SparseOracle
    c = W.config1()
    gates = _gates(c)
    blocks = engine.fuse_gates(gates, 4)
    assert len(blocks) < len(gates)
    sv = engine.SparseSV(c.n, 1 << 13)
    for q, U in blocks:
        sv.apply_gate(q, U)
    o = SparseOracle(c.n)
    for q, U in gates:
        o.apply_gate(q, U)
    gk, ga, _ = sv.export()
    ok_, oa, _ = o.export()
    od = dict(zip(ok_.tolist(), oa))
    gd = dict(zip(gk.tolist(), ga))
    for k in set(od) | set(gd):                                # a key missing on one side counts as 0 there
        assert abs(gd.get(k, 0.0) - od.get(k, 0.0)) <= 1e-11
    assert abs(sv.norm() - 1.0) <= 1e-12


@pytest.mark.gpu
def test_gpu_fused_blocks_with_truncation_once_per_block():
    """one update and one truncation per block.  The engine (fused call) against the oracle applying the
    SAME fused blocks, step-locked, config 5 scaled (n = 40, cap 2^14)."""
    from paper_2607_07816_b200 import engine
    from oracle.sparse import SparseOracle
    from util_parity import assert_truncation_parity, MASS_TOL
    K = 1 << 14
    c = W.config5(n=40, num_gates=160, max_terms=K)
    blocks = engine.fuse_gates(_gates(c), 4)                   # (the circuit has 4-qubit Toffolis)
    assert len(blocks) < len(c.gates)
    sv = engine.SparseSV(c.n, 16 * K)
    sv.set_option(engine.OPT_SAMPLE_MIN_TERMS, 512)
    for q, U in blocks:
        k0, a0, _ = sv.export()
        o = SparseOracle(c.n)
        o.load(k0, a0)
        kg = sv.apply_gate_truncate(q, U, K, c.min_mass)
        o.apply_gate(q, U)
        ko = o.truncate(K, c.min_mass)
        assert abs(kg - ko) <= MASS_TOL
        assert_truncation_parity(sv.export()[:2], o.export()[:2])
    assert sv.check_invariants()
