"""GPU parity of sv_apply_circuit (include/sparse_sv.h): a list of gates, each followed by the same
truncation, as one call -- through the single-block small-state path (sv_small.cu) while the state fits it, through the
streaming passes otherwise -- against the CPU oracle step by step, against the gate-by-gate calls, and across the
hand-over between the two paths."""
import numpy as np
import pytest

from paper_2607_07816_b200 import workloads as W

pytestmark = pytest.mark.gpu

from util_parity import assert_same_state, assert_truncation_parity, MASS_TOL  # noqa: E402


@pytest.fixture(scope="module")
def eng():
    from paper_2607_07816_b200 import engine
    return engine


def _oracle(n):
    from oracle.sparse import SparseOracle
    return SparseOracle(n)


def _ring_blocks(eng, n=44, layers=4, seed=5):
    c = W.ring_peaked(n=n, layers=layers, seed=seed)
    gates = [(list(g.qubits), g.U) for g in c.gates]
    order = eng.reorder_gates(gates, [W.is_diagonal(U) for _, U in gates])
    return c, eng.fuse_gates([gates[i] for i in order], 4)


@pytest.mark.parametrize("K", [16, 64, 700])
def test_ring_blocks_step_locked_vs_oracle(eng, K):
    """The paper's experiment shape (u3 + cz ring, reordered, fused into <= 4-qubit blocks, top-k after every block,
    PAPER.md:146-190) through the small-state path, one block per call: every block is compared with the oracle from the
    same pre-block state (kept fraction to 1e-10, kept sets identical except within 1e-9 of the cut)."""
    c, blocks = _ring_blocks(eng, n=30, layers=3)
    sv = eng.SparseSV(c.n, 1 << 16)
    for q, U in blocks:
        k0, a0, _ = sv.export()
        o = _oracle(c.n)
        o.load(k0, a0)
        kg = sv.apply_circuit([(q, U)], K, 1.0)[0]
        o.apply_gate(q, U)
        ko = o.truncate(K, 1.0)
        assert abs(kg - ko) <= MASS_TOL
        assert sv.num_terms() == o.num_terms() <= K
        assert_truncation_parity(sv.export()[:2], o.export()[:2])
        assert sv.check_invariants()
    sg = sv.stats()["small_gates"]
    assert sg == len(blocks) if K * 16 <= 4096 else 0 < sg < len(blocks)     # (K = 700: a 16x expansion does not fit one block)
    assert abs(sv.norm() - 1.0) <= 1e-12


def test_ring44_one_call_finds_the_secret_and_equals_block_by_block(eng):
    """n = 44, 594 instructions, K = 64: ONE call for the whole circuit (batches of 64 single-block launches) gives the
    bits of the block-by-block calls, and the most probable bit string is the secret."""
    c, blocks = _ring_blocks(eng)
    a, b = eng.SparseSV(c.n, 1 << 12), eng.SparseSV(c.n, 1 << 12)
    ka = a.apply_circuit(blocks, 64, 1.0)
    kb = np.array([b.apply_circuit([blk], 64, 1.0)[0] for blk in blocks])
    assert np.array_equal(ka, kb)
    ea, eb = a.export(), b.export()
    assert np.array_equal(ea[0], eb[0]) and np.array_equal(ea[1], eb[1])
    assert a.stats()["small_gates"] == len(blocks)
    k, _, p = a.top(1)
    assert int(k[0]) == c.secret and p[0] > 0.05


def test_config1_through_the_circuit_call(eng):
    """BASELINE.json configs[0] (n = 12, dense 4096-term state, no truncation) as one call: complete tuples take the
    in-place branch of the small-state kernel; free-running against the oracle (max |da| <= 1e-11, identical keys)."""
    c = W.config1()
    sv = eng.SparseSV(c.n, 1 << 13)
    o = _oracle(c.n)
    kept = sv.apply_circuit([(g.qubits, g.U) for g in c.gates], 0, 1.0)
    for g in c.gates:
        o.apply_gate(g.qubits, g.U)
    assert np.all(kept == 1.0)
    assert sv.stats()["small_gates"] == len(c.gates)
    assert_same_state(sv.export()[:2], o.export()[:2])
    assert abs(sv.norm() - 1.0) <= 1e-12
    assert sv.check_invariants()


@pytest.mark.parametrize("n,count,seed", [(20, 900, 0), (64, 1500, 1), (40, 4096, 2), (12, 300, 3)])
def test_random_gates_small_path_vs_oracle(eng, n, count, seed):
    """Every gate class, m = 1..4, random qubits (bit 63 included), lazy X masks and renamed qubits in the layout,
    mass + cap cuts: the small-state path step-locked against the oracle."""
    rng = np.random.default_rng(seed)
    keys, amps = W.random_state(rng, n, count, spread=1.0)
    if n == 64:
        keys[0] = np.uint64(0xFFFFFFFFFFFFFFFF); keys = np.unique(keys); amps = amps[:keys.size]
        amps /= np.sqrt(np.sum(np.abs(amps) ** 2))
    sv = eng.SparseSV(n, 1 << 16)
    sv.load(keys, amps)
    sv.apply_gate([0], W.mat_x()); sv.apply_gate([n - 1, 1], np.eye(4)[[0, 2, 1, 3]].astype(np.complex128))   # lazy mask + renamed qubits
    mats = {1: [W.mat_h(), W.mat_rz(0.3), W.mat_x(), W.haar_unitary(rng, 2)], 2: [W.mat_mcx(2), W.haar_unitary(rng, 4), W.mat_diag_minus_last(2)],
            3: [W.mat_mcx(3), W.haar_unitary(rng, 8)], 4: [W.mat_mcx(4), W.haar_unitary(rng, 16)]}
    small = 0
    for step in range(24):
        m = int(rng.integers(1, 5))
        qs = [int(x) for x in rng.choice(n, size=m, replace=False)]
        if n == 64 and step % 5 == 0:
            qs[0] = 63 if 63 not in qs else qs[0]
        U = mats[m][int(rng.integers(len(mats[m])))]
        K, f = (600, 1.0) if step % 3 == 0 else ((0, 0.999) if step % 3 == 1 else (1500, 0.9999))
        k0, a0, _ = sv.export()
        o = _oracle(n)
        o.load(k0, a0)
        before = sv.stats()["small_gates"]
        kg = sv.apply_circuit([(qs, U)], K, f)[0]
        small += sv.stats()["small_gates"] - before
        o.apply_gate(qs, U)
        ko = o.truncate(K, f)
        assert abs(kg - ko) <= MASS_TOL, (step, qs)
        assert sv.num_terms() == o.num_terms(), (step, qs)
        assert_truncation_parity(sv.export()[:2], o.export()[:2])
        assert sv.check_invariants()
    assert small >= 4          # (expansions beyond 4096 entries take the streaming passes)


def test_hand_over_between_the_paths(eng):
    """Scaled configs[4] (K = 2^13): the state grows through the small-state limit, is cut back, grows again.  One call for
    the whole list must give THE BITS of the gate-by-gate streaming calls (small path off): the single-block kernel takes
    its mass sums in double-double, which round to the doubles of the streaming path's exact sums (D3), so
    threshold, cut, scale and every later exact cancellation are the same -- 160 gates free-running."""
    c = W.config5(num_gates=160, max_terms=1 << 13)
    gl = [(g.qubits, g.U) for g in c.gates]
    a, b = eng.SparseSV(c.n, 1 << 17), eng.SparseSV(c.n, 1 << 17)
    b.set_option(eng.OPT_SMALL_STATE_PATH, 0)
    ka = a.apply_circuit(gl, c.max_terms, c.min_mass)
    kb = b.apply_circuit(gl, c.max_terms, c.min_mass)
    assert 0 < a.stats()["small_gates"] < len(gl) and b.stats()["small_gates"] == 0
    assert np.array_equal(ka, kb)
    ea, eb = a.export(), b.export()
    assert np.array_equal(ea[0], eb[0]) and np.array_equal(ea[1], eb[1])
    assert a.check_invariants()


def test_circuit_call_errors(eng):
    sv = eng.SparseSV(10, 256)
    with pytest.raises(eng.SvError):
        sv.apply_circuit([([0], W.mat_h()), ([10], W.mat_h())], 0, 1.0)          # validated up front
    assert sv.num_terms() == 1
    with pytest.raises(eng.SvError):
        sv.apply_circuit([([0, 0], W.mat_mcx(2))], 0, 1.0)
    assert sv.apply_circuit([], 0, 1.0).size == 0
    # capacity: the streaming path reports it, the gates before it stay applied
    with pytest.raises(eng.SvError) as ei:
        sv.apply_circuit([([q], W.mat_h()) for q in range(10)], 0, 1.0)
    assert ei.value.code in (eng.SV_ERR_CAPACITY,)


def test_qasm_text_through_the_circuit_call(eng):
    """OpenQASM 2.0 text in the shape of the paper's excerpt (u3 + cz on a ring; own seeded angles) ->
    qasm.loads -> reorder + fuse -> ONE sv_apply_circuit call with top-k after every block, against the oracle running
    the same blocks, and the peak is found."""
    from paper_2607_07816_b200 import qasm
    import math
    rng = np.random.default_rng(21)
    n, layers = 16, 3
    ring, ops = [], []
    for layer in range(layers):
        for a in range(layer % 2, n - 1 + layer % 2, 2):
            b = (a + 1) % n
            ring += [("u3", a, float(rng.uniform(0, math.pi)), 0.0, -0.5 * math.pi), ("u3", b, float(rng.uniform(0, math.pi)), 0.0, 0.5 * math.pi), ("cz", a, b)]
    ops += ring
    ops += [("u3", q, float(rng.normal(0.0, 0.3)), 0.0, 0.0) for q in range(n)]
    for o in reversed(ring):          # R^dagger: cz is its own inverse, u3(t, p, l)^-1 = u3(-t, -l, -p)
        ops.append(o if o[0] == "cz" else ("u3", o[1], -o[2], -o[4], -o[3]))
    secret = int(rng.integers(0, 1 << n))
    ops += [("u3", q, math.pi, 0.0, math.pi) for q in range(n) if (secret >> q) & 1]
    c = qasm.loads(qasm.dumps_u3_cz(n, ops))
    assert c.n == n and len(c.gates) == len(ops)
    gates = [(list(g.qubits), g.U) for g in c.gates]
    order = eng.reorder_gates(gates, [W.is_diagonal(U) for _, U in gates])
    blocks = eng.fuse_gates([gates[i] for i in order], 4)
    K = 128
    sv = eng.SparseSV(n, 1 << 14)
    kf = sv.apply_circuit(blocks, K, 1.0)
    o = _oracle(n)
    ko = []
    for q, U in blocks:
        o.apply_gate(q, U)
        ko.append(o.truncate(K, 1.0))
    assert np.allclose(kf, ko, atol=1e-9, rtol=0)
    k, _, p = sv.top(1)
    k2, _, p2 = o.top(1)
    assert int(k[0]) == int(k2[0]) == secret
    assert abs(p[0] - p2[0]) <= 1e-9
