"""GPU parity of the TWO-BIT final pass (sv_dense.cu TWO, sv_gate.cu find_splits2): a dense multi-qubit gate whose last
two missing qubits are brought to the low bit positions by the final pass itself (SURVEY.md rows
a-4 .. a-7).  Checked against the CPU oracle (north_star tolerance) and, bit for bit, against the same engine with
one pass per missing qubit (SV_OPT_TWO_BIT_PASS = 0)."""
import numpy as np
import pytest

from paper_2607_07816_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def eng():
    from paper_2607_07816_b200 import engine
    return engine


def _oracle(n):
    from oracle.sparse import SparseOracle
    return SparseOracle(n)


from util_parity import assert_same_state, assert_truncation_parity, MASS_TOL  # noqa: E402


def _subspace_state(rng, n, free_bits, count=None):
    """All (or `count` random) patterns on `free_bits`, the other bits a fixed random constant: tuples with every
    number of members, blocks of every length."""
    const = int(rng.integers(0, 1 << min(n, 62), dtype=np.uint64))
    fb = list(free_bits)
    for b in fb:
        const &= ~(1 << b)
    tot = 1 << len(fb)
    idx = np.arange(tot, dtype=np.uint64) if count is None or count >= tot else np.sort(rng.choice(tot, size=count, replace=False)).astype(np.uint64)
    keys = np.full(idx.size, const, dtype=np.uint64)
    for j, b in enumerate(fb):
        keys |= ((idx >> np.uint64(j)) & np.uint64(1)) << np.uint64(b)
    mag = np.exp(1.5 * rng.standard_normal(keys.size))
    amps = (mag * np.exp(1j * rng.uniform(0, 2 * np.pi, keys.size))).astype(np.complex128)
    amps /= np.sqrt(np.sum(np.abs(amps) ** 2))
    return np.ascontiguousarray(keys), np.ascontiguousarray(amps)


def _three_way(eng, n, keys, amps, gates, cap):
    """The same gates on: the engine (two-bit pass on), the engine (off), the oracle."""
    a = eng.SparseSV(n, cap)
    a.set_option(eng.OPT_TWO_BIT_PASS, 1)
    b = eng.SparseSV(n, cap)
    b.set_option(eng.OPT_TWO_BIT_PASS, 0)
    o = _oracle(n)
    for s in (a, b, o):
        s.load(keys, amps)
    saved = 0
    for qs, U in gates:
        a.apply_gate(qs, U)
        pa = a.stats()["passes"]
        b.apply_gate(qs, U)
        pb = b.stats()["passes"]
        o.apply_gate(qs, U)
        assert pa <= pb
        saved += pb - pa
        ka, aa, _ = a.export()
        kb, ab, _ = b.export()
        assert np.array_equal(ka, kb) and np.array_equal(aa.view(np.uint64), ab.view(np.uint64)), "two-bit pass differs from two single-bit passes"
        assert_same_state((ka, aa), o.export()[:2])
        assert a.check_invariants()
    return saved


# (n, free bits of the state, qubits of the gate): adjacent and distant bits, the top bit, bits inside and outside the
# populated subspace, small and long blocks
CASES = [
    (20, list(range(0, 14)), [9, 4]),
    (20, list(range(0, 14)), [13, 12]),
    (20, list(range(3, 17)), [1, 0]),            # both bits constant over the state
    (20, list(range(3, 17)), [16, 2]),
    (24, [0, 2, 3, 5, 8, 9, 11, 12, 14, 17, 18, 20, 21, 23], [23, 0]),
    (24, [0, 2, 3, 5, 8, 9, 11, 12, 14, 17, 18, 20, 21, 23], [12, 11]),
    (64, [1, 7, 13, 20, 26, 33, 40, 41, 47, 52, 58, 60, 62, 63], [63, 62]),
    (64, [1, 7, 13, 20, 26, 33, 40, 41, 47, 52, 58, 60, 62, 63], [63, 1]),
    (64, [1, 7, 13, 20, 26, 33, 40, 41, 47, 52, 58, 60, 62, 63], [30, 50]),
    (56, list(range(20, 35)), [34, 20, 27]),
    (56, list(range(20, 35)), [55, 33, 3]),
    (40, list(range(5, 19)), [18, 5, 11, 30]),
    (40, list(range(5, 19)), [6, 7, 8, 9]),
]


@pytest.mark.parametrize("case", range(len(CASES)))
@pytest.mark.parametrize("fill", ["full", "ragged"])
def test_two_bit_pass_subspace_states(eng, case, fill):
    n, fb, qs = CASES[case]
    rng = np.random.default_rng(4000 + case)
    keys, amps = _subspace_state(rng, n, fb, None if fill == "full" else (1 << len(fb)) * 5 // 8 + 3)
    m = len(qs)
    gates = [(qs, W.haar_unitary(rng, 1 << m)), (qs[::-1], W.haar_unitary(rng, 1 << m))]
    # a second gate on fresh qubits of the (now wider) state
    others = [q for q in fb if q not in qs]
    q2 = [int(x) for x in rng.choice(others, size=2, replace=False)]
    gates.append((q2, W.haar_unitary(rng, 4)))
    saved = _three_way(eng, n, keys, amps, gates, cap=(keys.size << (m + 2)) + 64)
    assert saved >= 1      # the pass was taken: at least one pass less than with single-bit moves


@pytest.mark.parametrize("n,count,seed", [(30, 40000, 0), (64, 25013, 1), (18, 100000, 2), (12, 4096, 3), (50, 1, 4), (50, 2, 5), (44, 1017, 6)])
def test_two_bit_pass_random_states(eng, n, count, seed):
    """Sparse uniform states (few partners), several tiles and a ragged tail; m = 2, 3, 4 on random qubits."""
    rng = np.random.default_rng(5000 + seed)
    keys, amps = W.random_state(rng, n, count)
    gates = []
    for m in (2, 3, 4, 2):
        qs = [int(q) for q in rng.choice(n, size=m, replace=False)]
        gates.append((qs, W.haar_unitary(rng, 1 << m)))
    cap = keys.size * (1 << 11) + 64 if keys.size < 3000 else keys.size * 16 + 64
    a = eng.SparseSV(n, cap)
    a.set_option(eng.OPT_TWO_BIT_PASS, 1)
    b = eng.SparseSV(n, cap)
    b.set_option(eng.OPT_TWO_BIT_PASS, 0)
    o = _oracle(n)
    for s in (a, b, o):
        s.load(keys, amps)
    for qs, U in gates:
        if o.num_terms() << len(qs) > cap:
            break
        a.apply_gate(qs, U); b.apply_gate(qs, U); o.apply_gate(qs, U)
        ka, aa, _ = a.export()
        kb, ab, _ = b.export()
        assert np.array_equal(ka, kb) and np.array_equal(aa.view(np.uint64), ab.view(np.uint64))
        assert_same_state((ka, aa), o.export()[:2])
        assert a.check_invariants()
        if o.num_terms() > 50000:
            k, am, _ = o.top(20000)
            for s in (a, b, o):
                s.load(k, am)


def test_two_bit_pass_with_pending_cut_and_fused_call(eng):
    """A truncation is pending when the gate runs (dropped terms are squeezed out in the partition); every third gate goes
    through the fused call, which never uses the two-bit pass (sv_api.cu) and must leave the layout in a state the next
    two-bit pass can start from: all against the oracle, step-locked."""
    rng = np.random.default_rng(6001)
    n = 40
    fb = [2, 5, 6, 9, 13, 17, 18, 22, 25, 29, 31, 33, 36, 38, 39]
    keys, amps = _subspace_state(rng, n, fb)
    K = 6000
    sv = eng.SparseSV(n, 1 << 20)
    sv.set_option(eng.OPT_SAMPLE_MIN_TERMS, 512)
    sv.set_option(eng.OPT_TWO_BIT_PASS, 1)
    sv.load(keys, amps)
    used_two = 0
    for step in range(10):
        m = 2 + step % 3
        qs = [int(q) for q in rng.choice(fb if step % 2 else n, size=m, replace=False)]
        U = W.haar_unitary(rng, 1 << m)
        k0, a0, _ = sv.export()
        o = _oracle(n)
        o.load(k0, a0)
        if step % 3 == 2:
            kg = sv.apply_gate_truncate(qs, U, K, 1.0 - 1e-4)
            st = sv.stats()
        else:
            sv.apply_gate(qs, U)
            st = sv.stats()
            o_mid = _oracle(n); o_mid.load(k0, a0); o_mid.apply_gate(qs, U)
            assert_same_state(sv.export()[:2], o_mid.export()[:2])
            kg = sv.truncate(K, 1.0 - 1e-4)
        used_two += 1 if st["passes"] < m else 0
        o.apply_gate(qs, U)
        ko = o.truncate(K, 1.0 - 1e-4)
        assert abs(kg - ko) <= MASS_TOL
        assert_truncation_parity(sv.export()[:2], o.export()[:2])
        assert sv.check_invariants()
    assert used_two >= 3


def test_two_bit_option_values_and_pass_counts(eng):
    """SV_OPT_TWO_BIT_PASS: 0 = one pass per missing qubit, 1 = two-bit final pass for every dense gate, 2 (the default) =
    for dense gates on three or four mixing qubits only.  Same bits in every mode."""
    rng = np.random.default_rng(7001)
    n = 30
    keys, amps = W.random_state(rng, n, 20000)
    gates = [([25, 11], W.haar_unitary(rng, 4)), ([29, 3, 17], W.haar_unitary(rng, 8)), ([8, 21, 14, 27], W.haar_unitary(rng, 16))]
    want = {0: [2, 3, 4], 1: [1, 2, 3], 2: [2, 2, 3], None: [2, 2, 3]}
    ref = None
    for mode, passes in want.items():
        sv = eng.SparseSV(n, 1 << 22)
        if mode is not None:
            sv.set_option(eng.OPT_TWO_BIT_PASS, mode)
        out = []
        for (qs, U), p in zip(gates, passes):
            sv.load(keys, amps)
            sv.apply_gate(qs, U)
            assert sv.stats()["passes"] == p, (mode, qs, sv.stats()["passes"])
            k, a, _ = sv.export()
            out.append((k, a))
        if ref is None:
            ref = out
        for (k, a), (k0, a0) in zip(out, ref):
            assert np.array_equal(k, k0) and np.array_equal(a.view(np.uint64), a0.view(np.uint64))


def test_definite_qubits_hook(eng):
    """sv_test_definite_qubits (include/sparse_sv_test.h): the qubits with one value over the whole state, through the lazy
    layout (an X only flips the mask), a gate that spreads one of them, and a pending truncation that removes the spread."""
    rng = np.random.default_rng(7002)
    n = 20
    free = [0, 2, 5, 7, 8, 11, 13, 16]
    const = (1 << 3) | (1 << 19)                       # qubits 3 and 19 are 1, the other non-free ones 0
    idx = np.arange(1 << len(free), dtype=np.uint64)
    keys = np.full(idx.size, const, dtype=np.uint64)
    for j, b in enumerate(free):
        keys |= ((idx >> np.uint64(j)) & np.uint64(1)) << np.uint64(b)
    amps = (rng.standard_normal(keys.size) + 1j * rng.standard_normal(keys.size)).astype(np.complex128)
    amps /= np.sqrt(np.sum(np.abs(amps) ** 2))
    sv = eng.SparseSV(n, 1 << 12)
    sv.load(keys, amps)
    definite = sum(1 << q for q in range(n) if q not in free)
    assert sv.test_definite_qubits() == definite
    sv.apply_gate([19], W.mat_x())                     # lazy: still definite (now 0)
    sv.apply_gate([3, 0], W.mat_mcx(2))                # CNOT 3 -> 0: qubit 0 stays spread, qubit 3 stays definite
    assert sv.test_definite_qubits() == definite
    sv.apply_gate([4], W.mat_rx(0.02))                 # qubit 4 is spread, weakly: |1> carries sin^2(0.01) of the mass
    assert sv.test_definite_qubits() == definite & ~(1 << 4)
    sv.truncate(0, 0.999)                              # the cut (pending) drops the weak branch again
    assert sv.test_definite_qubits() == definite
