"""GPU parity: sv_apply_gate / sv_norm / sv_top / sv_load through the C ABI vs the CPU oracle."""
import math
import os

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


from util_parity import assert_same_state, AMP_TOL  # noqa: E402
from test_oracle_gate import _parse_golden, NAMED  # noqa: E402


@pytest.mark.parametrize("case", _parse_golden())
def test_closed_forms_gpu(eng, case):
    n, gl, exp = case
    sv = eng.SparseSV(n, 64)
    for name, qs in gl:
        sv.apply_gate(qs, NAMED[name][1]())
    k, a, p = sv.export()
    got = {int(x): complex(y) for x, y in zip(k, a)}
    assert set(got) == set(exp)
    for key in exp:
        assert abs(got[key] - exp[key]) <= 4e-16
    assert sv.check_invariants()


def test_config1_free_running(eng):
    """BASELINE.json configs[0]; truncation off: identical key sets, max |da| <= 1e-11, every gate."""
    c = W.config1()
    sv = eng.SparseSV(c.n, 1 << 13)
    o = _oracle(c.n)
    for g in c.gates:
        sv.apply_gate(g.qubits, g.U)
        o.apply_gate(g.qubits, g.U)
        gk, ga, _ = sv.export()
        ok, oa, _ = o.export()
        assert_same_state((gk, ga), (ok, oa))
        assert sv.check_invariants()
    assert sv.num_terms() <= 4096
    assert abs(sv.norm() - 1.0) <= 1e-13 * len(c.gates)


@pytest.mark.parametrize("n,count,seed", [(20, 5000, 0), (40, 30011, 1), (64, 7777, 2), (12, 4096, 3), (30, 1, 4), (56, 100003, 5)])
def test_random_gates_on_random_states(eng, n, count, seed):
    """Every gate class, m = 1..4, random (unordered, non-adjacent) qubits, states spanning
    several tiles with a ragged tail.  Free running, truncation off."""
    rng = np.random.default_rng(1000 + seed)
    keys, amps = W.random_state(rng, n, count)
    cap = 16 * keys.size + 64
    sv = eng.SparseSV(n, cap)
    o = _oracle(n)
    sv.load(keys, amps)
    o.load(keys, amps)
    assert_same_state(sv.export()[:2], o.export()[:2], tol=0.0)
    for step in range(14):
        m = 1 + (step % 4)
        if m > n:
            m = n
        qs = [int(q) for q in rng.choice(n, size=m, replace=False)]
        kind = step % 5
        if kind == 0:
            U = W.haar_unitary(rng, 1 << m)
        elif kind == 1:
            U = np.diag(np.exp(1j * rng.uniform(0, 2 * np.pi, 1 << m)))
        elif kind == 2:
            U = W.mat_mcx(m) if m > 1 else W.mat_x()
        elif kind == 3:   # controlled-U: block diagonal in the first qubit
            U = np.eye(1 << m, dtype=np.complex128)
            if m > 1:
                sub = W.haar_unitary(rng, 1 << (m - 1))
                idx = [c for c in range(1 << m) if c & 1]
                U[np.ix_(idx, idx)] = sub
            else:
                U = W.mat_h()
        else:
            U = W.mat_h() if m == 1 else W.haar_unitary(rng, 1 << m)
        if o.num_terms() * (1 << m) > cap:
            U = np.diag(np.exp(1j * rng.uniform(0, 2 * np.pi, 1 << m)))
        sv.apply_gate(qs, U)
        o.apply_gate(qs, U)
        assert sv.num_terms() == o.num_terms()
        assert_same_state(sv.export()[:2], o.export()[:2])
        assert sv.check_invariants()
        assert abs(sv.norm() - o.norm()) <= 1e-12
        if o.num_terms() > 60000:   # keep the oracle fast: cut back to a manageable size on both sides
            k, a, _ = o.top(20000)
            sv.load(k, a)
            o.load(k, a)


def test_repeated_gates_same_qubits(eng):
    """Active bits already at the LSBs: the no-move path, including permuted qubit order."""
    rng = np.random.default_rng(77)
    n = 24
    keys, amps = W.random_state(rng, n, 9000)
    sv = eng.SparseSV(n, 1 << 18)
    o = _oracle(n)
    sv.load(keys, amps)
    o.load(keys, amps)
    for qs in ([5, 9], [9, 5], [5], [9, 5, 17], [17, 9], [5, 17, 9, 2], [2, 5]):
        U = W.haar_unitary(rng, 1 << len(qs))
        sv.apply_gate(qs, U)
        o.apply_gate(qs, U)
        assert_same_state(sv.export()[:2], o.export()[:2])
        assert sv.check_invariants()


def test_h_growth_and_cancellation(eng):
    """PAPER.md:53 growth, then H again: exact cancellation drops the zeros."""
    n = 40
    sv = eng.SparseSV(n, 1 << 12)
    qs = [3, 17, 39, 0, 8, 21, 11, 5]
    amp = 1.0
    for j, q in enumerate(qs, 1):
        sv.apply_gate([q], W.mat_h())
        amp = (1.0 / math.sqrt(2.0)) * amp
        k, a, _ = sv.export()
        assert k.size == 1 << j
        assert np.all(a.real == amp) and np.all(a.imag == 0.0)
    o = _oracle(n)
    k, a, _ = sv.export()
    o.load(k, a)
    for q in qs:
        sv.apply_gate([q], W.mat_h())
        o.apply_gate([q], W.mat_h())
        assert sv.num_terms() == o.num_terms()
    assert sv.num_terms() == 1


def test_ghz_64(eng):
    n = 64
    sv = eng.SparseSV(n, 16)
    sv.apply_gate([0], W.mat_h())
    for q in range(1, n):
        sv.apply_gate([q - 1, q], W.mat_mcx(2))
    k, a, p = sv.export()
    r = 1.0 / math.sqrt(2.0)
    assert [int(x) for x in k] == [0, (1 << 64) - 1]
    assert np.all(a == complex(r, 0))


def test_xor_class_is_lazy(eng):
    rng = np.random.default_rng(3)
    n = 30
    keys, amps = W.random_state(rng, n, 5000)
    sv = eng.SparseSV(n, 1 << 15)
    o = _oracle(n)
    sv.load(keys, amps)
    o.load(keys, amps)
    Y = np.array([[0, -1j], [1j, 0]])
    for q, U, lazy in [(4, W.mat_x(), True), (29, W.mat_x(), True), (4, Y, False), (11, W.mat_h(), False),
                       (4, W.mat_rz(0.7), False), (4, W.mat_h(), False), (29, W.mat_x(), True)]:
        sv.apply_gate([q], U)
        o.apply_gate([q], U)
        if lazy:
            assert sv.stats()["class"] == "xor" and sv.stats()["passes"] == 0
        assert_same_state(sv.export()[:2], o.export()[:2])
    XX = np.kron(W.mat_x(), W.mat_x())
    sv.apply_gate([7, 19], XX)
    o.apply_gate([7, 19], XX)
    assert sv.stats()["class"] == "xor" and sv.stats()["passes"] == 0
    sv.apply_gate([19, 3, 7], W.mat_mcx(3))
    o.apply_gate([19, 3, 7], W.mat_mcx(3))
    assert_same_state(sv.export()[:2], o.export()[:2])


def test_capacity_error_leaves_state(eng):
    n = 20
    sv = eng.SparseSV(n, 40)
    for q in range(5):
        sv.apply_gate([q], W.mat_h())
    before = sv.export()
    with pytest.raises(eng.SvError) as ei:
        sv.apply_gate([7], W.mat_h())
    assert ei.value.code == eng.SV_ERR_CAPACITY
    after = sv.export()
    assert np.array_equal(before[0], after[0]) and np.array_equal(before[1], after[1])
    sv.apply_gate([7], W.mat_x())   # still usable


def test_invalid_arguments(eng):
    sv = eng.SparseSV(8, 64)
    for qs, U in (([0, 0], W.mat_mcx(2)), ([8], W.mat_h()), ([-1], W.mat_h())):
        with pytest.raises(eng.SvError) as ei:
            sv.apply_gate(qs, U)
        assert ei.value.code == eng.SV_ERR_INVALID_ARG
    with pytest.raises(eng.SvError):
        sv.load(np.array([1, 1], dtype=np.uint64), np.array([0.6, 0.8], dtype=np.complex128))
    with pytest.raises(eng.SvError):
        sv.load(np.array([256], dtype=np.uint64), np.array([1.0], dtype=np.complex128))
    with pytest.raises(eng.SvError):
        sv.truncate(0, 0.0)
    assert sv.num_terms() == 1   # unchanged


def test_own_allocation_path(eng):
    sv = eng.SparseSV(10, 2048, torch_arena=False)
    o = _oracle(10)
    c = W.config1(n=10, layers=2, seed=5)
    for g in c.gates:
        sv.apply_gate(g.qubits, g.U)
        o.apply_gate(g.qubits, g.U)
    assert_same_state(sv.export()[:2], o.export()[:2])
    sv.close()


def test_top_order(eng):
    rng = np.random.default_rng(21)
    n = 50
    keys, amps = W.random_state(rng, n, 40000)
    amps[100:200] = amps[100]   # exact ties, ordered by key
    sv = eng.SparseSV(n, 1 << 16)
    o = _oracle(n)
    sv.load(keys, amps)
    o.load(keys, amps)
    for k in (1, 7, 150, 5000, 40000, 10 ** 6):
        gk, ga, gp = sv.top(k)
        ok, oa, op = o.top(k)
        assert np.array_equal(gk, ok)
        assert np.array_equal(ga, oa)
        assert np.array_equal(gp, op)


@pytest.mark.parametrize("fused", [False, True])
def test_singular_diagonal_gates_drop_terms(eng, fused):
    """U need not be unitary (reading R10): a diagonal U with exact zeros on its diagonal -- a projector -- annihilates
    terms, and an annihilated term is no longer stored ("only nonzero amplitudes").  diag(1,0),
    diag(1,0,1,0), a three-qubit projector and the all-zero matrix, on a state whose storage order has been permuted
    and with a truncation still pending on it, against the oracle."""
    rng = np.random.default_rng(31)
    n = 40
    keys, amps = W.random_state(rng, n, 30000, spread=1.0)
    sv = eng.SparseSV(n, 1 << 17)
    sv.set_option(eng.OPT_SAMPLE_MIN_TERMS, 512)
    o = _oracle(n)
    sv.load(keys, amps); o.load(keys, amps)
    for q in (7, 33):
        sv.apply_gate([q], W.mat_h()); o.apply_gate([q], W.mat_h())
    gates = [([7], np.diag([1.0, 0.0]).astype(np.complex128)),
             ([33, 2], np.diag([1.0, 0.0, 1.0j, 0.0]).astype(np.complex128)),
             ([5, 39, 11], np.diag([0, 1, 1, 0, 0.5, 0, 0, -1]).astype(np.complex128)),
             ([20], np.diag([0.0, 2.0]).astype(np.complex128))]
    for qs, U in gates:
        sv.truncate(0, 0.999); o.truncate(0, 0.999)          # leaves a cut pending on the engine's side
        if fused:
            sv.apply_gate_truncate(qs, U, 0, 1.0)
        else:
            sv.apply_gate(qs, U)
        o.apply_gate(qs, U)
        assert sv.stats()["class"] == "diagonal"
        assert sv.num_terms() == o.num_terms()
        assert_same_state(sv.export()[:2], o.export()[:2])
        assert sv.check_invariants()
    assert sv.num_terms() < 30000
    sv.apply_gate([3, 4], np.zeros((4, 4), dtype=np.complex128)); o.apply_gate([3, 4], np.zeros((4, 4), dtype=np.complex128))
    assert sv.num_terms() == o.num_terms() == 0
    sv.apply_gate([3], W.mat_h())                                  # an empty state stays empty
    assert sv.num_terms() == 0


def test_gates_while_another_stream_keeps_the_sms_busy(eng):
    """The persistent passes wait on one another in their look-back; they are launched cooperatively, so that work
    from another stream cannot leave part of their grid unscheduled while the rest spins (include/sparse_sv.h, "Streams").
    A side stream runs long matmuls while the engine (own stream, own allocation) applies gates of every class and
    truncates; the result must match the oracle and nothing may hang."""
    import torch
    rng = np.random.default_rng(5)
    n = 44
    keys, amps = W.random_state(rng, n, 300000, spread=1.0)
    sv = eng.SparseSV(n, 1 << 22, torch_arena=False)             # its own non-blocking stream
    sv.set_option(eng.OPT_SAMPLE_MIN_TERMS, 512)
    o = _oracle(n)
    sv.load(keys, amps); o.load(keys, amps)
    side = torch.cuda.Stream()
    a = torch.randn(8192, 8192, device="cuda", dtype=torch.float32)
    gates = [([9], W.mat_h()), ([9, 30], W.mat_mcx(2)), ([30, 2], W.haar_unitary(rng, 4)), ([17], W.mat_rz(0.3)),
             ([40, 3, 22], W.haar_unitary(rng, 8)), ([1, 40, 9], W.mat_mcx(3)), ([22], W.haar_unitary(rng, 2))]
    with torch.cuda.stream(side):
        for _ in range(60):
            a = torch.tanh(a @ a) * 0.01
    for qs, U in gates:
        with torch.cuda.stream(side):
            for _ in range(10):
                a = torch.tanh(a @ a) * 0.01
        kg = sv.apply_gate_truncate(qs, U, 400000, 0.9999)
        o.apply_gate(qs, U)
        ko = o.truncate(400000, 0.9999)
        assert abs(kg - ko) <= 1e-10
        assert sv.num_terms() == o.num_terms()
    torch.cuda.synchronize()
    from util_parity import assert_truncation_parity
    assert_truncation_parity(sv.export()[:2], o.export()[:2])
    assert sv.check_invariants()
    sv.close()


def _perm_matrix(sigma, phases=None):
    d = len(sigma)
    U = np.zeros((d, d), dtype=np.complex128)
    for c, r in enumerate(sigma):
        U[r, c] = 1.0 if phases is None else phases[c]
    return U


def test_qubit_relabelling_gates_touch_no_data(eng):
    """SWAP, X (x) SWAP, a cyclic shift of three qubits, iSWAP: monomial gates whose permutation of basis states is a
    permutation of the gate's QUBITS (plus bit flips) only rename qubits: zero passes
    when the entries are 1, one diagonal pass for phases.  Checked against the oracle, with gates of every other class
    and truncations by logical key in between (the lazy layout must stay consistent)."""
    rng = np.random.default_rng(17)
    n = 48
    keys, amps = W.random_state(rng, n, 20000, spread=1.0)
    sv = eng.SparseSV(n, 1 << 17)
    sv.set_option(eng.OPT_SAMPLE_MIN_TERMS, 512)
    o = _oracle(n)
    sv.load(keys, amps); o.load(keys, amps)
    swap = _perm_matrix([0, 2, 1, 3])
    xswap = _perm_matrix([1, 3, 0, 2])                       # r = swap(c) ^ 01
    cyc3 = _perm_matrix([((c << 1) | (c >> 2)) & 7 for c in range(8)])
    iswap = _perm_matrix([0, 2, 1, 3], [1, 1j, 1j, 1])
    x3 = _perm_matrix([c ^ 5 for c in range(8)], np.exp(1j * rng.uniform(0, 6, 8)))
    seq = [("relabel", [3, 40], swap), ("other", [40], W.mat_h()), ("relabel", [40, 3], xswap), ("other", [3, 17], W.mat_mcx(2)),
           ("relabel", [47, 0, 21], cyc3), ("other", [0, 47], W.haar_unitary(rng, 4)), ("phase", [21, 9], iswap),
           ("other", [9], W.mat_rz(0.4)), ("phase", [9, 21, 47], x3), ("relabel", [9, 47], swap), ("other", [47, 3, 9], W.mat_mcx(3))]
    for kind, qs, U in seq:
        sv.truncate(0, 0.9995); o.truncate(0, 0.9995)        # a cut stays pending on the engine's side
        l0 = sv.stats()["launches"]
        sv.apply_gate(qs, U); o.apply_gate(qs, U)
        st = sv.stats()
        if kind == "relabel":
            assert st["class"] == "xor" and st["passes"] == 0 and st["launches"] == l0, (qs, st)
        elif kind == "phase":
            assert st["class"] == "xor" and st["passes"] == 1, (qs, st)
        assert sv.num_terms() == o.num_terms()
        assert_same_state(sv.export()[:2], o.export()[:2])
        assert sv.check_invariants()
    # ties by LOGICAL key after renaming: a flat state cut by the cap alone
    sv2 = eng.SparseSV(20, 1 << 12); o2 = _oracle(20)
    for q in range(10):
        sv2.apply_gate([q], W.mat_h()); o2.apply_gate([q], W.mat_h())
    for qs, U in (([0, 19], swap), ([5, 12, 18], cyc3), ([7, 15], xswap)):
        sv2.apply_gate(qs, U); o2.apply_gate(qs, U)
    kg, ko = sv2.truncate(300, 1.0), o2.truncate(300, 1.0)
    assert abs(kg - ko) <= 1e-12
    assert_same_state(sv2.export()[:2], o2.export()[:2])


def test_controlled_permutation_in_place_when_target_is_lsb(eng):
    """CNOT / Toffoli / controlled-Y whose target already sits at the physical LSB (the previous gate left it there) run
    IN PLACE: partners are stored neighbours, pairs trade amplitudes, lone members get their key's LSB flipped (SURVEY
    row f-4).  With pairs and lone members, phases, and a pending cut; against the oracle."""
    rng = np.random.default_rng(23)
    n = 52
    keys, amps = W.random_state(rng, n, 60000, spread=1.0)
    keys = np.unique(np.concatenate([keys, keys[:25000] ^ np.uint64(1 << 30)]))       # many stored partners on qubit 30
    amps = (rng.standard_normal(keys.size) + 1j * rng.standard_normal(keys.size)) * np.exp(rng.standard_normal(keys.size))
    amps /= np.sqrt(np.sum(np.abs(amps) ** 2))
    sv = eng.SparseSV(n, 1 << 19)
    sv.set_option(eng.OPT_SAMPLE_MIN_TERMS, 512)
    o = _oracle(n)
    sv.load(keys, amps); o.load(keys, amps)
    cy = np.zeros((4, 4), dtype=np.complex128)       # controlled-Y, qubits = (control, target)
    cy[0, 0] = cy[2, 2] = 1
    cy[3, 1] = 1j
    cy[1, 3] = -1j
    sv.apply_gate([30], W.mat_rx(0.9)); o.apply_gate([30], W.mat_rx(0.9))              # qubit 30 is the physical LSB now
    sv.profile(True)
    for i, (qs, U) in enumerate([([11, 30], W.mat_mcx(2)), ([5, 44, 30], W.mat_mcx(3)), ([2, 30], cy), ([1, 7, 50, 30], W.mat_mcx(4)),
                                 ([30, 11], W.mat_mcx(2))]):
        if i % 2 == 0:
            sv.truncate(0, 0.999); o.truncate(0, 0.999)
        sv.apply_gate(qs, U); o.apply_gate(qs, U)
        assert sv.stats()["class"] == "group"
        assert sv.num_terms() == o.num_terms()
        assert_same_state(sv.export()[:2], o.export()[:2])
        assert sv.check_invariants()
    pr = sv.profile_get()
    assert pr["diag"]["launches"] == 4 and pr["bitpass"]["launches"] == 1, pr      # four in place, the last one moves qubit 11
    sv.profile(False)
