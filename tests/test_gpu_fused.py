"""GPU parity of sv_apply_gate_truncate (include/sparse_sv.h; "apply, then truncate"):
the one call must give what sv_apply_gate + sv_truncate give -- against a twin engine that makes the
two calls, and against the CPU oracle -- also when the pass leaves out the outputs below a sampled
floor (sv_presample.cu), when that floor's margin fails and the pass is re-run, with a truncation
still pending on the input, and for gates the floor does not cover."""
import numpy as np
import pytest

from paper_2607_07816_b200 import workloads as W

pytestmark = pytest.mark.gpu

from util_parity import assert_truncation_parity, MASS_TOL  # noqa: E402


def _engines(n, cap, sample_min=512):
    from paper_2607_07816_b200 import engine
    a, b = engine.SparseSV(n, cap), engine.SparseSV(n, cap)
    for sv in (a, b):
        sv.set_option(engine.OPT_SAMPLE_MIN_TERMS, sample_min)
    return engine, a, b


def _oracle(n):
    from oracle.sparse import SparseOracle
    return SparseOracle(n)


def _rand_u2(rng):
    z = rng.normal(size=(2, 2)) + 1j * rng.normal(size=(2, 2))
    q, r = np.linalg.qr(z)
    return q * (np.diag(r) / np.abs(np.diag(r)))


def _ctrl(U, nctrl=1):
    d = 2 << nctrl
    M = np.eye(d, dtype=np.complex128)
    # target = local bit 0, controls = the higher local bits, all ones
    M[d - 2:, d - 2:] = 0
    for r in range(2):
        for c in range(2):
            M[(d - 2) | r, (d - 2) | c] = U[r, c]
    return M


def _same(a, b, exact=True):
    ka, aa, _ = a.export()
    kb, ab, _ = b.export()
    assert np.array_equal(ka, kb), "kept sets differ: %d vs %d terms" % (ka.size, kb.size)
    if exact:
        assert np.array_equal(aa, ab)
    else:
        assert np.allclose(aa, ab, rtol=1e-13, atol=0)


@pytest.mark.parametrize("qubit", [0, 1, 17, 43])
@pytest.mark.parametrize("frac,f", [(0.55, 1.0), (0.8, 1.0), (0.5, 1 - 1e-4), (1.4, 1.0)])
def test_fused_equals_two_calls(qubit, frac, f):
    """A dense one-qubit gate on 2^18 generic terms (every output is new: 2^19 before the cut)."""
    n, N = 44, 1 << 18
    rng = np.random.default_rng(qubit * 7 + int(frac * 100))
    keys, amps = W.random_state(rng, n, N, spread=1.5)
    eng, a, b = _engines(n, 2 * N + 64)
    a.load(keys, amps); b.load(keys, amps)
    U = _rand_u2(rng)
    K = int(frac * N)
    ka = a.apply_gate_truncate([qubit], U, K, f)
    st = a.stats()
    b.apply_gate([qubit], U)
    n_mid = b.num_terms()
    kb = b.truncate(K, f)
    assert st["n_mid"] == n_mid and st["n_in"] == N and st["n_out"] == b.num_terms()
    assert st["pre_dropped"] > 0 and st["fallbacks"] == 0, st      # the floor was used, and it held
    assert st["pre_dropped"] < n_mid - K
    assert abs(ka - kb) <= 1e-13
    _same(a, b, exact=(f >= 1.0))
    assert a.check_invariants()
    assert abs(a.norm() - 1.0) <= 1e-13


def _ctrl_block(V, nctrl=1):
    """V on the low local bits, applied when the nctrl high local bits are all ones."""
    d = V.shape[0]
    D = d << nctrl
    M = np.eye(D, dtype=np.complex128)
    M[D - d:, D - d:] = V
    return M


@pytest.mark.parametrize("qubits,frac", [((5, 30), 0.9), ((0, 1), 1.5), ((43, 2), 3.0), ((7, 19, 33), 1.2), ((1, 0, 2), 5.0),
                                          ((12, 40, 3, 27), 2.0)])
def test_fused_multi_bit_gate_equals_two_calls(qubits, frac):
    """Haar gates on 2, 3 and 4 qubits on generic terms (4x, 8x, 16x outputs before the cut): the count pass +
    write pass of sv_group.cu (PRE) against apply + truncate."""
    m = len(qubits)
    n, N = 44, (1 << 17) if m < 4 else (1 << 15)
    rng = np.random.default_rng(sum(qubits) + m)
    keys, amps = W.random_state(rng, n, N, spread=1.5)
    eng, a, b = _engines(n, (1 << m) * N + 64)
    a.load(keys, amps); b.load(keys, amps)
    U = W.haar_unitary(rng, 1 << m)
    K = int(frac * N)
    ka = a.apply_gate_truncate(list(qubits), U, K, 1.0)
    st = a.stats()
    b.apply_gate(list(qubits), U)
    n_mid = b.num_terms()
    kb = b.truncate(K, 1.0)
    assert st["n_mid"] == n_mid and st["n_out"] == b.num_terms() == K
    assert st["pre_dropped"] > 0 and st["fallbacks"] == 0, st
    assert abs(ka - kb) <= 1e-13
    _same(a, b)
    assert a.check_invariants()


def test_fused_multi_bit_chain_with_controls_and_pending_cuts():
    """A chain of fused calls: SU(4), controlled SU(4) (3 qubits, 2 active), 8x8, H, diagonal and CNOT gates in
    between, mass + cap criteria, so that every pass meets a pending cut and dead entries."""
    n, N = 40, 1 << 16
    rng = np.random.default_rng(77)
    keys, amps = W.random_state(rng, n, N, spread=1.0)
    eng, a, b = _engines(n, 16 * N)
    a.load(keys, amps); b.load(keys, amps)
    K = N
    used = 0
    for step in range(14):
        kind = step % 7
        if kind == 0:
            q, U = [int(x) for x in rng.choice(n, 2, replace=False)], W.haar_unitary(rng, 4)
        elif kind == 1:
            q, U = [int(x) for x in rng.choice(n, 3, replace=False)], _ctrl_block(W.haar_unitary(rng, 4))
        elif kind == 2:
            q, U = [int(x) for x in rng.choice(n, 1)], W.mat_rz(0.7)
        elif kind == 3:
            q, U = [int(x) for x in rng.choice(n, 3, replace=False)], W.haar_unitary(rng, 8)
        elif kind == 4:
            q, U = [int(x) for x in rng.choice(n, 2, replace=False)], W.mat_mcx(2)
        elif kind == 5:
            q, U = [int(x) for x in rng.choice(n, 1)], W.mat_h()
        else:
            q, U = [int(x) for x in rng.choice(n, 2, replace=False)], _ctrl_block(_rand_u2(rng))
        fa, fb = a.stats()["fallbacks"], b.stats()["fallbacks"]
        ka = a.apply_gate_truncate(q, U, K, 1 - 1e-6)
        used += 1 if a.stats()["pre_dropped"] else 0
        b.apply_gate(q, U); kb = b.truncate(K, 1 - 1e-6)
        assert abs(ka - kb) <= 1e-13, (step, ka, kb)
        _same(a, b, exact=False)
        print("step", step, kind, a.stats()["n_in"], a.stats()["n_mid"], a.stats()["n_out"], "pre", a.stats()["pre_dropped"],
              "fallbacks +%d / +%d" % (a.stats()["fallbacks"] - fa, b.stats()["fallbacks"] - fb))
    assert used >= 6, used
    assert a.stats()["fallbacks"] <= b.stats()["fallbacks"] + 1
    assert a.check_invariants()


def test_fused_with_pending_cut_and_controls():
    """The input carries a deferred truncation and dead entries; controlled gates (only the control = 1
    tuples mix), then a chain of fused calls."""
    n, N = 40, 1 << 17
    rng = np.random.default_rng(5)
    keys, amps = W.random_state(rng, n, N, spread=1.0)
    eng, a, b = _engines(n, 4 * N)
    a.load(keys, amps); b.load(keys, amps)
    K = N // 2
    for sv in (a, b):
        sv.truncate(int(0.9 * N), 1.0)                    # stays pending
        sv.apply_gate([3, 20], W.mat_mcx(2))              # position preserving: dropped terms become dead entries
        sv.truncate(int(0.85 * N), 1.0)
    used = 0
    for step in range(8):
        q = [int(x) for x in rng.choice(n, size=2, replace=False)]
        U = _ctrl(_rand_u2(rng)) if step % 2 else None
        if U is None:
            q, U = q[:1], _rand_u2(rng)
        ka = a.apply_gate_truncate(q, U, K, 1 - 1e-6)
        used += 1 if a.stats()["pre_dropped"] else 0
        b.apply_gate(q, U); kb = b.truncate(K, 1 - 1e-6)
        assert abs(ka - kb) <= 1e-13
        _same(a, b, exact=False)
    assert used >= 4
    assert a.check_invariants()


def test_fused_floor_margin_failure_reruns():
    """A floor that is far too high (negative slack) leaves fewer than max_terms outputs: the pass must be
    re-run without it and the result must not change."""
    n, N = 44, 1 << 17
    rng = np.random.default_rng(9)
    keys, amps = W.random_state(rng, n, N, spread=1.5)
    eng, a, b = _engines(n, 4 * N)
    a.load(keys, amps); b.load(keys, amps)
    a.test_set_pre_slack(-3000)
    U = _rand_u2(rng)
    K = int(0.6 * N)
    ka = a.apply_gate_truncate([5], U, K, 1.0)
    st = a.stats()
    assert st["fallbacks"] == 1 and st["pre_dropped"] == 0, st
    b.apply_gate([5], U); kb = b.truncate(K, 1.0)
    assert abs(ka - kb) <= 1e-13
    _same(a, b)
    U4 = W.haar_unitary(rng, 4)                           # the same for the multi-bit pass
    ka = a.apply_gate_truncate([8, 21], U4, K, 1.0)
    st = a.stats()
    assert st["fallbacks"] == 2 and st["pre_dropped"] == 0, st
    b.apply_gate([8, 21], U4); kb = b.truncate(K, 1.0)
    assert abs(ka - kb) <= 1e-13
    _same(a, b)


@pytest.mark.parametrize("pending", [False, True])
def test_fused_diagonal_gate_rides_on_the_classification_pass(pending):
    """Diagonal gates (RZ, T, CZ, CCZ, a non-unitary diagonal): the fused call applies them inside the sampled
    truncation's pass over the state; with and without a truncation pending on the input (dead entries)."""
    n, N = 44, 1 << 18
    rng = np.random.default_rng(31 + pending)
    keys, amps = W.random_state(rng, n, N, spread=1.5)
    eng, a, b = _engines(n, N + 64)
    a.load(keys, amps); b.load(keys, amps)
    if pending:
        for sv in (a, b):
            sv.truncate(int(0.97 * N), 1.0)
            sv.apply_gate([2, 30], W.mat_mcx(2))          # position preserving: the dropped 3 % are dead entries now
            sv.truncate(int(0.95 * N), 1.0)               # and this one stays pending
    gates = [([7], W.mat_rz(0.3)), ([40], W.mat_t()), ([3, 25], W.mat_diag_minus_last(2)), ([0, 43, 12], W.mat_diag_minus_last(3)),
             ([9, 1], np.diag([1.0, 0.5j, -2.0, 0.25]).astype(np.complex128))]
    K = int(0.9 * N)
    for i, (q, U) in enumerate(gates):
        f = 1.0 if i % 2 == 0 else 1 - 1e-5
        l0 = a.stats()["launches"]
        ka = a.apply_gate_truncate(q, U, K, f)
        la = a.stats()["launches"] - l0
        l0 = b.stats()["launches"]
        b.apply_gate(q, U); kb = b.truncate(K, f)
        lb = b.stats()["launches"] - l0
        assert la == lb - 1, "the fused call must save exactly the diagonal pass (%d vs %d launches)" % (la, lb)
        assert ka == kb
        _same(a, b)
        K = int(0.97 * K)
    assert a.check_invariants()
    assert a.stats()["fallbacks"] == 0


def test_fused_diagonal_without_a_cut_still_applies_the_gate():
    n, N = 40, 1 << 16
    rng = np.random.default_rng(3)
    keys, amps = W.random_state(rng, n, N, spread=1.0)
    eng, a, b = _engines(n, N + 64)
    a.load(keys, amps); b.load(keys, amps)
    assert a.apply_gate_truncate([5], W.mat_rz(1.1), 0, 1.0) == 1.0          # nothing to cut
    assert a.apply_gate_truncate([6], W.mat_t(), 2 * N, 2.0) == 1.0
    b.apply_gate([5], W.mat_rz(1.1)); b.apply_gate([6], W.mat_t())
    _same(a, b)


def test_fused_mass_only_and_count_only_criteria():
    """max_terms = 0 (p-mass threshold only: no output floor, but the diagonal gate still rides on the classify pass)
    and min_mass >= 1 (cap only), general and diagonal gates, after a host load (total mass not yet known exactly)."""
    n, N = 42, 1 << 17
    rng = np.random.default_rng(12)
    keys, amps = W.random_state(rng, n, N, spread=1.5)
    amps *= 1.7                                            # not normalised: S != 1
    eng, a, b = _engines(n, 16 * N)
    a.load(keys, amps); b.load(keys, amps)
    seq = [([4], _rand_u2(rng), 0, 1 - 1e-3), ([9], W.mat_rz(0.4), 0, 1 - 1e-4), ([30, 2], W.haar_unitary(rng, 4), 0, 0.99),
           ([11], W.mat_t(), N // 2, 2.0), ([6], _rand_u2(rng), N // 3, 1.0), ([1, 40], W.mat_diag_minus_last(2), 0, 0.999)]
    for q, U, K, f in seq:
        ka = a.apply_gate_truncate(q, U, K, f)
        b.apply_gate(q, U); kb = b.truncate(K, f)
        assert abs(ka - kb) <= 1e-13, (q, K, f, ka, kb)
        _same(a, b, exact=False)
    assert a.check_invariants()
    assert abs(a.norm() - 1.0) <= 1e-13


@pytest.mark.parametrize("f", [1.0, 1 - 1e-3])
def test_fused_floor_then_full_state_select(f):
    """The input is large enough for the output floor, but the cap is so small that what the pass stores falls below
    the sampling threshold: the truncation then runs the FULL-state select, which must still count the left-out
    outputs' mass in S (kept fraction) and treat them as dropped."""
    n, N = 44, 1 << 17
    rng = np.random.default_rng(21)
    keys, amps = W.random_state(rng, n, N, spread=1.5)
    eng, a, b = _engines(n, 4 * N, sample_min=N)
    a.load(keys, amps); b.load(keys, amps)
    K = 1 << 12
    for q, U in (([7], _rand_u2(rng)),):
        ka = a.apply_gate_truncate(q, U, K, f)
        st = a.stats()
        assert st["pre_dropped"] > 0 and st["n_mid"] - st["pre_dropped"] < N, st
        b.apply_gate(q, U); kb = b.truncate(K, f)
        assert abs(ka - kb) <= 1e-13, (ka, kb)
        _same(a, b, exact=(f >= 1.0))
    o = _oracle(n)
    o.load(keys, amps); o.apply_gate([7], U); ko = o.truncate(K, f)
    assert abs(ka - ko) <= MASS_TOL
    assert_truncation_parity(a.export()[:2], o.export()[:2])


def test_fused_uncovered_gates_and_small_states():
    """Diagonal, permutation and multi-bit gates, and states below the sampling threshold, take the
    two calls internally."""
    n = 30
    rng = np.random.default_rng(2)
    keys, amps = W.random_state(rng, n, 20000, spread=1.0)
    eng, a, b = _engines(n, 1 << 19, sample_min=1 << 40)
    a.load(keys, amps); b.load(keys, amps)
    gates = [([4], W.mat_h()), ([7, 2], W.mat_mcx(2)), ([1, 9], np.diag(np.exp(1j * rng.normal(size=4)))),
             ([3, 11], W.haar_unitary(rng, 4)), ([6], _rand_u2(rng))]
    for q, U in gates:
        ka = a.apply_gate_truncate(q, U, 15000, 1 - 1e-5)
        assert a.stats()["pre_dropped"] == 0
        b.apply_gate(q, U); kb = b.truncate(15000, 1 - 1e-5)
        assert ka == kb
        _same(a, b)


def test_fused_vs_oracle_step_locked():
    """Config-5-like steps at a scaled cap, every gate through the fused call, against the oracle's
    apply + truncate from the same pre-gate state."""
    n, K = 40, 1 << 15
    c = W.config5(n=n, num_gates=200, max_terms=K)
    from paper_2607_07816_b200 import engine
    sv = engine.SparseSV(c.n, 16 * K)
    sv.set_option(engine.OPT_SAMPLE_MIN_TERMS, 512)
    used = 0
    for i, g in enumerate(c.gates[:140]):
        k0, a0, _ = sv.export()
        o = _oracle(c.n)
        o.load(k0, a0)
        kg = sv.apply_gate_truncate(g.qubits, g.U, K, c.min_mass)
        used += 1 if sv.stats()["pre_dropped"] else 0
        o.apply_gate(g.qubits, g.U)
        ko = o.truncate(K, c.min_mass)
        assert abs(kg - ko) <= MASS_TOL, (i, kg, ko)
        gk, ga, gp = sv.export()
        ok_, oa, _ = o.export()
        assert_truncation_parity((gk, ga), (ok_, oa))
    assert used > 0, "no gate of the sequence used the output floor"
    assert sv.check_invariants()
