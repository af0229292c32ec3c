"""GPU parity: sv_truncate through the C ABI vs the CPU oracle, and
step-locked circuit parity with truncation on (BASELINE.json configs[1], [3], [4] at scaled caps)."""
import numpy as np
import pytest

from paper_2607_07816_b200 import workloads as W

pytestmark = pytest.mark.gpu

from util_parity import assert_same_state, assert_truncation_parity, step_locked, MASS_TOL  # noqa: E402


class _Eng:
    """The engine module with the truncation-cut path pinned: 'full' = the full-state radix select,
    'sampled' = the one-pass sampled path (sv_sample_select.cu) from 512 terms on."""

    def __init__(self, engine, mode):
        self.engine, self.mode = engine, mode

    def SparseSV(self, n, cap, **kw):
        sv = self.engine.SparseSV(n, cap, **kw)
        sv.set_option(self.engine.OPT_SAMPLE_MIN_TERMS, (1 << 62) if self.mode == "full" else 512)
        return sv


@pytest.fixture(scope="module", params=["full", "sampled"])
def eng(request):
    from paper_2607_07816_b200 import engine
    return _Eng(engine, request.param)


def _oracle(n):
    from oracle.sparse import SparseOracle
    return SparseOracle(n)


def _pair(eng, n, keys, amps, cap=None):
    sv = eng.SparseSV(n, cap or (keys.size + 64))
    o = _oracle(n)
    sv.load(keys, amps)
    o.load(keys, amps)
    return sv, o


@pytest.mark.parametrize("count,K,f,spread", [
    (50000, 12345, 1.0, 2.0), (50000, 0, 0.97, 2.0), (50000, 20000, 0.999, 1.0), (50000, 100, 0.9999, 3.0),
    (3000, 1, 1.0, 2.0), (3000, 2999, 1.0, 0.1), (70001, 0, 0.5, 0.01), (70001, 0, 1e-9, 2.0), (1, 1, 0.5, 1.0),
    (200000, 65536, 1 - 1e-4, 1.5)])
def test_truncate_random(eng, count, K, f, spread):
    rng = np.random.default_rng(count + K)
    keys, amps = W.random_state(rng, 44, count, spread=spread)
    sv, o = _pair(eng, 44, keys, amps)
    kg = sv.truncate(K, f)
    ko = o.truncate(K, f)
    assert abs(kg - ko) <= MASS_TOL
    assert abs(sv.num_terms() - o.num_terms()) <= 2
    assert_truncation_parity(sv.export()[:2], o.export()[:2])
    assert sv.check_invariants()
    assert abs(sv.norm() - 1.0) <= 1e-13
    if eng.mode == "sampled" and count >= 50000:
        assert sv.stats()["fallbacks"] == 0, "the sampled band missed the cut on a generic state"


@pytest.mark.parametrize("K,f", [(1 << 20, 1.0), (0, 1 - 1e-4), (3 << 20, 0.9999), (0, 0.5), (16, 1.0)])
def test_truncate_large_sampled(eng, K, f):
    """2^22 generic terms: the sampled path with its full-size sample (2^17), vs the oracle."""
    if eng.mode != "sampled":
        pytest.skip("covered by the sampled mode")
    rng = np.random.default_rng(K + 7)
    keys, amps = W.random_state(rng, 50, 1 << 22, spread=1.5)
    sv, o = _pair(eng, 50, keys, amps)
    kg = sv.truncate(K, f)
    ko = o.truncate(K, f)
    assert abs(kg - ko) <= MASS_TOL
    assert abs(sv.num_terms() - o.num_terms()) <= 2
    assert_truncation_parity(sv.export()[:2], o.export()[:2])
    assert sv.stats()["fallbacks"] == 0
    assert sv.check_invariants()


def test_truncate_peaked_mass(eng):
    """One term carries most of the mass (a peaked state): the p-mass pivots must come from the
    tail, not from the sample's estimate of S."""
    rng = np.random.default_rng(11)
    keys, amps = W.random_state(rng, 44, 300000, spread=0.5)
    amps[12345] *= 3000.0
    amps /= np.sqrt(np.sum(np.abs(amps) ** 2))
    sv, o = _pair(eng, 44, keys, amps)
    for f in (1 - 1e-3, 1 - 1e-4):
        kg = sv.truncate(0, f)
        ko = o.truncate(0, f)
        assert abs(kg - ko) <= MASS_TOL
        assert abs(sv.num_terms() - o.num_terms()) <= 2
        assert_truncation_parity(sv.export()[:2], o.export()[:2])


def test_truncate_noop_bitwise(eng):
    rng = np.random.default_rng(0)
    keys, amps = W.random_state(rng, 30, 5000)
    sv, o = _pair(eng, 30, keys, amps)
    before = sv.export()
    for K, f in ((0, 1.0), (5000, 1.0), (10 ** 9, 2.0), (0, 1.0 - 1e-17)):
        assert sv.truncate(K, f) == 1.0
    after = sv.export()
    assert np.array_equal(before[0], after[0]) and np.array_equal(before[1], after[1])


def test_truncate_flat_ties_by_key(eng):
    """All p equal: the cut is decided by the LOGICAL key, ascending (reading R4), even after
    gates have permuted the storage order and set the lazy X mask."""
    n = 40
    sv = eng.SparseSV(n, 1 << 13)
    o = _oracle(n)
    for q in (3, 39, 17, 0, 8, 21, 11, 5, 30, 2, 25, 13):
        sv.apply_gate([q], W.mat_h())
        o.apply_gate([q], W.mat_h())
    for g in ((39,), (8,)):
        sv.apply_gate(list(g), W.mat_x())
        o.apply_gate(list(g), W.mat_x())
    sv.apply_gate([3, 30], W.mat_mcx(2))
    o.apply_gate([3, 30], W.mat_mcx(2))
    for K, f in ((1000, 1.0), (0, 0.3005), (77, 0.4995)):   # thresholds off the knife edge t*p == f*S (R5)
        kg = sv.truncate(K, f)
        ko = o.truncate(K, f)
        assert abs(kg - ko) <= MASS_TOL
        assert_same_state(sv.export()[:2], o.export()[:2])


@pytest.mark.parametrize("f,want", [(0.3, 300), (0.2999, 300), (0.3001, 301), (0.299, 299), (0.1, 100), (0.7, 700), (0.5, 500),
                                    (0.999, 999), (0.9991, 1000), (1e-9, 1)])
def test_truncate_knife_edge_closed_form(eng, f, want):
    """1000 equal terms of amplitude 2^-5 (p = 2^-10, every sum exact in fp64): thresholds at and beside the knife
    edge j * p == f * S.  min_mass = 0.3 keeps exactly 300 terms, the lowest logical keys ("minimum
    fraction of probability mass to keep"; readings R5, R22) -- a closed form, checked against the engine AND the
    oracle.  The storage order is scrambled first (H . H on two qubits moves bits, X sets the lazy mask)."""
    rng = np.random.default_rng(12)
    n = 30
    keys = np.sort(rng.choice(1 << n, size=1000, replace=False).astype(np.uint64))
    amps = np.full(1000, 2.0 ** -5 + 0.0j)
    sv, o = _pair(eng, n, keys, amps, cap=1 << 12)
    for q in (17, 3):                      # CNOT pairs: storage order changes, amplitudes stay bitwise
        for _ in range(2):
            sv.apply_gate([q, (q + 5) % n], W.mat_mcx(2))
    sv.apply_gate([29], W.mat_x()); sv.apply_gate([29], W.mat_x())
    kg = sv.truncate(0, f)
    ko = o.truncate(0, f)
    k, a, _ = sv.export()
    assert k.size == want == o.num_terms()
    assert np.array_equal(np.sort(k), keys[:want])
    assert kg == ko == want / 1000.0
    scale = 1.0 if want == 1000 else 1.0 / np.sqrt(want * 2.0 ** -10)
    assert np.all(a == (2.0 ** -5) * scale)
    assert_same_state(sv.export()[:2], o.export()[:2], tol=0.0)


def test_truncate_many_ties_mixed(eng):
    rng = np.random.default_rng(5)
    keys, amps = W.random_state(rng, 36, 60000, spread=1.0)
    amps = (np.round(amps * 512) / 512).astype(np.complex128)
    amps[amps == 0] = 1 / 512
    sv, o = _pair(eng, 36, keys, amps)
    for K, f in ((40000, 1.0), (0, 0.9), (5000, 0.99)):
        kg = sv.truncate(K, f)
        ko = o.truncate(K, f)
        assert abs(kg - ko) <= MASS_TOL
        assert sv.num_terms() == o.num_terms()
        assert_truncation_parity(sv.export()[:2], o.export()[:2])


def _run_step_locked(eng, c, cap, every=1):
    sv = eng.SparseSV(c.n, cap)
    make = lambda: _oracle(c.n)
    for i, g in enumerate(c.gates):
        if i % every == 0:
            step_locked(sv, make, g, c.max_terms, c.min_mass, c.truncate_every_gate)
        else:
            sv.apply_gate(g.qubits, g.U)
            if c.truncate_every_gate:
                sv.truncate(c.max_terms, c.min_mass)
        assert sv.check_invariants()
    return sv


def test_config2_scaled_step_locked(eng):
    """configs[1] mix at n=24 with the cap scaled to 2^12; every gate compared from the same pre-gate state."""
    c = W.config2(num_gates=250, max_terms=1 << 12)
    sv = _run_step_locked(eng, c, cap=1 << 14)
    assert sv.num_terms() <= 1 << 12


@pytest.mark.parametrize("variant", ["noh", "hboth"])
def test_config4_scaled_step_locked(eng, variant):
    """configs[3] (peaked, 3 layers, 10% 8x8, cap + mass 0.9999 after every gate) at n=16, K=2^11.  `hboth` is the
    variant bench.py runs: its flat 2^n H layer is cut by the key tie-break alone (reading R4)."""
    c = W.config4(n=16, max_terms=1 << 11, variant=variant)
    _run_step_locked(eng, c, cap=1 << 15)


def test_config5_scaled_step_locked(eng):
    """configs[4] mix at n=56 with K=2^12 and mass 1-1e-4; every gate compared."""
    c = W.config5(num_gates=300, max_terms=1 << 12)
    sv = _run_step_locked(eng, c, cap=1 << 16)
    assert sv.num_terms() <= 1 << 12


def test_config3_small_peak(eng):
    """configs[2] construction at n=14 (cap = 2^n, never binding): top bit string equals s."""
    c = W.config3(n=14, seed=2)
    sv = eng.SparseSV(c.n, 1 << 15)
    o = _oracle(c.n)
    for g in c.gates:
        sv.apply_gate(g.qubits, g.U)
        o.apply_gate(g.qubits, g.U)
        sv.truncate(c.max_terms, 1.0)
    k, a, p = sv.top(1)
    assert int(k[0]) == c.secret
    assert_same_state(sv.export()[:2], o.export()[:2], strict_keys=False)
    assert abs(sv.norm() - 1.0) <= 1e-12


def test_pending_cut_and_dead_entries_twin(eng):
    """The hot loop as the bench runs it: the truncation stays PENDING (and dead entries stay in place)
    when the next gate arrives -- no export in between.  A twin engine fed the same calls is exported
    before every gate to give the oracle the pre-gate state; the first engine's result must match."""
    c = W.config5(num_gates=220, max_terms=1 << 13)
    sv = eng.SparseSV(c.n, 1 << 17)
    twin = eng.SparseSV(c.n, 1 << 17)
    seen = set()
    for g in c.gates:
        k0, a0, _ = twin.export()            # (materialises the twin only)
        o = _oracle(c.n)
        o.load(k0, a0)
        sv.apply_gate(g.qubits, g.U)
        twin.apply_gate(g.qubits, g.U)
        o.apply_gate(g.qubits, g.U)
        assert sv.num_terms() == o.num_terms(), "term count after %s %r" % (g.name, g.qubits)
        kg = sv.truncate(c.max_terms, c.min_mass)
        kt = twin.truncate(c.max_terms, c.min_mass)
        ko = o.truncate(c.max_terms, c.min_mass)
        assert abs(kg - ko) <= MASS_TOL and abs(kt - ko) <= MASS_TOL
        assert sv.num_terms() == twin.num_terms()
        seen.add(g.klass)
    assert {"diag", "perm", "gen1", "gen2", "gen3"} <= seen
    assert_truncation_parity(sv.export()[:2], twin.export()[:2])
    assert sv.check_invariants()
    assert abs(sv.norm() - 1.0) <= 1e-12


def test_monomial_phase_gates_and_bit63_with_pending_cut(eng):
    """Position-preserving passes under a pending cut: monomial blocks with phases (controlled-Y), a plain
    CNOT on qubit 63, pure moves inside a 3-qubit gate, a diagonal gate -- each applied right after a
    truncation (no export in between) and compared with the oracle through a twin engine."""
    rng = np.random.default_rng(21)
    n = 64
    keys, amps = W.random_state(rng, n, 40000, spread=1.0)
    # give many terms a stored partner on qubits 63 and 7
    keys = np.unique(np.concatenate([keys, keys[:15000] ^ np.uint64(1 << 63), keys[5000:20000] ^ np.uint64(1 << 7)]))
    amps = (rng.standard_normal(keys.size) + 1j * rng.standard_normal(keys.size)) * np.exp(rng.standard_normal(keys.size))
    amps /= np.sqrt(np.sum(np.abs(amps) ** 2))
    sv = eng.SparseSV(n, 1 << 20)
    twin = eng.SparseSV(n, 1 << 20)
    sv.load(keys, amps)
    twin.load(keys, amps)
    cy = np.zeros((4, 4), dtype=np.complex128)       # controlled-Y, qubits = (control, target)
    cy[0, 0] = cy[2, 2] = 1
    cy[3, 1] = 1j
    cy[1, 3] = -1j
    gates = [([5, 63], cy), ([63, 7], W.mat_mcx(2)), ([7, 63], W.mat_mcx(2)), ([63], W.mat_rz(0.7)),
             ([63, 7, 30], W.haar_unitary(rng, 8)), ([11, 7], cy), ([7], W.mat_h()), ([40, 41, 63], W.mat_mcx(3)),
             ([63, 2], np.diag(np.exp(1j * rng.uniform(0, 6, 4)))), ([2, 63], W.haar_unitary(rng, 4))]
    for i, (qs, U) in enumerate(gates):
        f = 0.999 if i % 2 == 0 else 0.97
        kcap = 0 if i % 3 else 30000
        kg, kt = sv.truncate(kcap, f), twin.truncate(kcap, f)
        assert kg == kt
        k0, a0, _ = twin.export()
        o = _oracle(n)
        o.load(k0, a0)
        sv.apply_gate(qs, U)
        twin.apply_gate(qs, U)
        o.apply_gate(qs, U)
        assert sv.num_terms() == o.num_terms(), "gate %d" % i
        assert_same_state(sv.export()[:2], o.export()[:2])
        assert sv.check_invariants()
