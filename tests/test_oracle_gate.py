"""Pins for the CPU oracle's gate step (oracle/sv_oracle.cpp orc_apply_gate).

Everything here checks the oracle against something other than itself: the dense 2^n
simulator (oracle/dense.py, Eq. 3 / :47-49), hand-derived closed forms
(tests/golden/closed_forms.txt), and invariants the paper states.
"""
import math
import os

import numpy as np
import pytest

from oracle import dense
from oracle.sparse import SparseOracle
from paper_2607_07816_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")

NAMED = {
    "h": (1, W.mat_h), "x": (1, W.mat_x), "s": (1, W.mat_s), "t": (1, W.mat_t),
    "cx": (2, lambda: W.mat_mcx(2)), "ccx": (3, lambda: W.mat_mcx(3)),
    "c3x": (4, lambda: W.mat_mcx(4)), "cz": (2, lambda: W.mat_diag_minus_last(2)),
    "ccz": (3, lambda: W.mat_diag_minus_last(3)),
}


def _parse_golden():
    cases = []
    sym = {"r": 1.0 / math.sqrt(2.0), "h": 0.5, "-r": -1.0 / math.sqrt(2.0), "-h": -0.5}
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        n, gates, terms = [x.strip() for x in line.split("|")]
        gl = []
        for g in gates.split(";"):
            tok = g.split()
            gl.append((tok[0], [int(t) for t in tok[1:]]))
        exp = {}
        for t in terms.split():
            k, v = t.split(":")
            re, im = v.split(",")
            f = lambda s: sym[s] if s in sym else float(s)
            exp[int(k)] = complex(f(re), f(im))
        cases.append((int(n), gl, exp))
    return cases


@pytest.mark.parametrize("case", _parse_golden())
def test_closed_forms(case):
    n, gl, exp = case
    o = SparseOracle(n)
    for name, qs in gl:
        m, f = NAMED[name]
        assert len(qs) == m
        o.apply_gate(qs, f())
    got = o.as_dict()
    assert set(got) == set(exp)
    for k in exp:
        assert abs(got[k] - exp[k]) <= 4e-16


def _compare_dense(o: SparseOracle, psi: np.ndarray, tol=1e-12):
    got = np.zeros_like(psi)
    k, a, _ = o.export()
    got[k.astype(np.int64)] = a
    assert np.max(np.abs(got - psi)) <= tol


def test_config1_every_gate_vs_dense():
    """BASELINE.json configs[0]: n=12, H layer + 6 brickwork layers of SU(4); every gate."""
    c = W.config1()
    assert len(c.gates) == 12 + 33
    o = SparseOracle(c.n)
    psi = dense.ground(c.n)
    for g in c.gates:
        o.apply_gate(g.qubits, g.U)
        psi = dense.apply_gate(psi, c.n, g.qubits, g.U)
        _compare_dense(o, psi)
    assert o.num_terms() <= 4096
    assert abs(o.norm() - 1.0) <= 1e-13 * len(c.gates)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_random_circuits_vs_dense(seed):
    """Random gates of every kind, m = 1..4, unordered and non-adjacent qubits: a wrong
    index order (R2), a transposed U, or a dropped contribution fails here."""
    rng = np.random.default_rng(100 + seed)
    n = 9
    o = SparseOracle(n)
    psi = dense.ground(n)
    for step in range(60):
        m = int(rng.integers(1, 5))
        qs = [int(q) for q in rng.choice(n, size=m, replace=False)]
        kind = int(rng.integers(0, 4))
        if kind == 0:
            U = W.haar_unitary(rng, 1 << m)
        elif kind == 1:
            U = np.diag(np.exp(1j * rng.uniform(0, 2 * np.pi, 1 << m)))
        elif kind == 2:
            U = W.mat_mcx(m) if m > 1 else W.mat_x()
        else:  # a non-unitary dense matrix: the update rule is linear algebra, not physics
            U = rng.standard_normal((1 << m, 1 << m)) + 1j * rng.standard_normal((1 << m, 1 << m))
            U = U / np.linalg.norm(U, 2)
        o.apply_gate(qs, U)
        psi = dense.apply_gate(psi, n, qs, U)
        _compare_dense(o, psi, tol=1e-12)


def test_dense_simulator_matches_kron():
    """Pin the dense simulator itself against numpy kron (library routine) at n = 3."""
    rng = np.random.default_rng(7)
    n = 3
    psi = rng.standard_normal(8) + 1j * rng.standard_normal(8)
    U = W.haar_unitary(rng, 2)
    I = np.eye(2)
    # qubit q is bit q: index = b2 b1 b0, kron order (q2, q1, q0)
    for q, full in [(0, np.kron(np.kron(I, I), U)), (1, np.kron(np.kron(I, U), I)), (2, np.kron(np.kron(U, I), I))]:
        assert np.allclose(dense.apply_gate(psi, n, [q], U), full @ psi, atol=1e-14)
    U4 = W.haar_unitary(rng, 4)
    # qubits (0, 1): local index = b1 b0 -> kron(I, U4) acts on the low two bits
    assert np.allclose(dense.apply_gate(psi, n, [0, 1], U4), np.kron(I, U4) @ psi, atol=1e-14)
    # qubits (1, 0): local bit 0 = qubit 1 -> U4 with its two local bits swapped
    P = np.eye(4)[[0, 2, 1, 3]]
    assert np.allclose(dense.apply_gate(psi, n, [1, 0], U4), np.kron(I, P @ U4 @ P) @ psi, atol=1e-14)


def test_ground_state_single_term():
    o = SparseOracle(40)
    k, a, p = o.export()
    assert list(k) == [0] and a[0] == 1.0 and p[0] == 1.0


def test_h_growth_bitwise():
    """H on j fresh qubits -> exactly 2^j terms, all equal to (1/sqrt2)^j
    multiplied out one factor at a time."""
    n = 30
    o = SparseOracle(n)
    amp = 1.0
    r = 1.0 / math.sqrt(2.0)
    qs = [3, 17, 29, 0, 8, 21, 11, 5]
    for j, q in enumerate(qs, 1):
        o.apply_gate([q], W.mat_h())
        amp = r * amp
        k, a, _ = o.export()
        assert k.size == 1 << j
        assert np.all(a.real == amp) and np.all(a.imag == 0.0)
        mask = sum(1 << x for x in qs[:j])
        assert np.all((k & ~np.uint64(mask)) == 0)


def test_monomial_gates_preserve_count_and_amplitudes():
    """CNOT / Toffoli / 4-qubit Toffoli only permute."""
    rng = np.random.default_rng(5)
    n = 20
    keys, amps = W.random_state(rng, n, 3000)
    o = SparseOracle(n)
    o.load(keys, amps)
    for m in (1, 2, 3, 4):
        qs = [int(q) for q in rng.choice(n, size=m, replace=False)]
        before = o.as_dict()
        o.apply_gate(qs, W.mat_mcx(m) if m > 1 else W.mat_x())
        after = o.as_dict()
        assert len(after) == len(before)
        cm = sum(1 << q for q in qs[:-1])
        for k, a in before.items():
            k2 = k ^ (1 << qs[-1]) if (k & cm) == cm else k
            assert after[k2] == a  # bitwise


def test_diagonal_gates_keep_keys():
    rng = np.random.default_rng(6)
    n = 18
    keys, amps = W.random_state(rng, n, 2000)
    o = SparseOracle(n)
    o.load(keys, amps)
    th = 1.234
    o.apply_gate([7], W.mat_rz(th))
    after = o.as_dict()
    for k, a in zip(keys, amps):
        ph = np.exp(1j * th / 2) if (int(k) >> 7) & 1 else np.exp(-1j * th / 2)
        assert abs(after[int(k)] - ph * a) <= 4e-16 * abs(a) + 1e-300


def test_ghz_64():
    n = 64
    o = SparseOracle(n)
    o.apply_gate([0], W.mat_h())
    for q in range(1, n):
        o.apply_gate([q - 1, q], W.mat_mcx(2))
    d = o.as_dict()
    r = 1.0 / math.sqrt(2.0)
    assert d == {0: complex(r, 0), (1 << 64) - 1: complex(r, 0)}


def test_r_rdagger_returns_ground_state():
    """R then R^dagger = identity; exact-zero drop leaves ~1e-16 residues (reading R3), so
    the check is tolerance based, not a term count."""
    rng = np.random.default_rng(11)
    n = 10
    R = W.brickwork(rng, n, 3)
    o = SparseOracle(n)
    for g in R + W.adjoint(R):
        o.apply_gate(g.qubits, g.U)
    d = o.as_dict()
    assert abs(d[0] - 1.0) <= 1e-12
    assert sum(abs(a) ** 2 for k, a in d.items() if k != 0) <= 1e-24
    o.truncate(1, 1.0)
    k, a, _ = o.export()
    assert list(k) == [0]


@pytest.mark.parametrize("variant", ["hboth", "noh"])
@pytest.mark.parametrize("n", [10, 12])
def test_peaked_circuit_top_is_secret(variant, n):
    c = W.config3(n=n, seed=2 + n, variant=variant)
    o = SparseOracle(n)
    for g in c.gates:
        o.apply_gate(g.qubits, g.U)
    k, a, p = o.top(1)
    assert int(k[0]) == c.secret
    assert 0.3 < p[0] <= 1.0
    assert abs(o.norm() - 1.0) <= 1e-12


def test_invalid_arguments():
    o = SparseOracle(4)
    with pytest.raises(ValueError):
        o.apply_gate([0, 0], W.mat_mcx(2))
    with pytest.raises(ValueError):
        o.apply_gate([4], W.mat_h())
