"""Seeded synthetic circuits (input generators only).

This module builds gate lists: (name, qubits, U) records.  It holds none of the
method's arithmetic (no gate application, no truncation), so both the CPU oracle
(`oracle/`) and the CUDA engine may be fed from it without sharing code.

The five circuits are the ones BASELINE.json `configs[0..4]` describes; they
stand in for the paper's BlueQubit "sharp peak" workload,
which is not available.  Conventions:

* qubit q is bit q of the uint64 key (LSB = qubit 0)                      [R1]
* U is row-major 2^m x 2^m, U[r, c]; bit j of the local index r / c is the
  key's bit ``qubits[j]``                                                  [R2]
* named gates are the OpenQASM 2.0 / qelib1 matrices (ref [1]) [R16]
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np

C128 = np.complex128


@dataclass
class Gate:
    name: str
    qubits: Tuple[int, ...]
    U: np.ndarray            # (2^m, 2^m) complex128, row-major U[r, c]
    klass: str = ""          # reporting class: diag | perm | gen1 | gen2 | gen3

    @property
    def m(self) -> int:
        return len(self.qubits)


@dataclass
class Circuit:
    name: str
    n: int
    gates: List[Gate]
    max_terms: int = 0           # 0 = no cap             (PAPER.md:91 top-k)
    min_mass: float = 1.0        # >= 1 = no mass cut     (PAPER.md:92 p-mass)
    truncate_every_gate: bool = False
    secret: Optional[int] = None  # peak bit string, when known by construction
    notes: dict = field(default_factory=dict)


# --------------------------------------------------------------------------
# gate library (qelib1 matrices, PAPER.md:57 ref [1])
# --------------------------------------------------------------------------
_S2 = 1.0 / math.sqrt(2.0)


def mat_h() -> np.ndarray:
    return np.array([[_S2, _S2], [_S2, -_S2]], dtype=C128)


def mat_x() -> np.ndarray:
    return np.array([[0, 1], [1, 0]], dtype=C128)


def mat_s() -> np.ndarray:
    return np.array([[1, 0], [0, 1j]], dtype=C128)


def mat_t() -> np.ndarray:
    return np.array([[1, 0], [0, complex(_S2, _S2)]], dtype=C128)


def mat_rz(theta: float) -> np.ndarray:
    h = 0.5 * theta
    return np.array([[complex(math.cos(h), -math.sin(h)), 0],
                     [0, complex(math.cos(h), math.sin(h))]], dtype=C128)


def mat_rx(theta: float) -> np.ndarray:
    h = 0.5 * theta
    c, s = math.cos(h), math.sin(h)
    return np.array([[c, complex(0, -s)], [complex(0, -s), c]], dtype=C128)


def mat_u3(theta: float, phi: float, lam: float) -> np.ndarray:
    """qelib1 u3(theta, phi, lambda) (PAPER.md:150-171 uses u3 and cz only)."""
    c, sn = math.cos(0.5 * theta), math.sin(0.5 * theta)
    if theta == math.pi:
        c = 0.0              # cos(fl(pi)/2) rounds to 6e-17; with the exact 0, u3(pi, 0, pi) is the monomial X
    return np.array([[c, -cmath_exp(lam) * sn],
                     [cmath_exp(phi) * sn, cmath_exp(phi + lam) * c]], dtype=C128)


def cmath_exp(a: float) -> complex:
    return complex(math.cos(a), math.sin(a))


def mat_diag_minus_last(m: int) -> np.ndarray:
    """CZ (m=2) / CCZ (m=3): identity with -1 on |1..1>."""
    d = np.ones(1 << m, dtype=C128)
    d[-1] = -1
    return np.diag(d)


def mat_mcx(m: int) -> np.ndarray:
    """(m-1)-controlled X.  qubits = (controls..., target): local bits
    0..m-2 are controls, bit m-1 is the target  [R2]."""
    d = 1 << m
    U = np.zeros((d, d), dtype=C128)
    cmask = (1 << (m - 1)) - 1
    for c in range(d):
        r = c ^ (1 << (m - 1)) if (c & cmask) == cmask else c
        U[r, c] = 1
    return U


def haar_unitary(rng: np.random.Generator, d: int, special: bool = False) -> np.ndarray:
    """Haar-random d x d unitary: Ginibre matrix + modified Gram-Schmidt
    (= QR with positive diagonal R).  special=True divides by det^(1/d)  [R18]."""
    g = rng.standard_normal((d, d)) + 1j * rng.standard_normal((d, d))
    q = np.zeros((d, d), dtype=C128)
    for j in range(d):
        v = g[:, j].astype(C128).copy()
        for _ in range(2):  # re-orthogonalise once; keeps U^dagger U = I to ~1e-16
            for i in range(j):
                v = v - np.vdot(q[:, i], v) * q[:, i]
        q[:, j] = v / math.sqrt(float(np.vdot(v, v).real))
    if special:
        det = complex(np.linalg.det(q))
        q = q * np.exp(-1j * np.angle(det) / d)
    return np.ascontiguousarray(q)


def G(name: str, qubits: Sequence[int], U: np.ndarray, klass: str) -> Gate:
    return Gate(name, tuple(int(q) for q in qubits), np.ascontiguousarray(U, dtype=C128), klass)


# --------------------------------------------------------------------------
# building blocks
# --------------------------------------------------------------------------

def h_layer(n: int) -> List[Gate]:
    return [G("h", (q,), mat_h(), "gen1") for q in range(n)]


def brickwork(rng, n: int, layers: int, p3: float = 0.0) -> List[Gate]:
    """Brickwork of Haar SU(4) on (a, a+1), a = layer mod 2, +2, ... <= n-2 (no
    wrap-around) [R15].  With p3 > 0 a gate is replaced with probability p3 by a
    Haar 8x8 on (a, a+1, a+2) when that fits, advancing by 3  [R14]."""
    out: List[Gate] = []
    for layer in range(layers):
        a = layer % 2
        while a + 1 <= n - 1:
            if p3 > 0.0 and a + 2 <= n - 1 and rng.random() < p3:
                out.append(G("u8", (a, a + 1, a + 2), haar_unitary(rng, 8), "gen3"))
                a += 3
            else:
                out.append(G("su4", (a, a + 1), haar_unitary(rng, 4, special=True), "gen2"))
                a += 2
    return out


def adjoint(gates: List[Gate]) -> List[Gate]:
    return [G(g.name + "_dg", g.qubits, g.U.conj().T, g.klass) for g in reversed(gates)]


def peaked(rng, n: int, layers: int, p3: float, variant: str) -> Tuple[List[Gate], int]:
    """BASELINE.json configs[2]/[3]: H^n, R, D = RZ(theta_q ~ N(0, 0.3^2)), R^dagger,
    X where s has a 1.  variant (reading R12):
      'literal' - exactly that list (not peaked at s: R^dagger D R ~ I on |+>^n)
      'hboth'   - a closing H layer before the X layer (peaked at s); default
      'noh'     - no H layers at all (peaked at s, sparse start)."""
    R = brickwork(rng, n, layers, p3)
    D = [G("rz", (q,), mat_rz(float(rng.normal(0.0, 0.3))), "diag") for q in range(n)]
    s = int(rng.integers(0, 1 << n, dtype=np.uint64)) if n < 64 else int(rng.integers(0, 1 << 63, dtype=np.uint64))
    gates: List[Gate] = []
    if variant in ("literal", "hboth"):
        gates += h_layer(n)
    gates += R + D + adjoint(R)
    if variant == "hboth":
        gates += h_layer(n)
    gates += [G("x", (q,), mat_x(), "perm") for q in range(n) if (s >> q) & 1]
    return gates, s


def _pick(rng, n: int, m: int, pool: Optional[np.ndarray] = None) -> Tuple[int, ...]:
    if pool is None:
        return tuple(int(q) for q in rng.choice(n, size=m, replace=False))
    return tuple(int(q) for q in rng.choice(pool, size=m, replace=False))


# --------------------------------------------------------------------------
# the five configs (BASELINE.json configs[0..4])
# --------------------------------------------------------------------------

def config1(n: int = 12, layers: int = 6, seed: int = 0) -> Circuit:
    rng = np.random.default_rng(seed)
    gates = h_layer(n) + brickwork(rng, n, layers)
    return Circuit("cfg1", n, gates)


def config2(n: int = 24, num_gates: int = 400, seed: int = 1, max_terms: int = 1 << 20) -> Circuit:
    """25% H, 15% RZ, 10% RX, 10% T/S, 20% CNOT, 10% CZ, 5% Haar U3, 5% Toffoli;
    qubits uniform over all n, distinct within a gate  [R17]."""
    rng = np.random.default_rng(seed)
    kinds = ["h", "rz", "rx", "ts", "cnot", "cz", "u3", "ccx"]
    probs = [0.25, 0.15, 0.10, 0.10, 0.20, 0.10, 0.05, 0.05]
    gates: List[Gate] = []
    for _ in range(num_gates):
        k = kinds[int(rng.choice(len(kinds), p=probs))]
        if k == "h":
            gates.append(G("h", _pick(rng, n, 1), mat_h(), "gen1"))
        elif k == "rz":
            q = _pick(rng, n, 1)
            gates.append(G("rz", q, mat_rz(float(rng.uniform(0, 2 * math.pi))), "diag"))
        elif k == "rx":
            q = _pick(rng, n, 1)
            gates.append(G("rx", q, mat_rx(float(rng.uniform(0, 2 * math.pi))), "gen1"))
        elif k == "ts":
            q = _pick(rng, n, 1)
            gates.append(G("t", q, mat_t(), "diag") if rng.random() < 0.5 else G("s", q, mat_s(), "diag"))
        elif k == "cnot":
            gates.append(G("cx", _pick(rng, n, 2), mat_mcx(2), "perm"))
        elif k == "cz":
            gates.append(G("cz", _pick(rng, n, 2), mat_diag_minus_last(2), "diag"))
        elif k == "u3":
            q = _pick(rng, n, 1)
            gates.append(G("u3", q, haar_unitary(rng, 2), "gen1"))
        else:
            gates.append(G("ccx", _pick(rng, n, 3), mat_mcx(3), "perm"))
    return Circuit("cfg2", n, gates, max_terms=max_terms, min_mass=1.0, truncate_every_gate=True)


def config3(n: int = 26, seed: int = 2, variant: str = "hboth", max_terms: Optional[int] = None) -> Circuit:
    rng = np.random.default_rng(seed)
    gates, s = peaked(rng, n, layers=2, p3=0.0, variant=variant)
    return Circuit("cfg3", n, gates, max_terms=(1 << n) if max_terms is None else max_terms,
                   secret=s, notes={"variant": variant})


def config4(n: int = 32, seed: int = 3, variant: str = "hboth", max_terms: int = 1 << 27,
            min_mass: float = 0.9999) -> Circuit:
    rng = np.random.default_rng(seed)
    gates, s = peaked(rng, n, layers=3, p3=0.10, variant=variant)
    return Circuit("cfg4", n, gates, max_terms=max_terms, min_mass=min_mass,
                   truncate_every_gate=True, secret=s, notes={"variant": variant})


def config5(n: int = 56, num_gates: int = 4000, seed: int = 4, max_terms: int = 1 << 28,
            min_mass: float = 1.0 - 1e-4, h_subset: int = 30) -> Circuit:
    """40% diagonal (RZ, T, CZ, CCZ), 30% permutation (CNOT, Toffoli, 4-qubit
    Toffoli), 20% H on a fixed random subset of `h_subset` qubits, 8% Haar SU(4),
    2% Haar 8x8 on random triples  [R17]."""
    rng = np.random.default_rng(seed)
    pool = np.sort(rng.choice(n, size=min(h_subset, n), replace=False))
    kinds = ["diag", "perm", "h", "su4", "u8"]
    probs = [0.40, 0.30, 0.20, 0.08, 0.02]
    gates: List[Gate] = []
    for _ in range(num_gates):
        k = kinds[int(rng.choice(len(kinds), p=probs))]
        if k == "diag":
            sub = int(rng.integers(0, 4))
            if sub == 0:
                q = _pick(rng, n, 1)
                gates.append(G("rz", q, mat_rz(float(rng.uniform(0, 2 * math.pi))), "diag"))
            elif sub == 1:
                gates.append(G("t", _pick(rng, n, 1), mat_t(), "diag"))
            elif sub == 2:
                gates.append(G("cz", _pick(rng, n, 2), mat_diag_minus_last(2), "diag"))
            else:
                gates.append(G("ccz", _pick(rng, n, 3), mat_diag_minus_last(3), "diag"))
        elif k == "perm":
            m = 2 + int(rng.integers(0, 3))
            gates.append(G({2: "cx", 3: "ccx", 4: "c3x"}[m], _pick(rng, n, m), mat_mcx(m), "perm"))
        elif k == "h":
            gates.append(G("h", _pick(rng, n, 1, pool), mat_h(), "gen1"))
        elif k == "su4":
            gates.append(G("su4", _pick(rng, n, 2), haar_unitary(rng, 4, special=True), "gen2"))
        else:
            gates.append(G("u8", _pick(rng, n, 3), haar_unitary(rng, 8), "gen3"))
    return Circuit("cfg5", n, gates, max_terms=max_terms, min_mass=min_mass,
                   truncate_every_gate=True, notes={"h_pool": [int(q) for q in pool]})


def is_diagonal(U: np.ndarray) -> bool:
    U = np.asarray(U)
    return not np.any(U[~np.eye(U.shape[0], dtype=bool)] != 0)


def ring_layers(rng, n: int, layers: int) -> List[Gate]:
    """u3 + cz blocks on a ring, the SHAPE of the paper's workload ("layers of arbitrary
    single-qubit rotations (u3), interleaved with controlled-Z (cz) entangling gates between neighboring qubits",
    with a wrap-around coupling that closes the ring).  A block on (a, b) is u3(t, 0, -pi/2) on a, u3(t', 0, pi/2)
    on b, cz a,b with t, t' ~ U[0, pi) drawn from the seed (the hackathon file's own angles are not available and
    not reconstructed).  Even layers pair (0,1),(2,3),...; odd layers pair (1,2),...,(n-1,0)  [R21]."""
    out: List[Gate] = []
    for layer in range(layers):
        a0 = layer % 2
        for a in range(a0, n - 1 + a0, 2):
            b = (a + 1) % n
            out.append(G("u3", (a,), mat_u3(float(rng.uniform(0.0, math.pi)), 0.0, -0.5 * math.pi), "gen1"))
            out.append(G("u3", (b,), mat_u3(float(rng.uniform(0.0, math.pi)), 0.0, 0.5 * math.pi), "gen1"))
            out.append(G("cz", (a, b), mat_diag_minus_last(2), "diag"))
    return out


def ring_peaked(n: int = 44, layers: int = 4, seed: int = 5, sigma: float = 0.3, max_terms: int = 1 << 20,
                min_mass: float = 1.0) -> Circuit:
    """Row f-3: a peaked u3 + cz ring circuit of the paper's size (n = 44, 4 layers: 594 instructions; the paper's
    has 580).  R = ring_layers, D = u3(theta_q ~ N(0, sigma^2), 0, 0) on every qubit, then R^dagger (cz, then the
    inverse rotations u3(-t, -lambda, -phi)), then u3(pi, 0, pi) = X where the secret s has a 1: the state starts in
    |0..0> and R^dagger D R is close to the identity, so the output is peaked at s."""
    if n % 2:
        raise ValueError("the ring pairing needs an even n")
    rng = np.random.default_rng(seed)
    R = ring_layers(rng, n, layers)
    D = [G("u3", (q,), mat_u3(float(rng.normal(0.0, sigma)), 0.0, 0.0), "gen1") for q in range(n)]
    s = int(rng.integers(0, 1 << n, dtype=np.uint64))
    X = [G("u3", (q,), mat_u3(math.pi, 0.0, math.pi), "perm") for q in range(n) if (s >> q) & 1]
    return Circuit("ring_peaked", n, R + D + adjoint(R) + X, max_terms=max_terms, min_mass=min_mass,
                   truncate_every_gate=True, secret=s, notes={"layers": layers, "sigma": sigma})


def random_state(rng: np.random.Generator, n: int, count: int, spread: float = 2.0):
    """A synthetic sparse state for kernel-level tests and bench warm starts:
    `count` distinct uniform n-bit keys, amplitudes with log-normal magnitudes
    (sigma = spread) and uniform phases, normalised.  Returns (keys u64, amps c128)."""
    if n < 64:
        hi = 1 << n
        want = min(count, hi)
        if want * 4 >= hi:
            keys = rng.permutation(hi).astype(np.uint64)[:want]
        else:
            keys = np.unique(rng.integers(0, hi, size=int(want * 1.2) + 16, dtype=np.uint64))
            rng.shuffle(keys)
            keys = keys[:want]
    else:
        keys = np.unique(rng.integers(0, np.iinfo(np.uint64).max, size=int(count * 1.1) + 16,
                                      dtype=np.uint64, endpoint=True))
        rng.shuffle(keys)
        keys = keys[:count]
    mag = np.exp(spread * rng.standard_normal(keys.size))
    ph = rng.uniform(0, 2 * math.pi, keys.size)
    amps = (mag * np.exp(1j * ph)).astype(C128)
    amps /= math.sqrt(float(np.sum(amps.real ** 2 + amps.imag ** 2)))
    return np.ascontiguousarray(keys), np.ascontiguousarray(amps)
