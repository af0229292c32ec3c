"""Pins for the CPU oracle's truncation (orc_truncate / orc_top / orc_norm).

PAPER.md:94-96 and :124 define the procedure; the pins are closed forms whose answer is
known without running it, plus a numpy lexsort brute force (library routine).
"""
import math

import numpy as np
import pytest

from oracle.sparse import SparseOracle
from paper_2607_07816_b200 import workloads as W


def _state(keys, amps, n=40):
    o = SparseOracle(n)
    o.load(np.asarray(keys, dtype=np.uint64), np.asarray(amps, dtype=np.complex128))
    return o


def test_noop_is_bitwise():
    rng = np.random.default_rng(0)
    keys, amps = W.random_state(rng, 30, 500)
    o = _state(keys, amps)
    before = o.as_dict()
    assert o.truncate(0, 1.0) == 1.0
    assert o.truncate(500, 1.0) == 1.0
    assert o.truncate(10 ** 9, 2.0) == 1.0
    assert o.as_dict() == before


def test_top1_keeps_phase():
    keys = [5, 9, 77]
    amps = [0.1 + 0.2j, -0.6 + 0.3j, 0.2 - 0.1j]
    o = _state(keys, amps)
    o.truncate(1, 1.0)
    k, a, p = o.export()
    assert list(k) == [9]
    z = complex(-0.6, 0.3)
    assert abs(a[0] - z / abs(z)) <= 2e-16
    assert abs(p[0] - 1.0) <= 4e-16


def test_flat_state_keeps_lowest_keys():
    """All p equal: ties are broken by key ascending (reading R4)."""
    rng = np.random.default_rng(1)
    keys = rng.permutation(1 << 12).astype(np.uint64)[:1000] * np.uint64(1 << 20)
    amps = np.full(1000, 0.25 + 0.0j)
    o = _state(keys, amps, n=40)
    kept = o.truncate(100, 1.0)
    k, a, _ = o.export()
    assert sorted(int(x) for x in k) == sorted(int(x) for x in np.sort(keys)[:100])
    assert abs(kept - 0.1) <= 1e-15
    assert np.allclose(a, 0.1, atol=1e-15)  # 100 equal terms, norm 1


def test_geometric_mass_closed_form():
    """p_i = 2^-(i+1), i = 0..39 (S = 1 - 2^-40).  Prefix mass after j terms is 1 - 2^-j,
    so the smallest prefix holding a fraction f = 1 - 2^-t - eps of S has j = t terms."""
    n_terms = 40
    p = np.array([2.0 ** -(i + 1) for i in range(n_terms)])
    amps = np.sqrt(p).astype(np.complex128)
    keys = np.arange(n_terms, dtype=np.uint64)[::-1].copy()  # key order opposite to p order
    for t in (1, 3, 7, 20):
        o = _state(keys, amps)
        f = (1.0 - 2.0 ** -t) * (1 - 1e-12)
        kept = o.truncate(0, f)
        assert o.num_terms() == t
        S = 1.0 - 2.0 ** -n_terms
        assert abs(kept - (1.0 - 2.0 ** -t) / S) <= 1e-15
        assert abs(o.norm() - 1.0) <= 4e-16
    # just above a prefix mass -> one more term
    o = _state(keys, amps)
    o.truncate(0, (1.0 - 2.0 ** -5) * (1 + 1e-9))
    assert o.num_terms() == 6


def test_mass_then_topk():
    """p-mass first, then top-k if still above the limit."""
    p = np.array([2.0 ** -(i + 1) for i in range(30)])
    amps = np.sqrt(p).astype(np.complex128)
    keys = np.arange(30, dtype=np.uint64)
    o = _state(keys, amps)
    o.truncate(4, 1.0 - 2.0 ** -10 - 1e-9)   # mass alone keeps 10 -> cap at 4
    assert o.num_terms() == 4
    o = _state(keys, amps)
    o.truncate(20, 1.0 - 2.0 ** -10 - 1e-9)  # cap not binding
    assert o.num_terms() == 10


def test_at_least_one_term():
    o = _state([1, 2], [0.8, 0.6])
    o.truncate(0, 1e-9)
    assert o.num_terms() == 1


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_brute_force_lexsort(seed):
    rng = np.random.default_rng(seed)
    keys, amps = W.random_state(rng, 36, 5000, spread=1.0 + seed)
    if seed == 3:  # force many exact ties
        amps = (np.round(amps * 64) / 64).astype(np.complex128)
        amps[amps == 0] = 1 / 64
    K = [0, 1234, 4000, 17][seed]
    f = [0.97, 1.0, 0.5, 0.9999][seed]
    o = _state(keys, amps)
    kept = o.truncate(K, f)
    # brute force with library sort
    p = amps.real * amps.real + amps.imag * amps.imag
    order = np.lexsort((keys, -p))
    ps = p[order]
    S = float(np.sum(ps))
    cum = np.cumsum(ps)
    j = int(np.searchsorted(cum, f * S, side="left")) + 1 if f < 1.0 else keys.size
    if K:
        j = min(j, K)
    j = max(1, min(j, keys.size))
    k, a, pk = o.export()
    assert k.size == j
    assert set(int(x) for x in k) == set(int(x) for x in keys[order[:j]])
    keptm = float(np.sum(ps[:j]))
    assert abs(kept - keptm / S) <= 1e-13
    exp = dict(zip((int(x) for x in keys[order[:j]]), amps[order[:j]] / math.sqrt(keptm)))
    for kk, aa in zip(k, a):
        assert abs(exp[int(kk)] - aa) <= 1e-13
    assert abs(o.norm() - 1.0) <= 1e-13
    # kept-min >= dropped-max
    if j < keys.size:
        assert ps[j - 1] >= ps[j]


def test_top_order_and_norm():
    rng = np.random.default_rng(9)
    keys, amps = W.random_state(rng, 50, 3000)
    o = _state(keys, amps, n=50)
    k, a, p = o.top(200)
    pp = amps.real ** 2 + amps.imag ** 2
    order = np.lexsort((keys, -pp))[:200]
    assert np.array_equal(k, keys[order])
    assert np.array_equal(a, amps[order])
    assert np.array_equal(p, pp[order])
    assert abs(o.norm() - math.fsum(pp)) <= 1e-14


def test_truncate_invalid():
    o = _state([1], [1.0])
    with pytest.raises(ValueError):
        o.truncate(0, 0.0)
    with pytest.raises(ValueError):
        o.truncate(0, float("nan"))


KNIFE_CASES = [(0.3, 300), (0.2999, 300), (0.3001, 301), (0.299, 299), (0.1, 100), (0.7, 700), (0.5, 500), (0.999, 999),
               (0.9991, 1000), (1e-9, 1)]


def knife_state():
    """1000 terms of amplitude 2^-5 (p = 2^-10 exactly): every prefix sum and S = 1000 * 2^-10 are exact in fp64 in
    any summation order, so the smallest prefix with j * 2^-10 >= fl(f * S) is a closed form ("minimum
    fraction of probability mass to keep"; reading R5 / R22)."""
    rng = np.random.default_rng(12)
    keys = np.sort(rng.choice(1 << 30, size=1000, replace=False).astype(np.uint64))
    amps = np.full(1000, 2.0 ** -5 + 0.0j)
    return keys, amps


@pytest.mark.parametrize("f,want", KNIFE_CASES)
def test_knife_edge_closed_form(f, want):
    """p-mass on a flat state, thresholds at and beside the knife edge j * p == f * S: f = 0.3 keeps exactly 300 of
    1000 equal terms (fl(0.3 * 1000/1024) = 300/1024), the lowest keys first (R4)."""
    keys, amps = knife_state()
    S = 1000 * 2.0 ** -10
    thr = f * S                                   # one rounding, as the procedure states it
    j = next(j for j in range(1, 1001) if j * 2.0 ** -10 >= thr)
    assert j == want, "the closed form itself"
    o = _state(keys, amps)
    kept = o.truncate(0, f)
    k, a, _ = o.export()
    assert k.size == want
    assert np.array_equal(np.sort(k), keys[:want])
    assert kept == want / 1000.0
    scale = 1.0 if want == 1000 else 1.0 / math.sqrt(want * 2.0 ** -10)     # nothing dropped: bitwise no-op (R7)
    assert np.all(a == (2.0 ** -5) * scale)
