"""Helpers for GPU-vs-oracle parity tests (north_star tolerances, BASELINE.json:5)."""
import numpy as np

AMP_TOL = 1e-11        # max |delta a| with truncation off
CUT_REL = 1e-9         # kept sets may differ only for terms this close (relative) to the cutoff p
MASS_TOL = 1e-10       # retained mass agreement


def by_key(keys, amps):
    o = np.argsort(keys, kind="stable")
    return keys[o], amps[o]


def assert_same_state(g, o, tol=AMP_TOL, strict_keys=True):
    """g, o: (keys, amps) tuples.  A key missing on one side counts as amplitude 0."""
    gk, ga = by_key(g[0], g[1])
    ok, oa = by_key(o[0], o[1])
    if strict_keys:
        assert gk.size == ok.size, "term counts differ: gpu %d oracle %d" % (gk.size, ok.size)
        assert np.array_equal(gk, ok), "key sets differ"
        d = np.max(np.abs(ga - oa)) if gk.size else 0.0
        assert d <= tol, "max |da| = %g" % d
        return d
    allk = np.union1d(gk, ok)
    fa = np.zeros(allk.size, dtype=np.complex128)
    fo = np.zeros(allk.size, dtype=np.complex128)
    fa[np.searchsorted(allk, gk)] = ga
    fo[np.searchsorted(allk, ok)] = oa
    d = np.max(np.abs(fa - fo)) if allk.size else 0.0
    assert d <= tol, "max |da| = %g" % d
    return d


def assert_truncation_parity(g, o, p_before_by_key=None):
    """Truncation on: kept sets identical except for terms whose probability lies within
    CUT_REL (relative) of the cutoff probability; amplitudes on common keys within AMP_TOL."""
    gk, ga = by_key(g[0], g[1])
    ok, oa = by_key(o[0], o[1])
    common = np.intersect1d(gk, ok)
    gi = np.searchsorted(gk, common)
    oi = np.searchsorted(ok, common)
    if common.size:
        d = np.max(np.abs(ga[gi] - oa[oi]))
        assert d <= AMP_TOL, "max |da| on common keys = %g" % d
    only_g = np.setdiff1d(gk, ok)
    only_o = np.setdiff1d(ok, gk)
    if only_g.size or only_o.size:
        # the cutoff probability = smallest kept probability (either side)
        pg = np.abs(ga) ** 2
        po = np.abs(oa) ** 2
        pcut = min(pg.min(), po.min())
        for ks, kk, pp in ((only_g, gk, pg), (only_o, ok, po)):
            idx = np.searchsorted(kk, ks)
            assert np.all(np.abs(pp[idx] - pcut) <= CUT_REL * pcut), "kept sets differ away from the cutoff"
    return only_g.size + only_o.size


def step_locked(gpu, make_oracle, gate, max_terms, min_mass, truncate):
    """Run one gate (+ truncation) on the GPU and, from the same pre-gate state, on the oracle."""
    k0, a0, _ = gpu.export()
    orc = make_oracle()
    orc.load(k0, a0)
    gpu.apply_gate(gate.qubits, gate.U)
    orc.apply_gate(gate.qubits, gate.U)
    gk, ga, _ = gpu.export()
    ok_, oa, _ = orc.export()
    assert_same_state((gk, ga), (ok_, oa))
    if truncate:
        kg = gpu.truncate(max_terms, min_mass)
        ko = orc.truncate(max_terms, min_mass)
        assert abs(kg - ko) <= MASS_TOL, "kept fraction gpu %r oracle %r" % (kg, ko)
        gk, ga, gp = gpu.export()
        ok_, oa, op = orc.export()
        assert_truncation_parity((gk, ga), (ok_, oa))
        if gk.size and ok_.size and (gp.size < 2 or gp[0] > gp[1] * (1 + 1e-9)):
            assert int(gk[0]) == int(ok_[0]), "top bit string differs"
        return kg
    return 1.0
