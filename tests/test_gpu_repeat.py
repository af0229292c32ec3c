"""Bit-for-bit repeatability of the hot path (stands in for compute-sanitizer racecheck, which is closed on the pool
this was built on: profiles/r2_sanitizer.md).  The passes coordinate through relaxed-atomic look-back words, parked
shared-memory buffers and spin-waits between persistent blocks; a race there changes an output position, a count or an
amplitude from one run to the next.  The same circuit is therefore run twice on fresh handles (different arenas and
streams, hence different timing) and every kept fraction, term count, key and amplitude bit must repeat."""
import numpy as np
import pytest

from paper_2607_07816_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _run(engine, c, cap, sample_min, torch_arena, fused, checkpoints):
    sv = engine.SparseSV(c.n, cap, torch_arena=torch_arena)
    if sample_min is not None:
        sv.set_option(engine.OPT_SAMPLE_MIN_TERMS, sample_min)
    kept, counts, snaps = [], [], {}
    for i, g in enumerate(c.gates):
        if fused:
            kept.append(sv.apply_gate_truncate(g.qubits, g.U, c.max_terms, c.min_mass))
        else:
            sv.apply_gate(g.qubits, g.U)
            kept.append(sv.truncate(c.max_terms, c.min_mass))
        counts.append(sv.num_terms())
        if i in checkpoints:
            snaps[i] = sv.export()[:2]
    snaps["end"] = sv.export()[:2]
    assert sv.check_invariants()
    sv.close()
    return kept, counts, snaps


@pytest.mark.parametrize("fused", [True, False])
@pytest.mark.parametrize("klog,gates,sample_min", [(13, 260, 512), (20, 170, None)])
def test_same_bits_every_run(fused, klog, gates, sample_min):
    from paper_2607_07816_b200 import engine
    c = W.config5(num_gates=gates, max_terms=1 << klog)
    cps = {gates // 3, (2 * gates) // 3}
    a = _run(engine, c, 8 << klog, sample_min, True, fused, cps)
    b = _run(engine, c, 8 << klog, sample_min, False, fused, cps)
    assert a[0] == b[0], "kept fractions differ between two runs"
    assert a[1] == b[1], "term counts differ between two runs"
    for k in a[2]:
        assert np.array_equal(a[2][k][0], b[2][k][0]), "keys differ at %r" % (k,)
        assert np.array_equal(a[2][k][1], b[2][k][1]), "amplitudes differ at %r" % (k,)


def test_dense_states_same_bits_every_run():
    """Configs[3] shape (dense tuples, SU(4) and 8x8 gates, cap + mass cut every gate) at n = 18: the multi-bit passes
    with full tuples, staging overflow and parking, twice."""
    from paper_2607_07816_b200 import engine
    c = W.config4(n=18, max_terms=1 << 15, variant="hboth")
    a = _run(engine, c, 1 << 19, 512, True, True, set())
    b = _run(engine, c, 1 << 19, 512, False, True, set())
    assert a[0] == b[0] and a[1] == b[1]
    assert np.array_equal(a[2]["end"][0], b[2]["end"][0]) and np.array_equal(a[2]["end"][1], b[2]["end"][1])
