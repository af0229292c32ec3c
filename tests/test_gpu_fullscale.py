"""GPU checks at BASELINE.json's full sizes, where the oracle cannot run the whole state: structural
invariants, norm preservation, and SAMPLED outputs recomputed one by one on the host from the
downloaded pre-gate state with the oracle's arithmetic (D1)."""
import numpy as np
import pytest

from paper_2607_07816_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _recompute(keys_sorted, amps_sorted, qubits, U, out_keys):
    """out amplitude of each key in out_keys: sum over columns c (ascending) of U[r, c] * a[base | scatter(c)],
    absent members skipped, every product and sum rounded separately (numpy scalar float64 arithmetic)."""
    m = len(qubits)
    mask = 0
    for q in qubits:
        mask |= 1 << q
    res = []
    for k in out_keys:
        k = int(k)
        base = k & ~mask
        r = sum(((k >> q) & 1) << j for j, q in enumerate(qubits))
        sr, si = np.float64(0.0), np.float64(0.0)
        for c in range(1 << m):
            kc = base
            for j, q in enumerate(qubits):
                if (c >> j) & 1:
                    kc |= 1 << q
            i = int(np.searchsorted(keys_sorted, np.uint64(kc)))
            if i < keys_sorted.size and int(keys_sorted[i]) == kc:
                a = amps_sorted[i]
                ur, ui = np.float64(U[r, c].real), np.float64(U[r, c].imag)
                ar, ai = np.float64(a.real), np.float64(a.imag)
                sr = sr + (ur * ar - ui * ai)
                si = si + (ur * ai + ui * ar)
        res.append(complex(sr, si))
    return np.array(res)


@pytest.mark.parametrize("log2n", [25])
def test_gates_at_scale_sampled_recompute(log2n):
    import torch
    from paper_2607_07816_b200 import engine
    n, nq = 1 << log2n, 52
    g = torch.Generator(device="cuda"); g.manual_seed(7)
    keys = torch.randint(0, 1 << nq, (int(n * 1.01),), device="cuda", dtype=torch.int64, generator=g).unique()[:n].contiguous()
    n = int(keys.numel())
    # make partners common: half of the keys get their qubit-40 partner stored as well
    keys = torch.cat([keys[: n // 2], keys[: n // 2] ^ (1 << 40)]).unique().contiguous()
    n = int(keys.numel())
    amps = torch.randn(n, 2, device="cuda", dtype=torch.float64, generator=g).view(torch.complex128).reshape(n).contiguous()
    amps /= amps.abs().pow(2).sum().sqrt()
    sv = engine.SparseSV(nq, 4 * n + 1024)
    rng = np.random.default_rng(3)
    gates = [([40], W.mat_h()), ([11, 40], W.mat_mcx(2)), ([3, 40, 17], W.mat_mcx(3)), ([40], W.mat_rz(0.37)),
             ([40, 9], W.haar_unitary(rng, 4, special=True)), ([45], W.haar_unitary(rng, 2))]
    for qubits, U in gates:
        sv.load_device(keys, amps)
        k0, a0, _ = sv.export()
        o = np.argsort(k0)
        k0, a0 = k0[o], a0[o]
        sv.apply_gate(qubits, U)
        assert sv.check_invariants()
        assert abs(sv.norm() - 1.0) <= 1e-12
        k1, a1, _ = sv.export()
        pick = rng.choice(k1.size, size=300, replace=False)
        want = _recompute(k0, a0, qubits, U, k1[pick])
        assert np.max(np.abs(want - a1[pick])) <= 1e-13, "sampled outputs differ from the definition"
        # every pre-gate term must have at least one image: spot-check that images of sampled inputs exist
        o1 = np.sort(k1)
        mask = 0
        for q in qubits:
            mask |= 1 << q
        pin = rng.choice(k0.size, size=300, replace=False)
        got = 0
        for k in k0[pin]:
            base = int(k) & ~mask
            lo = int(np.searchsorted(o1, np.uint64(base)))
            # some key of the tuple (base | pattern) must be present in the output
            hit = False
            for c in range(1 << len(qubits)):
                kc = base
                for j, q in enumerate(qubits):
                    if (c >> j) & 1:
                        kc |= 1 << q
                i = int(np.searchsorted(o1, np.uint64(kc)))
                hit = hit or (i < o1.size and int(o1[i]) == kc)
            got += hit
        assert got == 300


def test_config2_full_size_step_locked():
    """BASELINE.json configs[1] at its OWN size: n = 24, all 400 gates, hard cap K = 2^20 after every gate, default
    engine options.  Every 4th gate (and every gate while the state is small) is step-locked against the oracle from
    the GPU's pre-gate state: identical state after the gate, kept fraction to 1e-10, kept sets identical except
    within 1e-9 of the cutoff."""
    import sys, os
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    from util_parity import step_locked
    from oracle.sparse import SparseOracle
    from paper_2607_07816_b200 import engine
    c = W.config2()
    assert c.n == 24 and len(c.gates) == 400 and c.max_terms == 1 << 20
    sv = engine.SparseSV(c.n, 1 << 22)
    locked = 0
    for i, g in enumerate(c.gates):
        if i % 4 == 0 or sv.num_terms() < (1 << 14):
            step_locked(sv, lambda: SparseOracle(c.n), g, c.max_terms, c.min_mass, True)
            locked += 1
        else:
            sv.apply_gate_truncate(g.qubits, g.U, c.max_terms, c.min_mass)
        assert sv.num_terms() <= c.max_terms
    assert locked >= 100
    assert sv.check_invariants()
    assert abs(sv.norm() - 1.0) <= 1e-11


def test_config3_full_size_peak():
    """BASELINE.json configs[2] at its full size: n = 26, 2^26 terms from the first H layer on (1.6 GB),
    cap 2^26 never binding.  The most probable bit string must be the secret; the norm must stay 1."""
    from paper_2607_07816_b200 import engine
    c = W.config3()
    sv = engine.SparseSV(c.n, (1 << c.n) + 1024)
    for g in c.gates:
        sv.apply_gate(g.qubits, g.U)
        sv.truncate(c.max_terms, 1.0)
    assert sv.num_terms() <= 1 << c.n
    k, a, p = sv.top(4)
    assert int(k[0]) == c.secret, "top bit string is not the secret"
    assert p[0] > 0.2 and p[0] > 10 * p[1]
    assert abs(sv.norm() - 1.0) <= 1e-10
    assert sv.check_invariants()


def test_config5_at_2e24_properties():
    """BASELINE.json configs[4] (n = 56 mix, mass 1 - 1e-4) at K = 2^24: per-gate structural properties the
    method fixes at any size -- kept count <= K, kept fraction >= the threshold when the cap does not bind,
    norm 1 after every cut, strictly ascending unique keys."""
    from paper_2607_07816_b200 import engine
    K = 1 << 24
    c = W.config5(num_gates=170, max_terms=K)
    sv = engine.SparseSV(c.n, 8 * K)
    for i, g in enumerate(c.gates):
        sv.apply_gate(g.qubits, g.U)
        n_pre = sv.num_terms()
        kept = sv.truncate(c.max_terms, c.min_mass)
        n_post = sv.num_terms()
        assert n_post <= K
        if n_pre <= K:
            assert kept >= c.min_mass - 1e-12                  # only the mass rule cut: it keeps at least the threshold
        if kept < c.min_mass - 1e-12:
            assert n_pre > K and n_post == K                   # less than the threshold kept: then the cap bound, and binds exactly
        if n_post < n_pre:
            assert kept < 1.0                                   # something was dropped, and every dropped term is nonzero
        else:
            assert kept == 1.0                                  # nothing dropped: untouched (R7)
        assert 0.0 < kept <= 1.0
        if i % 10 == 9:
            assert abs(sv.norm() - 1.0) <= 1e-11
    assert sv.check_invariants()
    assert sv.stats()["fallbacks"] <= 2, "the sampled band missed the cut on config 5"


def test_config5_fused_call_equals_two_calls_at_2e22():
    """The launch configuration bench.py times (sv_apply_gate_truncate, default sampling threshold 2^21) against
    the two separate calls on a twin engine, config 5 at K = 2^22: identical term counts after every gate,
    identical kept fractions to 1e-13, and identical states (keys bitwise, amplitudes to 1e-13 relative)
    at check points; the fused path must have used its output floor and must not have needed a re-run."""
    from paper_2607_07816_b200 import engine
    K = 1 << 22
    c = W.config5(num_gates=150, max_terms=K)
    a, b = engine.SparseSV(c.n, 8 * K), engine.SparseSV(c.n, 8 * K)
    used, peak_a = 0, 0
    for i, g in enumerate(c.gates):
        ka = a.apply_gate_truncate(g.qubits, g.U, c.max_terms, c.min_mass)
        st = a.stats()
        b.apply_gate(g.qubits, g.U)
        n_mid = b.num_terms()
        kb = b.truncate(c.max_terms, c.min_mass)
        assert st["n_mid"] == n_mid, (i, g.name)
        assert a.num_terms() == b.num_terms(), (i, g.name)
        assert abs(ka - kb) <= 1e-13, (i, g.name, ka, kb)
        used += 1 if st["pre_dropped"] else 0
        if st["n_in"] >= (1 << 21):                      # (smaller states do not sample: they take the two calls)
            peak_a = max(peak_a, n_mid - st["pre_dropped"])
        if i in (110, 149):
            ea, eb = a.export(), b.export()
            assert np.array_equal(ea[0], eb[0])
            assert np.allclose(ea[1], eb[1], rtol=1e-13, atol=0)
    assert used >= 10, used
    assert a.stats()["fallbacks"] <= b.stats()["fallbacks"]
    assert peak_a <= int(1.2 * K), "the fused path stored %d outputs at its peak (K = %d)" % (peak_a, K)
    assert a.check_invariants()


def test_fused_floor_on_dense_tuples():
    """A state that is dense in the gate's qubits (every tuple has all its members): the pre-sample accepts one
    member per tuple, so its estimate of the output distribution must stay unbiased -- the floor is used and
    holds (no re-run), for one-bit and two-bit gates, with the moved bit far from and at the LSB."""
    from paper_2607_07816_b200 import engine
    n = 22
    rng = np.random.default_rng(8)
    N = 1 << 19
    keys = np.arange(N, dtype=np.uint64)                       # dense in qubits 0..18
    amps = (rng.normal(size=N) + 1j * rng.normal(size=N)) * np.exp(rng.normal(size=N))
    amps /= np.sqrt(np.sum(np.abs(amps) ** 2))
    for qubits in ([0], [18], [7], [0, 1], [18, 3], [9, 20]):
        a, b = engine.SparseSV(n, 4 * N), engine.SparseSV(n, 4 * N)
        for sv in (a, b):
            sv.set_option(engine.OPT_SAMPLE_MIN_TERMS, 512)
            sv.load(keys, amps)
        U = W.haar_unitary(rng, 1 << len(qubits))
        K = N // 2
        ka = a.apply_gate_truncate(qubits, U, K, 1.0)
        st = a.stats()
        b.apply_gate(qubits, U); kb = b.truncate(K, 1.0)
        assert st["pre_dropped"] > 0 and st["fallbacks"] == 0, (qubits, st)
        assert st["n_mid"] - st["pre_dropped"] <= int(1.15 * K), (qubits, st)
        assert abs(ka - kb) <= 1e-13
        ea, eb = a.export(), b.export()
        assert np.array_equal(ea[0], eb[0]) and np.array_equal(ea[1], eb[1])
        a.close(); b.close()


def _tuple_outputs(members, qubits, U):
    """All 2^m outputs of one tuple by the definition (D1): members = {local column c: amplitude}
    of the stored terms, absent ones skipped, columns ascending, every product and sum rounded separately."""
    d = 1 << len(qubits)
    out = []
    for r in range(d):
        sr, si = np.float64(0.0), np.float64(0.0)
        for c in range(d):
            if c in members:
                a = members[c]
                ur, ui = np.float64(U[r, c].real), np.float64(U[r, c].imag)
                ar, ai = np.float64(a.real), np.float64(a.imag)
                sr = sr + (ur * ar - ui * ai)
                si = si + (ur * ai + ui * ar)
        out.append(complex(sr, si))
    return out


def test_fused_call_at_2e28_sampled_recompute():
    """The launch configuration bench.py times -- config 5, K = 2^28, every gate through sv_apply_gate_truncate --
    checked against the definition on SAMPLED tuples, for the first gate of every class after the ramp (diagonal,
    permutation, H, SU(4), 8x8) and for a Haar 16x16 gate whose candidate outputs exceed 2^31.  The pre- and post-gate
    states are exported through the ABI, sorted by key on the device (torch), ~10^3 random pre-gate terms are picked,
    the outputs of their tuples are recomputed on the host with the test-local definition, and every output must be
    (a) kept, with amplitude = recomputed * scale, when its probability is above the cut by more than 1e-9 relative,
    (b) absent when it is below the cut by more than 1e-9.  kept_fraction must equal kept mass / mass before
    (PAPER.md:94-96: largest magnitudes kept, fewest terms; :96 renormalised)."""
    import torch
    from paper_2607_07816_b200 import engine
    K = 1 << 28
    free_b, _ = torch.cuda.mem_get_info()
    if engine.lib.sv_arena_bytes(8 * K) + (48 << 30) > free_b:
        pytest.skip("needs ~150 GB of device memory")
    c = W.config5(max_terms=K)
    sv = engine.SparseSV(c.n, 8 * K)
    rng = np.random.default_rng(99)
    gi = 0
    while sv.num_terms() < 0.9 * K:
        g = c.gates[gi]; gi += 1
        sv.apply_gate_truncate(g.qubits, g.U, c.max_terms, c.min_mass)

    def sorted_dev(keys, amps):
        kt = torch.from_numpy(keys.view(np.int64)).cuda()
        at = torch.from_numpy(amps).cuda()
        # order as unsigned: flip the sign bit, sort as int64
        o = torch.argsort(kt ^ (-(1 << 63)))
        return (kt[o] ^ (-(1 << 63))).contiguous(), kt[o].contiguous(), at[o].contiguous()

    def lookup(sk_flipped, amps_sorted, want_keys_u64):
        w = torch.from_numpy(np.asarray(want_keys_u64, dtype=np.uint64).view(np.int64)).cuda() ^ (-(1 << 63))
        i = torch.searchsorted(sk_flipped, w).clamp(max=sk_flipped.numel() - 1)
        hit = sk_flipped[i] == w
        return hit.cpu().numpy(), amps_sorted[i].cpu().numpy()

    def check_gate(qubits, U, name):
        m = len(qubits)
        mask = 0
        for q in qubits:
            mask |= 1 << q
        mass0 = sv.norm()
        k0, a0, _ = sv.export()
        n_in = k0.size
        pre_f, _, pre_a = sorted_dev(k0, a0)
        pick = k0[rng.choice(n_in, size=1000, replace=False)]
        del k0, a0
        kept = sv.apply_gate_truncate(list(qubits), U, c.max_terms, c.min_mass)
        st = sv.stats()
        assert st["fallbacks"] == fallbacks0[0], (name, st)
        k1, a1, p1 = sv.export()
        n_out = k1.size
        assert n_out <= K and n_out == st["n_out"]
        p_cut_scaled = float(p1[-1])                       # smallest kept probability (after renormalisation)
        assert abs(float(np.sum(p1)) - 1.0) <= 1e-9
        post_f, _, post_a = sorted_dev(k1, a1)
        del k1, a1, p1
        # tuples of the sampled inputs
        bases = np.unique(pick & np.uint64(~mask & ((1 << 64) - 1)))
        cols = []
        for cc in range(1 << m):
            off = 0
            for j, q in enumerate(qubits):
                if (cc >> j) & 1:
                    off |= 1 << q
            cols.append(np.uint64(off))
        want = np.concatenate([bases | cc for cc in cols])
        hit, amp = lookup(pre_f, pre_a, want)
        hit = hit.reshape(1 << m, -1); amp = amp.reshape(1 << m, -1)
        outs_key, outs_val = [], []
        for t in range(bases.size):
            members = {cc: complex(amp[cc, t]) for cc in range(1 << m) if hit[cc, t]}
            assert members
            vals = _tuple_outputs(members, qubits, U)
            for r, v in enumerate(vals):
                if v != 0:
                    outs_key.append(int(bases[t]) | int(cols[r])); outs_val.append(v)
        outs_key = np.array(outs_key, dtype=np.uint64); outs_val = np.array(outs_val)
        ohit, oamp = lookup(post_f, post_a, outs_key)
        # scale: from the kept outputs themselves (one number for the whole state)
        ratios = np.abs(oamp[ohit]) / np.abs(outs_val[ohit])
        scale = float(np.median(ratios))
        assert ohit.sum() >= 100, (name, int(ohit.sum()))
        assert np.max(np.abs(oamp[ohit] - outs_val[ohit] * scale)) <= 1e-13 * max(1.0, scale), name
        p_out = (outs_val.real ** 2 + outs_val.imag ** 2) * scale * scale
        if n_out < st["n_mid"]:                            # something was dropped: the cut separates kept from dropped
            assert np.all(p_out[~ohit] <= p_cut_scaled * (1 + 1e-9)), name
            assert np.all(p_out[ohit] >= p_cut_scaled * (1 - 1e-9)), name
            assert abs(kept - (1.0 / (scale * scale)) / mass0) <= 1e-10, (name, kept, scale, mass0)
        else:
            assert ohit.all() and kept == 1.0
        assert sv.check_invariants()
        return st

    fallbacks0 = [sv.stats()["fallbacks"]]
    seen = {}
    while len(seen) < 5 and gi < len(c.gates):
        g = c.gates[gi]; gi += 1
        if g.klass in seen or sv.num_terms() < 0.9 * K:
            sv.apply_gate_truncate(g.qubits, g.U, c.max_terms, c.min_mass)
            fallbacks0[0] = sv.stats()["fallbacks"]
            continue
        seen[g.klass] = check_gate(g.qubits, g.U, g.name)
    assert set(seen) == {"diag", "perm", "gen1", "gen2", "gen3"}, seen.keys()
    assert seen["gen3"]["pre_dropped"] > 0 and seen["gen2"]["pre_dropped"] > 0
    # a 4-qubit Haar gate: 16 x N_in candidate outputs (> 2^31), of which the pass may store about K
    while sv.num_terms() < 0.9 * K:
        g = c.gates[gi]; gi += 1
        sv.apply_gate_truncate(g.qubits, g.U, c.max_terms, c.min_mass)
    fallbacks0[0] = sv.stats()["fallbacks"]
    st = check_gate((3, 41, 17, 29), W.haar_unitary(rng, 16), "haar16")
    assert st["n_mid"] > (1 << 31), st
