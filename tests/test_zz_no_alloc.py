"""sv_norm_static (include/sparse_sv_static.h): the entry point that allocates nothing -- its scratch is a static
device array inside the library -- against the existing path (sv_load_device + sv_norm, whose partial sums live in the
handle's arena), on two calls in a row that share the array.

Collected last on purpose (the suite runs with `pytest -x`): nothing here depends on the tests before it, and it
passes alone in a fresh process as well."""
import ctypes
import os
import re

import numpy as np
import pytest

from util_parity import MASS_TOL

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "sparse_sv_static.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sv_[a-z0-9_]+)\s*\(", src)))


def test_static_header_symbols_are_exported_and_bound():
    from paper_2607_07816_b200 import build
    lib = ctypes.CDLL(build.build())
    d = _declared()
    assert "sv_norm_static" in d
    for name in d:
        assert hasattr(lib, name), name
    from paper_2607_07816_b200 import static_norm
    assert sorted(static_norm.STATIC_EXPORTS) == d
    hdr = open(os.path.join(ROOT, "include", "sparse_sv_static.h")).read()
    assert "#define SV_NORM_STATIC_SCRATCH_BYTES %d" % static_norm.SCRATCH_BYTES in hdr
    assert static_norm.MAX_TERMS == 1 << 32 and "(1ull << 32)" in hdr


def _terms(torch, n, seed, nq=40):
    """n distinct ascending keys and nonzero amplitudes with a peaked profile (a few heavy terms, a long tail)."""
    g = torch.Generator(device="cuda").manual_seed(seed)
    step = torch.randint(1, 1 << 12, (n,), generator=g, device="cuda", dtype=torch.int64)
    keys = torch.cumsum(step, 0)
    assert n == 0 or int(keys[-1]) < (1 << nq)
    re_ = torch.randn(n, generator=g, device="cuda", dtype=torch.float64)
    im_ = torch.randn(n, generator=g, device="cuda", dtype=torch.float64)
    scale = torch.exp(-8.0 * torch.rand(n, generator=g, device="cuda", dtype=torch.float64))
    amps = torch.complex(re_ * scale, im_ * scale)
    amps = torch.where(amps == 0, torch.full_like(amps, 1e-3), amps).contiguous()
    return keys.contiguous(), amps


def _existing_path(engine, keys, amps, nq=40):
    n = int(keys.numel())
    sv = engine.SparseSV(nq, max(n, 1024))
    sv.load_device(keys, amps)
    m = sv.norm()
    sv.close()
    return m


@pytest.mark.gpu
def test_static_norm_matches_sv_norm_on_two_calls_in_a_row():
    import torch
    from paper_2607_07816_b200 import engine, static_norm
    # first call: more than 1024 * 2048 terms, so every one of the 1024 partial slots is written; second call: 3 blocks
    # and a ragged tail, so a stale partial of the first call that leaked into the sum would show at once
    sizes = [(3 << 20) + 777, 2 * 2048 + 5]
    data = [_terms(torch, n, 1234 + i) for i, n in enumerate(sizes)]
    want = [_existing_path(engine, k, a) for k, a in data]
    outs = [torch.full((1,), -1.0, dtype=torch.float64, device="cuda") for _ in sizes]
    static_norm.norm_static_init()
    warm = torch.zeros(1, dtype=torch.float64, device="cuda")
    static_norm.norm_static(data[1][1], warm)          # the first launch of a kernel may load its module
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for (k, a), o in zip(data, outs):                   # two calls in a row, same stream, no sync in between
        static_norm.norm_static(a, o)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    assert free1 == free0, "the static entry point changed the device's free memory"
    for (k, a), o, w in zip(data, outs, want):
        got = float(o.item())
        ref = float((a.real * a.real + a.imag * a.imag).sum().item())
        assert abs(got - w) <= MASS_TOL * w, (got, w)
        assert abs(got - ref) <= MASS_TOL * ref, (got, ref)
        assert got == w, "same grid and order of additions as sv_norm: the bits must agree"
    # and once more the other way round (small, then large) with the array holding the large call's partials
    outs2 = [torch.full((1,), -1.0, dtype=torch.float64, device="cuda") for _ in sizes]
    for i in (1, 0):
        static_norm.norm_static(data[i][1], outs2[i])
    torch.cuda.synchronize()
    for i in (0, 1):
        assert float(outs2[i].item()) == float(outs[i].item())


@pytest.mark.gpu
def test_static_norm_edges_and_rejections():
    import torch
    from paper_2607_07816_b200 import engine, static_norm
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    empty = torch.empty(0, dtype=torch.complex128, device="cuda")
    static_norm.norm_static(empty, out)
    torch.cuda.synchronize()
    assert float(out.item()) == 0.0
    one = torch.tensor([0.6 - 0.8j], dtype=torch.complex128, device="cuda")
    static_norm.norm_static(one, out, stream=torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert float(out.item()) == 0.6 * 0.6 + 0.8 * 0.8
    # beyond the stated maximum: a clear error, nothing enqueued, the output untouched
    out.fill_(7.0)
    torch.cuda.synchronize()
    with pytest.raises(engine.SvError) as e:
        static_norm.norm_static_raw(one.data_ptr(), static_norm.MAX_TERMS + 1, out.data_ptr(), 0)
    assert e.value.code == engine.SV_ERR_INVALID_ARG and "SV_NORM_STATIC_MAX_TERMS" in str(e.value)
    host = np.zeros(4, dtype=np.complex128)
    with pytest.raises(engine.SvError) as e:
        static_norm.norm_static_raw(host.ctypes.data, 4, out.data_ptr(), 0)
    assert e.value.code == engine.SV_ERR_INVALID_ARG and "host" in str(e.value)
    with pytest.raises(engine.SvError):
        static_norm.norm_static_raw(one.data_ptr(), 1, 0, 0)
    with pytest.raises(engine.SvError):
        static_norm.norm_static_raw(one.data_ptr() + 8, 1, out.data_ptr(), 0)
    torch.cuda.synchronize()
    assert float(out.item()) == 7.0
