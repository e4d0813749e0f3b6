"""qcd_re_dot_static (include/qcd.h): the dot product for callers that cannot allocate -- no context, no cudaMalloc,
its reduction scratch a fixed __device__ array shared by every call.

Collected LAST (the file name sorts after every other test file): the suite runs with `pytest -x`, so a failure here
must not hide another test.  Every test passes alone in a fresh process and after the rest of the suite: the first
one makes its calls before this file creates any context, so alone it is the library's first CUDA work.

The comparison is with the existing path, qcd_re_dot on a context, on the same device buffers, within the tolerance
tests/test_gpu_parity.py uses for that call (1e-14 x |a| |b|); both use one summation order, so they should in fact
agree to the bit, which is asserted as well.
"""
import ctypes
import math

import numpy as np
import pytest

TOL = 1e-14          # x |a| |b| : test_gpu_parity.py::test_re_dot_matches_oracle_and_is_deterministic


def _real(prec):
    import torch
    return torch.float64 if prec == 64 else torch.float32


def _random_half_field(torch, ctx, q, seed):
    """A QCD_SPINOR_EVEN field of the context with Gaussian reals written on the device."""
    f = ctx.field(q.QCD_SPINOR_EVEN)
    g = torch.Generator(device=ctx.device).manual_seed(seed)
    v = f.buf.view(_real(ctx.precision))
    v.copy_(torch.randn(v.numel(), generator=g, device=ctx.device, dtype=v.dtype))
    return f


def _static(q, torch, fa, fb, prec, stream, result):
    """One call of the new entry point; returns the value it wrote."""
    result.fill_(float("nan"))
    q.qcd_re_dot_static(fa.buf.data_ptr(), fb.buf.data_ptr(), fa.nbytes // (prec // 8), prec, stream.cuda_stream, result.data_ptr())
    stream.synchronize()
    assert math.isnan(result[1].item()) and math.isnan(result[2].item())       # one double written, no more
    return result[0].item()


@pytest.mark.gpu
def test_no_alloc_first_cuda_work_of_the_library():
    """Raw torch buffers, no context yet: set-up (cudaGetSymbolAddress) happens inside the first call.  Two calls in a
    row, then the SAME buffers bound to a context and reduced by the existing path."""
    import torch
    import paper_2502_03249_b200 as q
    dims, prec = (8, 4, 6, 10), 64
    n = 3 * 2 * (int(np.prod(dims)) // 2)
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    g = torch.Generator(device=dev).manual_seed(11)
    a = torch.randn(n, generator=g, device=dev, dtype=torch.float64)
    b = torch.randn(n, generator=g, device=dev, dtype=torch.float64)
    result = torch.full((3,), float("nan"), dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream(dev)
    got = []
    for _ in range(2):
        result.fill_(float("nan"))
        q.qcd_re_dot_static(a.data_ptr(), b.data_ptr(), n, prec, stream.cuda_stream, result.data_ptr())
        stream.synchronize()
        got.append(result[0].item())
        assert math.isnan(result[1].item())
    scale = float(torch.linalg.vector_norm(a) * torch.linalg.vector_norm(b))
    assert abs(got[0] - float(torch.dot(a, b))) <= TOL * scale
    ctx = q.Context(dims, prec)
    fa = ctx.field(q.QCD_SPINOR_EVEN, buf=a.view(torch.uint8))
    fb = ctx.field(q.QCD_SPINOR_EVEN, buf=b.view(torch.uint8))
    ref = ctx.qcd_re_dot(fa, fb)
    for v in got:
        assert abs(v - ref) <= TOL * scale
        assert v == ref
    ctx.close()


@pytest.mark.gpu
@pytest.mark.parametrize("prec", [64, 32])
def test_no_alloc_matches_existing_path_on_calls_in_a_row(prec):
    """Large, small, large: the small call runs over the stale partial sums the large one left in the shared array.
    Each lattice three times in a row, on the default stream and on a side stream; device memory in use does not move."""
    import torch
    import paper_2502_03249_b200 as q
    dev = torch.device("cuda:0")
    side = torch.cuda.Stream(dev)
    for dims, stream in (((16, 16, 16, 16), None), ((8, 4, 6, 10), side), ((4, 4, 4, 4), None), ((16, 16, 16, 16), side)):
        with torch.cuda.stream(stream if stream is not None else torch.cuda.current_stream(dev)):
            ctx = q.Context(dims, prec, stream=stream)
            fa, fb = _random_half_field(torch, ctx, q, 3), _random_half_field(torch, ctx, q, 4)
            result = torch.full((3,), float("nan"), dtype=torch.float64, device=dev)
            ref = ctx.qcd_re_dot(fa, fb)
            scale = math.sqrt(ctx.qcd_re_dot(fa, fa) * ctx.qcd_re_dot(fb, fb))
            assert scale > 0 and math.isfinite(ref)
            aa = ctx.qcd_re_dot(fa, fa)
            free_before = None
            for call in range(3):
                got = _static(q, torch, fa, fb, prec, ctx.stream, result)
                assert abs(got - ref) <= TOL * scale, (dims, call, got, ref)
                assert got == ref, (dims, call)
                if free_before is None:
                    free_before = torch.cuda.mem_get_info(dev)[0]          # after the first call: module and set-up are in
            assert _static(q, torch, fa, fa, prec, ctx.stream, result) == aa                   # a aliasing b
            assert torch.cuda.mem_get_info(dev)[0] == free_before, "device memory in use changed across qcd_re_dot_static calls"
            ctx.close()


@pytest.mark.gpu
def test_no_alloc_maximum_size_and_rejections():
    """n_reals = QCD_RE_DOT_STATIC_MAX_REALS (one 64^4 half-field, 24 576 blocks) is accepted in both precisions; anything
    beyond, and every other bad argument, is refused with a message and without touching the result."""
    import torch
    import paper_2502_03249_b200 as q
    dev = torch.device("cuda:0")
    ctx = q.Context((64, 64, 64, 64), 64)
    fa = _random_half_field(torch, ctx, q, 5)
    assert fa.nbytes // 8 == q.QCD_RE_DOT_STATIC_MAX_REALS
    result = torch.full((3,), float("nan"), dtype=torch.float64, device=dev)
    ref = ctx.qcd_re_dot(fa, fa)
    for _ in range(2):
        got = _static(q, torch, fa, fa, 64, ctx.stream, result)
        assert abs(got - ref) <= TOL * ref and got == ref
    # the same bytes read as floats: MAX_REALS floats = the first half of the buffer (finite values are not guaranteed for
    # reinterpreted doubles, so only the call's acceptance is checked)
    q.qcd_re_dot_static(fa.buf.data_ptr(), fa.buf.data_ptr(), q.QCD_RE_DOT_STATIC_MAX_REALS, 32, ctx.stream.cuda_stream, result.data_ptr())
    ctx.stream.synchronize()
    result.fill_(float("nan"))
    host_raw = np.zeros(16 + 2, dtype=np.float64)
    host = host_raw[(-host_raw.ctypes.data // 8) % 2:][:16]                  # 16-byte aligned HOST memory
    assert host.ctypes.data % 16 == 0
    bad = [
        (dict(n=q.QCD_RE_DOT_STATIC_MAX_REALS + 2), "exceeds QCD_RE_DOT_STATIC_MAX_REALS"),
        (dict(n=2 ** 40), "exceeds QCD_RE_DOT_STATIC_MAX_REALS"),
        (dict(prec=16), "precision"),
        (dict(n=3), "multiple of 16 bytes"),
        (dict(a=fa.buf.data_ptr() + 8), "16-byte aligned"),
        (dict(a=0), "NULL"),
        (dict(res=0), "NULL"),
        (dict(b=host.ctypes.data, n=16), "not device memory"),
        (dict(res=host.ctypes.data, n=16), "not device memory"),
    ]
    for kw, msg in bad:
        with pytest.raises(q.QcdError) as e:
            q.qcd_re_dot_static(kw.get("a", fa.buf.data_ptr()), kw.get("b", fa.buf.data_ptr()), kw.get("n", 1024), kw.get("prec", 64),
                                ctx.stream.cuda_stream, kw.get("res", result.data_ptr()))
        assert e.value.status == q.QCD_EINVAL and msg in str(e.value), (kw, str(e.value))
    ctx.stream.synchronize()
    assert torch.isnan(result).all()
    # empty input: 0.0
    q.qcd_re_dot_static(fa.buf.data_ptr(), fa.buf.data_ptr(), 0, 64, ctx.stream.cuda_stream, result.data_ptr())
    ctx.stream.synchronize()
    assert result[0].item() == 0.0 and math.isnan(result[1].item())
    # the existing path is untouched by all of this
    assert ctx.qcd_re_dot(fa, fa) == ref
    ctx.close()


@pytest.mark.gpu
def test_no_alloc_call_can_be_captured_in_a_cuda_graph():
    """The callers this entry point is for: a stream under capture refuses cudaMalloc, so a capture that succeeds and
    replays to the existing path's value shows the call allocates nothing."""
    import torch
    import paper_2502_03249_b200 as q
    dev = torch.device("cuda:0")
    side = torch.cuda.Stream(dev)
    dims, prec = (8, 4, 6, 10), 64
    with torch.cuda.stream(side):
        ctx = q.Context(dims, prec, stream=side)
        fa, fb = _random_half_field(torch, ctx, q, 8), _random_half_field(torch, ctx, q, 9)
        ref = ctx.qcd_re_dot(fa, fb)
        result = torch.full((3,), float("nan"), dtype=torch.float64, device=dev)
        assert _static(q, torch, fa, fb, prec, side, result) == ref               # set-up is done outside the capture
        result.fill_(float("nan"))
        side.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            q.qcd_re_dot_static(fa.buf.data_ptr(), fb.buf.data_ptr(), fa.nbytes // 8, prec, torch.cuda.current_stream(dev).cuda_stream,
                                result.data_ptr())
        side.synchronize()
        assert math.isnan(result[0].item())                                       # captured, not run
        for _ in range(2):
            graph.replay()
            side.synchronize()
            assert result[0].item() == ref
            result.fill_(float("nan"))
            side.synchronize()
        del graph
        ctx.close()


def test_no_alloc_size_limit_is_checked_before_any_cuda_call():
    """No GPU needed: the limit, NULL and precision checks come before the first CUDA call."""
    from paper_2502_03249_b200 import QCD_EINVAL, QCD_RE_DOT_STATIC_MAX_REALS, build, load_library
    build.build()
    lib = load_library()
    err = ctypes.create_string_buffer(512)
    fake = ctypes.c_void_p(4096)
    s = lib.qcd_re_dot_static(fake, fake, QCD_RE_DOT_STATIC_MAX_REALS + 2, 64, None, fake, err, len(err))
    assert s == QCD_EINVAL and b"exceeds QCD_RE_DOT_STATIC_MAX_REALS = 50331648" in err.value
    assert lib.qcd_re_dot_static(None, fake, 16, 64, None, fake, err, len(err)) == QCD_EINVAL and b"NULL" in err.value
    assert lib.qcd_re_dot_static(fake, fake, 16, 8, None, fake, None, 0) == QCD_EINVAL
    text = open(__file__.replace("tests/test_zz_no_alloc.py", "include/qcd.h")).read()
    assert f"#define QCD_RE_DOT_STATIC_MAX_REALS {QCD_RE_DOT_STATIC_MAX_REALS}\n" in text
