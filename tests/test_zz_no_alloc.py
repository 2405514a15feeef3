"""-m gpu test of wd_norm2_noalloc (include/wilson_cg.h): the dot-product kernel <a,a> for callers that
cannot call cudaMalloc.  Its reduction scratch is a static __device__ array of the library, shared by every call, so the
test makes several calls in a row on fields of DIFFERENT sizes (a stale partial or a ticket counter left over from the
previous call would show) and compares each with the existing path, wd_norm2 on a context, within the tolerance of
test_norm2_matches_oracle_and_is_deterministic (1e-6 / 1e-13 relative), and with the fp64 oracle.

The file name sorts last on purpose: the run is `pytest -x`, and this entry point is an addition outside the
hot path, so a failure here must not hide any other test.  It passes alone in a fresh process and after the others.
"""
import ctypes

import numpy as np
import pytest

from paper_2111_14958_b200 import inputs
import gpu_util as gu

pytestmark = pytest.mark.gpu

TOL = {32: 1e-6, 64: 1e-13}
CFG_TEST = 760


@pytest.fixture(scope="module")
def wilson():
    import torch

    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_2111_14958_b200 import build as wbuild
    from paper_2111_14958_b200 import wilson as w

    wbuild.build()
    w.load_library()
    return w


def _noalloc(wilson, a_native, V, precision, stream=None):
    import torch

    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()            # `out` and the input are complete before another stream touches them
    wilson.wd_norm2_noalloc(a_native, V, precision, out, stream=stream)
    if stream is not None:
        stream.synchronize()
    torch.cuda.synchronize()
    return float(out.item())


@pytest.mark.parametrize("precision", [32, 64])
def test_noalloc_norm2_matches_existing_path_on_calls_in_a_row(wilson, oracle, precision):
    # large, small (ragged: V = 840 is not a multiple of the 16-site block, pad lanes must not count), large again
    cases = [(14, 14, 14, 14), (5, 7, 4, 6), (4, 4, 4, 4), (14, 14, 14, 14)]
    fields, want_ctx, want_oracle = [], [], []
    for k, dims in enumerate(cases):
        a = inputs.source_field(CFG_TEST + k, dims, dtype=gu.np_complex(precision))
        with wilson.WilsonContext(dims, precision) as ctx:
            an = ctx.wd_pack_spinor(gu.to_device(a))
            want_ctx.append(ctx.wd_norm2(an))
        fields.append((an, int(np.prod(dims))))
        want_oracle.append(oracle.norm2(a.astype(np.complex128)))
    wilson.wd_noalloc_prepare()
    got = [_noalloc(wilson, an, V, precision) for an, V in fields]       # the calls in a row, nothing in between
    again = [_noalloc(wilson, an, V, precision) for an, V in fields]
    for g, g2, wc, wo in zip(got, again, want_ctx, want_oracle):
        assert np.isfinite(g) and g > 0
        assert abs(g - wc) <= TOL[precision] * wc, (g, wc)
        assert abs(g - wo) <= TOL[precision] * wo, (g, wo)
        assert g == g2                                                     # fixed summation order: bit-identical


def test_noalloc_norm2_on_a_side_stream_and_at_full_size(wilson):
    """config 4 (48^3 x 96, fp32: 1.02 GB, 15 552 of the 16 384 partials) then a small field, on a non-default stream"""
    import torch

    dims = (48, 48, 48, 96)
    V = int(np.prod(dims))
    assert V <= wilson.wd_noalloc_max_sites(32)
    g = torch.Generator(device="cuda").manual_seed(CFG_TEST)
    big = torch.randn(24 * V, dtype=torch.float32, device="cuda", generator=g)     # any data is a native field when V % 16 == 0
    small = torch.randn(24 * 4096, dtype=torch.float32, device="cuda", generator=g)
    with wilson.WilsonContext(dims, 32) as ctx:
        want_big = ctx.wd_norm2(big)
    with wilson.WilsonContext((8, 8, 8, 8), 32) as ctx:
        want_small = ctx.wd_norm2(small)
    s = torch.cuda.Stream()
    torch.cuda.synchronize()
    got_big = _noalloc(wilson, big, V, 32, stream=s)
    got_small = _noalloc(wilson, small, 4096, 32, stream=s)
    got_big2 = _noalloc(wilson, big, V, 32, stream=s)
    assert abs(got_big - want_big) <= TOL[32] * want_big
    assert abs(got_small - want_small) <= TOL[32] * want_small
    assert got_big2 == got_big
    # the plain definition in fp64.  Like wd_norm2, the kernel squares and adds the four reals of a 128-bit vector in fp32
    # before the fp64 accumulation (reading G17: the products are in the field's precision), hence the fp32 tolerance;
    # the observed difference is 1e-11 relative (independent roundings of 6.4e7 vectors average out)
    ref = float((big.double() ** 2).sum().item())
    assert abs(got_big - ref) <= TOL[32] * ref
    assert abs(got_big - ref) <= 1e-9 * ref


def test_noalloc_norm2_rejects_what_it_cannot_do(wilson):
    import torch

    lib = wilson.load_library()
    a = torch.zeros(24 * 256, dtype=torch.float32, device="cuda")
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    for precision in (32, 64):
        limit = wilson.wd_noalloc_max_sites(precision)
        assert limit == {32: 11184800, 64: 5592400}[precision]
        with pytest.raises(wilson.WilsonError) as e:
            wilson.wd_norm2_noalloc(a, limit + 16, precision, out)       # rejected before anything is launched
        assert e.value.code == -2 and "exceed the static scratch" in str(e.value)
    with pytest.raises(wilson.WilsonError) as e:
        wilson.wd_norm2_noalloc(a, 0, 32, out)
    assert e.value.code == -2
    with pytest.raises(wilson.WilsonError) as e:
        wilson.wd_norm2_noalloc(a, 256, 16, out)
    assert e.value.code == -5
    assert lib.wd_norm2_noalloc(32, 256, None, ctypes.c_void_p(out.data_ptr()), None) == -1
    assert lib.wd_norm2_noalloc(32, 256, ctypes.c_void_p(a.data_ptr()), None, None) == -1
    assert b"NULL" in lib.wd_noalloc_last_error()
    # still usable after the errors, and the message is cleared by a success
    a.fill_(1.0)
    assert _noalloc(wilson, a, 256, 32) == 24.0 * 256
    assert lib.wd_noalloc_last_error() == b""


@pytest.mark.parametrize("precision", [32, 64])
def test_noalloc_norm2_reads_only_its_field(wilson, precision):
    """the field sits between two bands of NaNs and its own pad lanes (V = 840 is not a multiple of the 16-site block) hold
    NaNs too: a read outside the field, or of a pad lane, would make the result NaN; the result slot sits between guard
    words that must stay untouched"""
    import torch

    dims = (5, 7, 4, 6)
    V = int(np.prod(dims))
    a = inputs.source_field(CFG_TEST + 9, dims, dtype=gu.np_complex(precision))
    rdt = torch.float32 if precision == 32 else torch.float64
    with wilson.WilsonContext(dims, precision) as ctx:
        an = ctx.wd_pack_spinor(gu.to_device(a))
        want = ctx.wd_norm2(an)
    n = an.numel()
    guard = 4096
    buf = torch.full((n + 2 * guard,), float("nan"), dtype=rdt, device="cuda")
    field = buf[guard:guard + n]
    field.copy_(an)
    # poison the pad lanes of the last 16-site block: plane-major blocks of NSP planes x 16 sites x (128 bit)
    per_vec = 4 if precision == 32 else 2
    nsp = 6 if precision == 32 else 12
    blocks = field.view(-1, nsp, 16, per_vec)
    assert blocks.shape[0] * 16 >= V
    blocks[-1, :, V % 16:, :] = float("nan")
    res = torch.full((3,), -7.0, dtype=torch.float64, device="cuda")
    wilson.wd_norm2_noalloc(field, V, precision, res[1:2])
    torch.cuda.synchronize()
    got = res.cpu().numpy()
    assert got[0] == -7.0 and got[2] == -7.0
    assert np.isfinite(got[1]) and abs(got[1] - want) <= TOL[precision] * want
    assert torch.isnan(buf[:guard]).all() and torch.isnan(buf[guard + n:]).all()
