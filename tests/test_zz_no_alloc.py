"""gf8_quantize_f32_noalloc: the quantizer for callers that cannot allocate (static device scratch, no context).
Collected last on purpose (file name): the suite runs with `pytest -x`, and a failure here must not hide other tests.

The new entry point against the existing path (gf8_quantize_f32 through a context) at the tolerance that path is tested at
against the oracle -- bit for bit (gate G1) -- on two calls in a row that share the static scratch: the second call is a
different tensor of a different shape and scaling, so anything left over from the first would show.  The no-alloc calls come
first, so the test also passes alone in a fresh process, before any context exists."""
import pytest
import torch

from paper_2607_07494_b200 import gf8

pytestmark = pytest.mark.gpu


def _tensor(m, n, seed, scale):
    g = torch.Generator(device="cuda").manual_seed(seed)
    x = torch.randn(m, n, device="cuda", generator=g) * torch.exp(2.0 * torch.randn(m, n, device="cuda", generator=g)) * scale
    x[m // 2, n // 3] = 0.0
    return x.contiguous()


def _n_scales(scaling, m, n):
    return 1 if scaling == gf8.SCALE_TENSOR else ((m + 127) // 128) * ((n + 127) // 128)


def test_no_alloc_quantizer_matches_the_context_path_on_two_calls_in_a_row():
    calls = [  # (m, n, fmt, scaling, seed, magnitude): large first, then smaller values, fewer scales, the other format
        (515, 1040, gf8.E4M3, gf8.SCALE_BLOCK128, 1, 100.0),
        (208, 336, gf8.E5M2, gf8.SCALE_TENSOR, 2, 1e-3),
        (400, 272, gf8.E4M3, gf8.SCALE_TENSOR, 3, 5.0),
        (144, 400, gf8.E5M2, gf8.SCALE_BLOCK128, 4, 1e-2),
    ]
    xs = [_tensor(m, n, seed, mag) for m, n, _, _, seed, mag in calls]
    outs = [(torch.empty((m, n), dtype=torch.uint8, device="cuda"),
             torch.empty(_n_scales(sc, m, n), dtype=torch.float32, device="cuda")) for m, n, _, sc, _, _ in calls]
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for x, (codes, sinv), (m, n, fmt, sc, _, _) in zip(xs, outs, calls):        # back to back on one stream, no sync between
        gf8.quantize_f32_noalloc(x, codes, sinv, fmt, sc)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    ctx = gf8.create([gf8.Layer(256, 256, gf8.SIDE_NONE)])                     # the existing path
    for x, (codes, sinv), (m, n, fmt, sc, _, _) in zip(xs, outs, calls):
        want_codes, want_sinv = ctx.quantize_f32(x, fmt, sc)
        assert torch.equal(sinv.view(torch.int32), want_sinv.view(torch.int32)), (m, n, fmt, sc)
        assert torch.equal(codes, want_codes), (m, n, fmt, sc)
    # and again after the context path has run (same inputs, same static scratch): still identical
    codes2 = torch.empty_like(outs[0][0]); sinv2 = torch.empty_like(outs[0][1])
    gf8.quantize_f32_noalloc(xs[0], codes2, sinv2, calls[0][2], calls[0][3])
    torch.cuda.synchronize()
    assert torch.equal(codes2, outs[0][0]) and torch.equal(sinv2, outs[0][1])


def test_no_alloc_quantizer_rejects_what_its_static_scratch_cannot_hold():
    x = torch.zeros((16, 16), dtype=torch.float32, device="cuda")
    codes = torch.empty((16, 16), dtype=torch.uint8, device="cuda")
    sinv = torch.empty(1, dtype=torch.float32, device="cuda")
    L = gf8.lib()
    # 257 x 256 blocks of 128 x 128 = 65792 scales > GF8_NOALLOC_MAX_SCALES (argument check only: nothing is launched or read)
    st = L.gf8_quantize_f32_noalloc(gf8.E4M3, gf8.SCALE_BLOCK128, x.data_ptr(), 257 * 128, 256 * 128, codes.data_ptr(),
                                    sinv.data_ptr(), None)
    assert st == 3 and b"GF8_NOALLOC_MAX_SCALES" in L.gf8_noalloc_last_error()
    # per-tensor scaling has no size limit of its own; a bad argument is reported, not launched
    assert L.gf8_quantize_f32_noalloc(gf8.E4M3, gf8.SCALE_TENSOR, x.data_ptr(), 16, 24, codes.data_ptr(), sinv.data_ptr(), None) == 3
    assert L.gf8_quantize_f32_noalloc(gf8.E4M3, gf8.SCALE_TENSOR, None, 16, 16, codes.data_ptr(), sinv.data_ptr(), None) == 1
    with pytest.raises(gf8.Gf8Error):
        gf8.quantize_f32_noalloc(torch.zeros((16, 24), dtype=torch.float32, device="cuda"), codes, sinv)
