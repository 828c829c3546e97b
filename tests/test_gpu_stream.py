"""The opt-in streaming engine (GF8_STREAM=1; gf8_stream.cuh): one persistent launch per gf8_encode_many.
It is not the default (slower than the staged item engine), but it is part of the library, so it keeps the same gates:
G2 transform within the FAST tier of the oracle, G3-self (its codes and scales are bit-identical to the ORACLE quantizer
applied to its own tapped W~), per-tensor and per-128x128-block scaling, several tensors and ranks per launch."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_07494_b200 import gf8
from tests._util import Case, relfro, to_np64

pytestmark = pytest.mark.gpu

SHAPES = {
    "llama600m-q": dict(m=1536, n=1536, kG=64, kA=64, side=gf8.SIDE_BOTH, dtype="bf16", seed=5, T=4096, q=2),
    "tall-ragged-rows": dict(m=1168, n=640, kG=48, kA=64, side=gf8.SIDE_BOTH, dtype="bf16", seed=21, q=2),
    "block-scaled": dict(m=640, n=1024, kG=64, kA=32, side=gf8.SIDE_BOTH, dtype="bf16", seed=22, q=2, scaling=gf8.SCALE_BLOCK128),
    "in-only": dict(m=400, n=512, kG=0, kA=64, side=gf8.SIDE_IN, dtype="bf16", seed=23, q=2),
}


@pytest.mark.parametrize("name", list(SHAPES))
def test_streaming_engine_meets_the_fast_gates(name, monkeypatch):
    monkeypatch.setenv("GF8_STREAM", "1")              # read once, in gf8_create
    c = Case(precision=gf8.PREC_FAST, **SHAPES[name])
    R = 3
    gs = [c.rank_grad(r).contiguous() for r in range(R)]
    codes = [torch.empty((c.m, c.n), dtype=torch.uint8, device="cuda") for _ in range(R)]
    sinvs = [torch.empty(c.layer.n_scales(), dtype=torch.float32, device="cuda") for _ in range(R)]
    before = c.ctx.launch_count()
    c.ctx.encode_many([0] * R, gs, codes, sinvs)
    c.ctx.sync_check()
    assert c.ctx.launch_count() - before <= 2, "the call did not go through the single-launch engine (pointer patch + one launch)"
    for r in range(R):
        tap = c.ctx.whiten_f32(0, gs[r])
        c.ctx.sync_check()
        _, _, wt = c.oracle_encode(gs[r])
        assert relfro(to_np64(tap), wt) <= 2e-3, (name, r)
        oc, os_ = oracle.quantize(tap.cpu().numpy(), c.fmt, c.scaling)
        assert np.array_equal(codes[r].cpu().numpy(), oc), (name, r)
        assert np.array_equal(sinvs[r].cpu().numpy().view(np.uint32), os_.view(np.uint32)), (name, r)
    # same buffers again (plan reuse, no pointer patching) and new buffers (device-side tensor-map patching)
    c.ctx.encode_many([0] * R, gs, codes, sinvs)
    codes2 = [torch.empty_like(x) for x in codes]
    sinvs2 = [torch.empty_like(x) for x in sinvs]
    c.ctx.encode_many([0] * R, [g.clone() for g in gs], codes2, sinvs2)
    c.ctx.sync_check()
    for r in range(R):
        assert torch.equal(codes[r], codes2[r]) and torch.equal(sinvs[r], sinvs2[r])
