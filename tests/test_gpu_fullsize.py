"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (DESIGN.md 2 "Parity at size").

Every config's shapes go through the batched calls with the argument lists bench.py builds; geometry state comes from
gf8_factor_update + gf8_refresh_basis on the GPU and is itself gated (G6 on sampled factor entries, G7 on T, Ritz values and
orthonormality at d up to 4096) before it is handed to the oracle, so each codec stage is compared in isolation:
  G2  transform tap vs the oracle's dense-form Eq. 14 on >= 1024 sampled elements (the whole-matrix oracle costs m n k^2)
  G3  FAST self-consistency on the WHOLE tensor: fused codes and scales bit-identical to the oracle quantizer on the GPU's tap
  G5  reduce_decoded vs oracle reduce (whole tensor, FP32, rank order) + dense-form Eq. 17 on sampled elements
  Euclidean tensors (32000 x h): codes, scales and the reduced BF16 gradient bit-exact.
Tolerances are the stated gates: 1e-4 on geometry state, 2e-3 on the FAST transform / decode in FP32, and for BF16 output
2e-3 + 2^-9 (one BF16 rounding of the result)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_07494_b200 import gf8, synth
from tests._util import bf16_bits, relfro, to_np64

pytestmark = pytest.mark.gpu

TOL_GEOM = 1e-4
TOL_FAST = 2e-3
TOL_FAST_BF16 = 2e-3 + 2.0 ** -9
NS = 1024                      # sampled elements per comparison


def sample_positions(m, n, ns, seed):
    """Uniform positions plus the corners and the elements on both sides of every kind of tile boundary."""
    rng = np.random.default_rng(seed)
    ii, jj = rng.integers(0, m, ns), rng.integers(0, n, ns)
    edge_r = [0, m - 1, 127, 128, 255, 256, m // 2]
    edge_c = [0, n - 1, 63, 64, 127, 128, n // 2]
    k = 0
    for r in edge_r:
        for c in edge_c:
            ii[k], jj[k] = min(r, m - 1), min(c, n - 1)
            k += 1
    return ii, jj


def rel_samples(got, want):
    return float(np.linalg.norm(np.asarray(got, np.float64) - want) / max(np.linalg.norm(want), 1e-300))


def gpu_basis(ctx, layer, side, lam):
    """The GPU's basis of one layer side as an oracle.Basis (handed across: the codec stages are compared in isolation)."""
    U, mu, rho = ctx.get_basis(layer, side)
    mu64 = to_np64(mu)
    D = np.sqrt(rho / (mu64 + lam))
    return oracle.Basis(to_np64(U), mu64, rho, D - 1.0, 1.0 / D - 1.0)


def check_g6_sampled(ctx, layer, side, X, seed, prev=None, beta=0.0):
    """Sampled entries of the GPU factor vs O1; with `prev` = (ii, jj, values) the EMA recursion runs on those entries."""
    d = X.shape[1]
    if prev is None:
        rng = np.random.default_rng(seed)
        ii, jj = rng.integers(0, d, 512), rng.integers(0, d, 512)
        ii[:4], jj[:4] = [0, d - 1, 127, 128], [0, d - 1, 128, 127]
        want = oracle.factor_entries(to_np64(X), ii, jj)
    else:
        ii, jj = prev[0], prev[1]
        want = beta * prev[2] + (1.0 - beta) * oracle.factor_entries(to_np64(X), ii, jj)
    got = to_np64(ctx.get_factor(layer, side))[ii, jj]
    assert rel_samples(got, want) <= TOL_GEOM, rel_samples(got, want)
    return ii, jj, want


def check_g7(ctx, layer, side, V0, q, lam):
    """GPU refresh vs O2 on the SAME factor bits, start basis and iteration count: orthonormality, Ritz values, rho, T."""
    F = to_np64(ctx.get_factor(layer, side))
    b = oracle.refresh_basis(F, to_np64(V0), q, lam)
    U, mu, rho = ctx.get_basis(layer, side)
    U, mu = to_np64(U), to_np64(mu)
    k = U.shape[1]
    assert np.abs(U.T @ U - np.eye(k)).max() <= 1e-5
    assert np.abs(mu - b.mu).max() <= 1e-4 * (b.mu.min() + lam) and abs(rho - b.rho) <= 1e-5 * b.rho
    D = np.sqrt(rho / (mu + lam))
    # T = I + U diag(D - 1) U^T is sign / rotation invariant; compare the low-rank parts (||T_gpu - T_orc||_F / ||T_orc||_F)
    Lg, Lo = (U * (D - 1)) @ U.T, (b.U * b.e) @ b.U.T
    d = U.shape[0]
    t_norm = np.sqrt(np.linalg.norm(Lo) ** 2 + 2.0 * np.trace(Lo) + d)
    assert np.linalg.norm(Lg - Lo) / t_norm <= TOL_GEOM


def codec_checks(ctx, lay_ids, shapes, grads, R, lam, fmt, scaling, rank_checked, seed, out_dtype=torch.bfloat16, k_note=""):
    """encode_many / reduce_decoded_many over `lay_ids` x R ranks with bench.py's argument lists, then G2 / G3-self / G5 per layer."""
    ids_all = [i for i in lay_ids for _ in range(R)]
    flat = [grads[i][r] for i in lay_ids for r in range(R)]
    lays = {i: shapes[i] for i in lay_ids}
    codes = [torch.empty(g.shape, dtype=torch.uint8, device="cuda") for g in flat]
    n_sc = lambda i: 1 if scaling == gf8.SCALE_TENSOR else ((lays[i][0] + 127) // 128) * ((lays[i][1] + 127) // 128)
    sinvs = [torch.empty(n_sc(i), dtype=torch.float32, device="cuda") for i in ids_all]
    a_ids, a_g, a_c, a_s = gf8.int_array(ids_all), gf8.ptr_array(flat), gf8.ptr_array(codes), gf8.ptr_array(sinvs)
    ctx.encode_many(a_ids, a_g, a_c, a_s, dt=gf8.DT_BF16)
    ctx.sync_check()
    outs = [torch.empty(shapes[i], dtype=out_dtype, device="cuda") for i in lay_ids]
    ctx.reduce_decoded_many(gf8.int_array(lay_ids), a_c, a_s, R, gf8.ptr_array(outs), average=True,
                            dt=gf8.DT_BF16 if out_dtype == torch.bfloat16 else gf8.DT_F32)
    ctx.sync_check()
    for q, i in enumerate(lay_ids):
        m, n = shapes[i]
        bA, bG = gpu_basis(ctx, i, gf8.SIDE_IN, lam), gpu_basis(ctx, i, gf8.SIDE_OUT, lam)
        ii, jj = sample_positions(m, n, NS, seed + i)
        g = grads[i][rank_checked]
        wt = ctx.whiten_f32(i, g)
        ctx.sync_check()
        want = oracle.whiten_samples(to_np64(g), ii, jj, bG.U, bG.e, bA.U, bA.e)
        wt_np = wt.cpu().numpy()
        assert rel_samples(wt_np[ii, jj], want) <= TOL_FAST, (i, k_note, rel_samples(wt_np[ii, jj], want))             # G2
        j = q * R + rank_checked
        oc, os_ = oracle.quantize(wt_np, fmt, scaling)
        assert np.array_equal(codes[j].cpu().numpy(), oc) and np.array_equal(sinvs[j].cpu().numpy(), os_), (i, k_note)  # G3-self
        pc = [codes[q * R + r].cpu().numpy() for r in range(R)]
        ps = [sinvs[q * R + r].cpu().numpy() for r in range(R)]
        uhat = oracle.reduce(pc, ps, fmt, scaling, True)
        want5 = oracle.whiten_samples(uhat.astype(np.float64), ii, jj, bG.U, bG.ebar, bA.U, bA.ebar)
        tol5 = TOL_FAST_BF16 if out_dtype == torch.bfloat16 else TOL_FAST
        got5 = outs[q].float().cpu().numpy()[ii, jj]
        assert rel_samples(got5, want5) <= tol5, (i, k_note, rel_samples(got5, want5))                                  # G5
    return codes, sinvs


def euclidean_checks(ctx, layer, grads_r, fmt=gf8.E4M3):
    """side = NONE tensor through the batched calls: codes, scales and the reduced BF16 gradient bit-exact."""
    R = len(grads_r)
    codes = [torch.empty(g.shape, dtype=torch.uint8, device="cuda") for g in grads_r]
    sinvs = [torch.empty(1, dtype=torch.float32, device="cuda") for _ in grads_r]
    ctx.encode_many([layer] * R, grads_r, codes, sinvs)
    ctx.sync_check()
    pays = [oracle.quantize(g.float().cpu().numpy(), fmt) for g in grads_r]
    for (oc, os_), c_, s_ in zip(pays, codes, sinvs):
        assert np.array_equal(c_.cpu().numpy(), oc) and np.array_equal(s_.cpu().numpy(), os_)
    out = torch.empty(grads_r[0].shape, dtype=torch.bfloat16, device="cuda")
    ctx.reduce_decoded_many([layer], codes, sinvs, R, [out], average=True)
    ctx.sync_check()
    want = oracle.reduce([p[0] for p in pays], [p[1] for p in pays], fmt)
    assert np.array_equal(bf16_bits(out), oracle.to_bf16_bits(want.astype(np.float64)))


def llama_shaped(cfg_index, tensors_wanted, refresh_iters=2):
    """One transformer layer of configs[cfg_index] + the embedding, geometry through the library as bench.py does it."""
    cfg = synth.config(cfg_index, layers=1)
    ts = [t for t in cfg.tensors if t.name.split(".")[-1] in tensors_wanted or t.name in tensors_wanted]
    layers = [gf8.Layer(t.d_out, t.d_in, t.side, t.rank, t.rank, cfg.fmt, cfg.scaling, cfg.damping) for t in ts]
    ctx = gf8.create(layers, gf8.PREC_FAST)
    whitened = [i for i, t in enumerate(ts) if t.side != synth.SIDE_NONE]
    starts = {}
    for i in whitened:
        t = ts[i]
        X = synth.tensor_factor_samples(cfg, t, "in", "cuda")
        D = synth.tensor_factor_samples(cfg, t, "out", "cuda")
        V0A, V0G = synth.tensor_start_basis(cfg, t, "in", "cuda"), synth.tensor_start_basis(cfg, t, "out", "cuda")
        ctx.set_basis(i, gf8.SIDE_IN, V0A)
        ctx.set_basis(i, gf8.SIDE_OUT, V0G)
        ctx.factor_update(i, X, D)
        ctx.sync_check()
        check_g6_sampled(ctx, i, gf8.SIDE_IN, X, 100 + i)
        check_g6_sampled(ctx, i, gf8.SIDE_OUT, D, 200 + i)
        starts[i] = (V0A, V0G)
        del X, D
    ctx.refresh_basis_many(whitened, refresh_iters)
    torch.cuda.synchronize()
    for i in whitened:
        check_g7(ctx, i, gf8.SIDE_IN, starts[i][0], refresh_iters, cfg.damping)
        check_g7(ctx, i, gf8.SIDE_OUT, starts[i][1], refresh_iters, cfg.damping)
    grads = {}
    for i, t in enumerate(ts):
        G = synth.tensor_gradient(cfg, t, "cuda")
        grads[i] = [synth.tensor_rank_gradient(cfg, t, G, r) for r in range(cfg.R)]
    return cfg, ts, ctx, whitened, grads


def test_cfg1_llama300m_shapes_at_size():
    """configs[1]: 1024 x 1024, 2816 x 1024, 1024 x 2816 at k = 32 (R = 4) and a 32000 x 1024 Euclidean tensor."""
    cfg, ts, ctx, whitened, grads = llama_shaped(1, ("q", "gate", "down", "embed"))
    shapes = {i: (t.d_out, t.d_in) for i, t in enumerate(ts)}
    codec_checks(ctx, whitened, shapes, grads, cfg.R, cfg.damping, cfg.fmt, cfg.scaling, rank_checked=1, seed=1000)
    e = [i for i, t in enumerate(ts) if t.side == synth.SIDE_NONE][0]
    euclidean_checks(ctx, e, grads[e])


def test_cfg2_llama600m_shapes_at_size_with_the_bench_argument_lists():
    """configs[2]: every tensor of one layer (q, k, v, o, gate, up, down at k = 64) + embedding and LM head, R = 8, through
    ONE encode_many and ONE reduce_decoded_many with bench.py's lists (tensor-major, rank-minor; whitened and Euclidean mixed)."""
    cfg, ts, ctx, whitened, grads = llama_shaped(2, ("q", "k", "v", "o", "gate", "up", "down", "embed", "lm_head"))
    R = cfg.R
    ids = list(range(len(ts)))
    shapes = {i: (t.d_out, t.d_in) for i, t in enumerate(ts)}
    flat = [grads[i][r] for i in ids for r in range(R)]
    codes = [torch.empty(g.shape, dtype=torch.uint8, device="cuda") for g in flat]
    sinvs = [torch.empty(1, dtype=torch.float32, device="cuda") for _ in flat]
    outs = [torch.empty(shapes[i], dtype=torch.bfloat16, device="cuda") for i in ids]
    a_c, a_s = gf8.ptr_array(codes), gf8.ptr_array(sinvs)
    ctx.encode_many(gf8.int_array([i for i in ids for _ in range(R)]), gf8.ptr_array(flat), a_c, a_s, dt=gf8.DT_BF16)
    ctx.reduce_decoded_many(gf8.int_array(ids), a_c, a_s, R, gf8.ptr_array(outs), average=True, dt=gf8.DT_BF16)
    ctx.sync_check()
    for i in ids:
        t = ts[i]
        pc = [codes[i * R + r].cpu().numpy() for r in range(R)]
        ps = [sinvs[i * R + r].cpu().numpy() for r in range(R)]
        uhat = oracle.reduce(pc, ps, cfg.fmt, cfg.scaling, True)
        if t.side == synth.SIDE_NONE:                           # bit-exact plain FP8
            for r in (0, R - 1):
                oc, os_ = oracle.quantize(grads[i][r].float().cpu().numpy(), cfg.fmt)
                assert np.array_equal(pc[r], oc) and np.array_equal(ps[r], os_)
            assert np.array_equal(bf16_bits(outs[i]), oracle.to_bf16_bits(uhat.astype(np.float64)))
            continue
        r = (3 + i) % R
        wt = ctx.whiten_f32(i, grads[i][r]).cpu().numpy()
        oc, os_ = oracle.quantize(wt, cfg.fmt, cfg.scaling)
        assert np.array_equal(pc[r], oc) and np.array_equal(ps[r], os_), t.name                                      # G3-self
        if t.name.split(".")[-1] in ("q", "gate", "down"):      # one tensor per distinct shape: G2 and G5 on sampled elements
            bA, bG = gpu_basis(ctx, i, gf8.SIDE_IN, cfg.damping), gpu_basis(ctx, i, gf8.SIDE_OUT, cfg.damping)
            ii, jj = sample_positions(t.d_out, t.d_in, NS, 2000 + i)
            want = oracle.whiten_samples(to_np64(grads[i][r]), ii, jj, bG.U, bG.e, bA.U, bA.e)
            assert rel_samples(wt[ii, jj], want) <= TOL_FAST, t.name
            want5 = oracle.whiten_samples(uhat.astype(np.float64), ii, jj, bG.U, bG.ebar, bA.U, bA.ebar)
            got5 = outs[i].float().cpu().numpy()[ii, jj]
            assert rel_samples(got5, want5) <= TOL_FAST_BF16, (t.name, rel_samples(got5, want5))


@pytest.mark.parametrize("k", [8, 32, 128, 512])
def test_cfg3_sweep_4096_square(k):
    """configs[3]: one 4096 x 4096 BF16 gradient, k in {8, 32, 128, 512} x {E4M3, E5M2} x {per-tensor, per-128x128-block}.
    Bases come from factor_update (T = 16384) + refresh_basis on the GPU (gated by G6 / G7) except at k = 512, where the
    oracle's refresh (d^2 k flops per product in plain loops) is out of reach and a seeded orthonormal basis with the
    config's i^-2 Ritz values is handed to both sides."""
    t = synth.sweep_tensor(k)
    lam, m, n = 1e-3, t.d_out, t.d_in
    combos = [(f, s) for f in (gf8.E4M3, gf8.E5M2) for s in (gf8.SCALE_TENSOR, gf8.SCALE_BLOCK128)]
    ctx = gf8.create([gf8.Layer(m, n, gf8.SIDE_BOTH, k, k, f, s, lam) for f, s in combos], gf8.PREC_FAST)
    if k < 512:
        X = synth.factor_samples(t.tokens, n, "cuda", 3, k, 0).to(torch.bfloat16)
        D = synth.factor_samples(t.tokens, m, "cuda", 3, k, 1).to(torch.bfloat16)
        V0A, V0G = synth.start_basis(n, k, "cuda", 3, k, 0), synth.start_basis(m, k, "cuda", 3, k, 1)
        ctx.set_basis(0, gf8.SIDE_IN, V0A)
        ctx.set_basis(0, gf8.SIDE_OUT, V0G)
        ctx.factor_update(0, X, D)
        ctx.sync_check()
        check_g6_sampled(ctx, 0, gf8.SIDE_IN, X, 31)
        check_g6_sampled(ctx, 0, gf8.SIDE_OUT, D, 32)
        ctx.refresh_basis(0, 2)
        torch.cuda.synchronize()
        check_g7(ctx, 0, gf8.SIDE_IN, V0A, 2, lam)
        check_g7(ctx, 0, gf8.SIDE_OUT, V0G, 2, lam)
        for side in (gf8.SIDE_IN, gf8.SIDE_OUT):
            U, mu, rho = ctx.get_basis(0, side)
            for l in range(1, len(combos)):
                ctx.set_basis(l, side, U, mu, rho)
    else:
        for side, d in ((gf8.SIDE_IN, n), (gf8.SIDE_OUT, m)):
            U = synth.rand_orthonormal(d, k, "cuda", 3, k, 40 + side).contiguous()
            mu = torch.arange(1, k + 1, device="cuda", dtype=torch.float32) ** -2.0
            for l in range(len(combos)):
                ctx.set_basis(l, side, U, mu, float(1.0 / k / d + lam))
    G = synth.gradient(m, n, "cuda", 3, k, 7, noise=0.01).to(torch.bfloat16)
    bA, bG = gpu_basis(ctx, 0, gf8.SIDE_IN, lam), gpu_basis(ctx, 0, gf8.SIDE_OUT, lam)
    ii, jj = sample_positions(m, n, NS, 3000 + k)
    wt = ctx.whiten_f32(0, G)
    ctx.sync_check()
    wt_np = wt.cpu().numpy()
    want = oracle.whiten_samples(to_np64(G), ii, jj, bG.U, bG.e, bA.U, bA.e)
    assert rel_samples(wt_np[ii, jj], want) <= TOL_FAST, rel_samples(wt_np[ii, jj], want)                              # G2
    for l, (fmt, scaling) in enumerate(combos):
        c_, s_ = ctx.encode(l, G)
        ctx.sync_check()
        # (the tap of the SAME layer: a basis copied with set_basis gets its multipliers from FP32 Ritz values, the refreshed
        #  layer 0 from the FP64 ones, so W~ of layer l and of layer 0 may differ in the last bits)
        wt_l = wt_np if l == 0 else ctx.whiten_f32(l, G).cpu().numpy()
        oc, os_ = oracle.quantize(wt_l, fmt, scaling)
        assert np.array_equal(c_.cpu().numpy(), oc) and np.array_equal(s_.cpu().numpy(), os_), (k, fmt, scaling)      # G3-self
        out = ctx.decode(l, c_, s_, dt=gf8.DT_F32)
        ctx.sync_check()
        uhat = oracle.reduce([oc], [os_], fmt, scaling, False)
        want5 = oracle.whiten_samples(uhat.astype(np.float64), ii, jj, bG.U, bG.ebar, bA.U, bA.ebar)
        got5 = out.cpu().numpy()[ii, jj]
        assert rel_samples(got5, want5) <= TOL_FAST, (k, fmt, scaling, rel_samples(got5, want5))                     # G5


def test_cfg4_stress_R16_with_periodic_refresh_at_size():
    """configs[4]: R = 16 perturbed replicas of the 600M-shaped q (1536 x 1536) and down (1536 x 4096) gradients and the
    embedding, 50 steps, EMA factor update (beta = 0.9) + warm refresh (q = 2) every 10 steps.  After the last refresh: G6 on
    sampled entries of the EMA chain, G7 on the last refresh, G5 on the last step (R = 16: the ungrouped-reduce path)."""
    cfg = synth.config(4, layers=1)
    ts = [t for t in cfg.tensors if t.name in ("l0.q", "l0.down", "embed")]
    beta, R, lam = 0.9, cfg.R, cfg.damping
    assert R == 16
    layers = [gf8.Layer(t.d_out, t.d_in, t.side, t.rank, t.rank, cfg.fmt, cfg.scaling, lam, beta) for t in ts]
    ctx = gf8.create(layers, gf8.PREC_FAST)
    wh = [0, 1]
    for i in wh:
        ctx.set_basis(i, gf8.SIDE_IN, synth.tensor_start_basis(cfg, ts[i], "in", "cuda"))
        ctx.set_basis(i, gf8.SIDE_OUT, synth.tensor_start_basis(cfg, ts[i], "out", "cuda"))
    G = [synth.tensor_gradient(cfg, t, "cuda") for t in ts]
    ids = list(range(len(ts)))
    codes = [torch.empty((ts[i].d_out, ts[i].d_in), dtype=torch.uint8, device="cuda") for i in ids for _ in range(R)]
    sinvs = [torch.empty(1, dtype=torch.float32, device="cuda") for _ in codes]
    outs = [torch.empty((t.d_out, t.d_in), dtype=torch.bfloat16, device="cuda") for t in ts]
    a_ids_all, a_ids = gf8.int_array([i for i in ids for _ in range(R)]), gf8.int_array(ids)
    a_c, a_s, a_o = gf8.ptr_array(codes), gf8.ptr_array(sinvs), gf8.ptr_array(outs)
    ema = {}                                                     # (layer, side) -> (ii, jj, running value of the sampled entries)
    grads = None
    for step in range(50):
        if step % 10 == 0:
            refresh = step // 10
            before = {}
            for i in wh:
                X = synth.tensor_factor_samples(cfg, ts[i], "in", "cuda", refresh)
                D = synth.tensor_factor_samples(cfg, ts[i], "out", "cuda", refresh)
                ctx.factor_update(i, X, D)
                ctx.sync_check()
                for side, S in ((gf8.SIDE_IN, X), (gf8.SIDE_OUT, D)):
                    ema[(i, side)] = check_g6_sampled(ctx, i, side, S, 400 + i, ema.get((i, side)), beta)
                    if step == 40:
                        before[(i, side)] = ctx.get_basis(i, side)[0].clone()      # warm start of the last refresh
                del X, D
            ctx.refresh_basis_many(wh, 8 if step == 0 else 2)
            torch.cuda.synchronize()
            if step == 40:
                for (i, side), V0 in before.items():
                    check_g7(ctx, i, side, V0, 2, lam)
        grads = [[synth.rank_gradient(G[i], r, 4, i, step).to(torch.bfloat16) for r in range(R)] for i in ids]
        ctx.encode_many(a_ids_all, gf8.ptr_array([grads[i][r] for i in ids for r in range(R)]), a_c, a_s, dt=gf8.DT_BF16)
        ctx.reduce_decoded_many(a_ids, a_c, a_s, R, a_o, average=True, dt=gf8.DT_BF16)
    ctx.sync_check()
    for i in ids:
        t = ts[i]
        pc = [codes[i * R + r].cpu().numpy() for r in range(R)]
        ps = [sinvs[i * R + r].cpu().numpy() for r in range(R)]
        uhat = oracle.reduce(pc, ps, cfg.fmt, cfg.scaling, True)
        if t.side == synth.SIDE_NONE:
            assert np.array_equal(bf16_bits(outs[i]), oracle.to_bf16_bits(uhat.astype(np.float64)))
            continue
        bA, bG = gpu_basis(ctx, i, gf8.SIDE_IN, lam), gpu_basis(ctx, i, gf8.SIDE_OUT, lam)
        ii, jj = sample_positions(t.d_out, t.d_in, NS, 4000 + i)
        want5 = oracle.whiten_samples(uhat.astype(np.float64), ii, jj, bG.U, bG.ebar, bA.U, bA.ebar)
        got5 = outs[i].float().cpu().numpy()[ii, jj]
        assert rel_samples(got5, want5) <= TOL_FAST_BF16, (t.name, rel_samples(got5, want5))
        # the fused codes of the last step, self-consistent against the tap (rank 7)
        wt = ctx.whiten_f32(i, grads[i][7]).cpu().numpy()
        oc, os_ = oracle.quantize(wt, cfg.fmt, cfg.scaling)
        assert np.array_equal(pc[7], oc) and np.array_equal(ps[7], os_), t.name
        # the 16 independent perturbations average out: the decoded mean is close to the shared gradient
        assert relfro(to_np64(outs[i]), to_np64(G[i])) <= 0.1


@pytest.mark.parametrize("scaling", [gf8.SCALE_TENSOR, gf8.SCALE_BLOCK128])
def test_largest_whitened_shape_embedding_sized(scaling):
    """Maximum sizes: a WHITENED tensor of the configs' largest shape (32000 x 1024: the embedding / LM head, which the
    configs leave Euclidean) and its transpose-shaped sibling (1024 x 8192), two ranks each, through the batched calls:
    250-row-block strips, 125 strips per tensor, side BOTH at k = 32.  Bases are seeded orthonormal matrices handed in with
    set_basis (a 32000^2 factor is not part of any config); G2 / G5 on sampled elements, G3-self on the whole tensor."""
    shapes = [(32000, 1024), (1024, 8192)]
    k, lam, R = 32, 1e-3, 2
    lays = [gf8.Layer(m, n, gf8.SIDE_BOTH, k, k, gf8.E4M3, scaling, lam) for m, n in shapes]
    ctx = gf8.create(lays, gf8.PREC_FAST)
    mu = torch.arange(1, k + 1, device="cuda", dtype=torch.float32) ** -2.0
    for i, (m, n) in enumerate(shapes):
        ctx.set_basis(i, gf8.SIDE_IN, synth.rand_orthonormal(n, k, "cuda", 77, i, 1).contiguous(), mu, 1.0 / k / n + lam)
        ctx.set_basis(i, gf8.SIDE_OUT, synth.rand_orthonormal(m, k, "cuda", 77, i, 2).contiguous(), mu, 1.0 / k / m + lam)
    grads = {}
    for i, (m, n) in enumerate(shapes):
        G = synth.gradient(m, n, "cuda", 78, i)
        grads[i] = [synth.rank_gradient(G, r, 79).to(torch.bfloat16).contiguous() for r in range(R)]
        del G
    codec_checks(ctx, [0, 1], {0: shapes[0], 1: shapes[1]}, grads, R, lam, gf8.E4M3, scaling, 1, 80, k_note="max-size")
