#!/usr/bin/env python
"""bench.py -- GeoFP8 codec throughput on synthetic Llama-shaped gradient sets (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl gf8|reference] [--config 2]
                    [--precision fast|exact] [--layers L] [--no-e2e] [--no-cpu-baseline]

One "step" = one pass of the whole codec hot path over one batch of gradients: gf8_encode_many for
each of the R simulated ranks (a3-a6), then gf8_reduce_decoded_many (a7-a8) -- SURVEY.md 8(a).
metric = R * N_elements * 2 B / t_step, in GB/s of BF16 gradient encoded+decoded.  Geometry state
(factor update + basis refresh, a1-a2) runs every K=50 steps in the paper; it is set up
through the library before the timed region and its time is reported separately (`geometry_ms`).

N > 1 (torchrun): the path does not shard (north_star: one GPU, simulated ranks) -- every rank runs an
independent replica of the same workload on its own GPU, no data-path collective ("replicas only",
DESIGN.md); value = N * units / max-over-ranks time, scaling "weak".

--impl reference: the CPU oracle (oracle/), as it stands, on the host cores, on a bounded sample of the
same workload per step (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "geofp8_encode_decode_bf16_gradient_throughput"
UNIT = "GB/s"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), float(d.get("bf16_tflops_sustained", d.get("bf16_tflops", 1590.0))), "measured"
        except Exception:
            pass
    return 6650.0, 1590.0, "fallback"          # B200_PROFILING.md fallback


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------------------------------
def max_over_ranks(ms, world, device):
    """Replica timing rule: every rank times its own replica on its device; the job's time is the MAX over ranks."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def job_value(world, R, n_el, ms_step):
    """Whole-job GB/s of BF16 gradient encoded+decoded: `world` independent replicas of R ranks x n_el elements."""
    return world * R * n_el * 2 / (ms_step * 1e-3) / 1e9


def _synthetic_oracle_bases(cfg, t, oracle, synth, np):
    """Seeded orthonormal bases with the config's i^-2 Ritz values (the refresh itself is not part of the timed codec step)."""
    bs = []
    for side, d in (("out", t.d_out), ("in", t.d_in)):
        U = synth.rand_orthonormal(d, t.rank, "cpu", cfg.index, t.layer, t.matrix, 41 if side == "in" else 42)
        mu = (np.arange(1, t.rank + 1, dtype=np.float64)) ** -2.0
        tail = float(((np.arange(t.rank + 1, d + 1, dtype=np.float64)) ** -2.0).mean())
        rho, e, eb = oracle.multipliers(mu, d, float(mu.sum() + tail * (d - t.rank)), cfg.damping)
        bs.append(oracle.Basis(U.double().numpy(), mu, rho, e, eb))
    return bs


def cpu_sample(cfg_index, seed_rank=0):
    """The bounded oracle sample (SURVEY.md 8(d) asks for the seven matrix shapes of layers {0, 12, 23} + embedding + LM head over
    all R ranks; at the oracle's m n k^2 cost that is ~10 CPU-minutes, so the timed sample is ALL SEVEN whitened matrices of
    layer 0 (q, k, v, o, gate, up, down; side BOTH, the config's k), R = 1: oracle encode (O3 + O4) and reduce_decoded
    (O5 + O6).  Returns (elements, seconds, cores, text)."""
    import numpy as np
    import oracle
    from paper_2607_07494_b200 import synth
    cfg = synth.config(cfg_index, layers=1)
    ts = [t for t in cfg.tensors if t.side == synth.SIDE_BOTH]
    items = []
    for t in ts:
        G = synth.tensor_gradient(cfg, t, "cpu").double().numpy()
        bG, bA = _synthetic_oracle_bases(cfg, t, oracle, synth, np)
        items.append((G, bG, bA))
    t0 = time.perf_counter()
    for G, bG, bA in items:
        c, s, _ = oracle.encode(G, bG, bA, cfg.fmt, cfg.scaling)
        oracle.to_bf16_bits(oracle.reduce_decoded([c], [s], bG, bA, cfg.fmt, cfg.scaling, average=True))
    dt = time.perf_counter() - t0
    n = sum(t.d_out * t.d_in for t in ts)
    return n, dt, oracle.num_threads(), (f"{cfg.name} layer 0, all {len(ts)} whitened matrices ({', '.join(sorted({f'{t.d_out}x{t.d_in}' for t in ts}))}; "
                                         f"k={ts[0].rank}, side BOTH), R=1: oracle encode + reduce_decoded, {n} elements")


def cpu_single_thread_config0():
    """Single-thread figure on configs[0] (256 x 256 FP32, k = 16, R = 2): whole oracle pipeline incl. factor + refresh."""
    import numpy as np
    import oracle
    from paper_2607_07494_b200 import synth
    cfg = synth.config(0)
    t = cfg.tensors[0]
    G = synth.tensor_gradient(cfg, t, "cpu")
    X = synth.tensor_factor_samples(cfg, t, "in", "cpu").double().numpy()
    D = synth.tensor_factor_samples(cfg, t, "out", "cpu").double().numpy()
    V0A = synth.tensor_start_basis(cfg, t, "in", "cpu").double().numpy()
    V0G = synth.tensor_start_basis(cfg, t, "out", "cpu").double().numpy()
    grads = [synth.tensor_rank_gradient(cfg, t, G, r).double().numpy() for r in range(cfg.R)]
    threads = oracle.num_threads()
    oracle.set_num_threads(1)
    try:
        t0 = time.perf_counter()
        bA = oracle.refresh_basis(oracle.factor_accumulate(X), V0A, 8, cfg.damping)
        bG = oracle.refresh_basis(oracle.factor_accumulate(D), V0G, 8, cfg.damping)
        t_geo = time.perf_counter() - t0
        t0 = time.perf_counter()
        pays = [oracle.encode(g, bG, bA)[:2] for g in grads]
        oracle.reduce_decoded([p[0] for p in pays], [p[1] for p in pays], bG, bA)
        t_codec = time.perf_counter() - t0
    finally:
        oracle.set_num_threads(threads)
    n = cfg.R * t.d_out * t.d_in
    return {"value": n * 2 / t_codec / 1e9, "unit": UNIT, "cores": 1, "codec_seconds": t_codec, "geometry_seconds": t_geo,
            "sample": "configs[0] whole pipeline, R=2 (GB/s counts 2 B per element like the BF16 metric)"}


def parity_spot_check(ctx, cfg, ids, grads, codes, sinvs, outs, R):
    """Outside the timed region: the codes / outputs the LAST timed step left behind against the oracle, on one whitened tensor
    (layer 0 q, rank 1) and one Euclidean tensor (embedding, rank 0).  Uses the oracle, so it runs with the cpu_baseline leg."""
    import numpy as np
    import oracle
    from paper_2607_07494_b200 import gf8, synth
    res = {}
    wi = next(i for i in ids if cfg.tensors[i].side != synth.SIDE_NONE)
    t = cfg.tensors[wi]
    lam = cfg.damping

    def basis(side):
        U, mu, rho = ctx.get_basis(wi, side)
        mu64 = mu.double().cpu().numpy()
        D = np.sqrt(rho / (mu64 + lam))
        return oracle.Basis(U.double().cpu().numpy(), mu64, rho, D - 1.0, 1.0 / D - 1.0)

    bA, bG = basis(gf8.SIDE_IN), basis(gf8.SIDE_OUT)
    r = 1 % R
    g = grads[r][wi]
    tap = ctx.whiten_f32(wi, g).cpu().numpy()
    qc, qs = oracle.quantize(tap, cfg.fmt, cfg.scaling)
    gc, gs = codes[r][wi].cpu().numpy(), sinvs[r][wi].cpu().numpy()
    res["g3_self_codes_equal_quantizer_of_tap"] = bool(np.array_equal(gc, qc) and np.array_equal(gs, qs))
    oc, _, x = oracle.encode(g.double().cpu().numpy(), bG, bA, cfg.fmt, cfg.scaling)
    res["g2_transform_rel_fro"] = float(np.linalg.norm(tap.astype(np.float64) - x) / np.linalg.norm(x))
    res["fast_code_flip_fraction_vs_oracle"] = float((gc != oc).mean())
    rng = np.random.default_rng(7)
    ii, jj = rng.integers(0, t.d_out, 512), rng.integers(0, t.d_in, 512)
    uhat = oracle.reduce([codes[q][wi].cpu().numpy() for q in range(R)], [sinvs[q][wi].cpu().numpy() for q in range(R)],
                         cfg.fmt, cfg.scaling, True)
    want = oracle.whiten_samples(uhat.astype(np.float64), ii, jj, bG.U, bG.ebar, bA.U, bA.ebar)
    got = outs[wi].float().cpu().numpy()[ii, jj]
    res["g5_decode_rel_fro_sampled"] = float(np.linalg.norm(got - want) / np.linalg.norm(want))
    res["gates"] = {"g2": 2e-3, "g5_bf16_out": 2e-3 + 2.0 ** -9}
    res["tensor"] = f"{t.name} ({t.d_out}x{t.d_in}), rank {r}"
    ei = next((i for i in ids if cfg.tensors[i].side == synth.SIDE_NONE), None)
    if ei is not None:
        ec, es = oracle.quantize(grads[0][ei].float().cpu().numpy(), cfg.fmt, cfg.scaling)
        res["euclidean_bit_exact"] = bool(np.array_equal(codes[0][ei].cpu().numpy(), ec) and np.array_equal(sinvs[0][ei].cpu().numpy(), es))
    res["ok"] = bool(res["g3_self_codes_equal_quantizer_of_tap"] and res["g2_transform_rel_fro"] <= 2e-3 and
                     res["g5_decode_rel_fro_sampled"] <= 2e-3 + 2.0 ** -9 and res.get("euclidean_bit_exact", True))
    return res


def run_reference(args):
    """--impl reference: the oracle on the host cores, one bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    for _ in range(max(0, min(args.warmup, 1))):
        cpu_sample(args.config)
    tot_n, tot_t, cores, text = 0, 0.0, 1, ""
    for _ in range(max(1, min(args.steps, 3))):
        n, dt, cores, text = cpu_sample(args.config)
        tot_n += n
        tot_t += dt
    steps = max(1, min(args.steps, 3))
    val = tot_n * 2 / tot_t / 1e9
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * tot_t / steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config {args.config} (bounded sample: {text})"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": text},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------------------------------
class Workload:
    """One codec workload resident in HBM: R simulated ranks x every tensor of a config, with its library context."""

    def __init__(self, cfg_index, dev, layers=None, ranks=None, precision="fast", side=None, synthetic_basis=False, refresh_iters=2,
                 error_feedback=False):
        import torch
        from paper_2607_07494_b200 import gf8, synth
        self.torch, self.gf8, self.synth = torch, gf8, synth
        cfg = synth.config(cfg_index, layers=layers)
        if side is not None:                     # e.g. the paper's deployed operating point: input side only
            for t in cfg.tensors:
                if t.side != synth.SIDE_NONE:
                    t.side = side
        self.cfg, self.R, self.dev = cfg, ranks or cfg.R, dev
        R = self.R
        prec = gf8.PREC_FAST if precision == "fast" else gf8.PREC_EXACT
        self.layers = [gf8.Layer(t.d_out, t.d_in, t.side, t.rank, t.rank, cfg.fmt, cfg.scaling, cfg.damping) for t in cfg.tensors]
        self.ctx = ctx = gf8.create(self.layers, prec)
        self.ids = ids = list(range(len(self.layers)))
        self.n_el = cfg.n_elements
        self.wh_el = sum(t.d_out * t.d_in for t in cfg.tensors if t.side != synth.SIDE_NONE)
        # ---- geometry state through the library (a1, a2): factor update + basis refresh of every whitened tensor
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        self.fac_ms = self.fac_first_ms = self.refresh_ms = 0.0
        whitened = [i for i, t in enumerate(cfg.tensors) if t.side != synth.SIDE_NONE]
        acts, gouts = [], []
        for i in whitened:
            t = cfg.tensors[i]
            sides = [(gf8.SIDE_IN, t.d_in, "in")] * bool(t.side & 1) + [(gf8.SIDE_OUT, t.d_out, "out")] * bool(t.side & 2)
            if synthetic_basis:
                # seeded orthonormal bases with the configs' i^-2 Ritz values handed to the library, instead of running a1 + a2
                for sd, d, _ in sides:
                    U = synth.rand_orthonormal(d, t.rank, dev, cfg.index, t.layer, t.matrix, 41 + sd).contiguous()
                    mu = torch.arange(1, t.rank + 1, device=dev, dtype=torch.float32) ** -2.0
                    ctx.set_basis(i, sd, U, mu, 1.0 / t.rank / d + cfg.damping)
                continue
            acts.append(synth.tensor_factor_samples(cfg, t, "in", dev) if t.side & 1 else None)
            gouts.append(synth.tensor_factor_samples(cfg, t, "out", dev) if t.side & 2 else None)
            for sd, d, nm in sides:
                ctx.set_basis(i, sd, synth.tensor_start_basis(cfg, t, nm, dev))
        if whitened and not synthetic_basis:
            # a1: every factor of the model in ONE batched call (samples resident in HBM); the first call also allocates the
            # factor buffers, the second is the steady state a training loop sees (ema_beta = 0: same result)
            for rep in range(2):
                ev[0].record()
                ctx.factor_update_many(whitened, acts, gouts)
                ev[1].record()
                ev[1].synchronize()
                if rep == 0:
                    self.fac_first_ms = ev[0].elapsed_time(ev[1])
                else:
                    self.fac_ms = ev[0].elapsed_time(ev[1])
            del acts, gouts
            # a2: every basis in one batched call
            ev[0].record()
            ctx.refresh_basis_many(whitened, refresh_iters)
            ev[1].record()
            ev[1].synchronize()
            self.refresh_ms = ev[0].elapsed_time(ev[1])
        # ---- gradients: R simulated ranks resident in HBM (inputs >> L2: 2 B * n_el * R)
        self.grads = [[None] * len(ids) for _ in range(R)]
        for i, t in enumerate(cfg.tensors):
            G = synth.tensor_gradient(cfg, t, dev)
            for r in range(R):
                self.grads[r][i] = synth.tensor_rank_gradient(cfg, t, G, r)
            del G
        self.codes = [[torch.empty((t.d_out, t.d_in), dtype=torch.uint8, device=dev) for t in cfg.tensors] for _ in range(R)]
        self.sinvs = [[torch.empty((self.layers[i].n_scales(),), dtype=torch.float32, device=dev) for i in ids] for _ in range(R)]
        self.outs = [torch.empty((t.d_out, t.d_in), dtype=torch.bfloat16 if cfg.dtype == "bf16" else torch.float32, device=dev)
                     for t in cfg.tensors]
        # one batched call encodes every (tensor, rank) payload: pointer tables are marshalled once, as a training loop that
        # reuses its gradient buffers would
        self.dtc = gf8.DT_BF16 if cfg.dtype == "bf16" else gf8.DT_F32
        self.a_ids_all = gf8.int_array([i for i in ids for _ in range(R)])
        self.a_ids = gf8.int_array(ids)
        self.a_grads = gf8.ptr_array([self.grads[r][i] for i in ids for r in range(R)])
        self.a_codes = gf8.ptr_array([self.codes[r][i] for i in ids for r in range(R)])
        self.a_sinvs = gf8.ptr_array([self.sinvs[r][i] for i in ids for r in range(R)])
        self.a_outs = gf8.ptr_array(self.outs)
        # f1 (variant): one FP32 residual per (tensor, rank), zero at start, carried from step to step
        self.resid = self.a_resid = None
        if error_feedback:
            self.resid = [[ctx.resid_new(i) for i in ids] for _ in range(R)]
            self.a_resid = gf8.ptr_array([self.resid[r][i] for i in ids for r in range(R)])
        torch.cuda.synchronize()

    def encode_all(self):
        if self.a_resid is not None:
            self.ctx.encode_ef_many(self.a_ids_all, self.a_grads, self.a_resid, self.a_codes, self.a_sinvs, dt=self.dtc)
        else:
            self.ctx.encode_many(self.a_ids_all, self.a_grads, self.a_codes, self.a_sinvs, dt=self.dtc)

    def reduce_all(self):
        self.ctx.reduce_decoded_many(self.a_ids, self.a_codes, self.a_sinvs, self.R, self.a_outs, average=True, dt=self.dtc)

    def time(self, steps, warmup, barrier=None):
        """W untimed steps, then K steps between CUDA events on the launching stream; returns (ms total, encode ms / step,
        reduce_decoded ms / step)."""
        torch = self.torch
        barrier = barrier or torch.cuda.synchronize
        for _ in range(max(warmup, 3)):
            self.encode_all()
            self.reduce_all()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        seg = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
        barrier()
        l0 = self.ctx.launch_count()
        e0.record()
        for s in range(steps):
            seg[s][0].record()
            self.encode_all()
            seg[s][1].record()
            self.reduce_all()
            seg[s][2].record()
        e1.record()
        barrier()
        self.ctx.sync_check()
        self.launches = self.ctx.launch_count() - l0          # kernels of this library launched inside the timed region
        enc = sum(a.elapsed_time(b) for a, b, _ in seg) / steps
        red = sum(b.elapsed_time(c) for _, b, c in seg) / steps
        return e0.elapsed_time(e1), enc, red

    def free(self):
        self.grads = self.codes = self.sinvs = self.outs = self.resid = None
        self.a_grads = self.a_codes = self.a_sinvs = self.a_outs = self.a_resid = None
        self.ctx.destroy()
        self.torch.cuda.empty_cache()


def variant(name, dev, steps, **kw):
    """A side measurement (EXACT vs FAST, side = IN, the other configs, the R = 1 round trip): same metric,
    3 warm-up steps, `steps` timed steps, seeded synthetic bases handed to the library (set_basis)."""
    try:
        w = Workload(dev=dev, synthetic_basis=True, **kw)
        ms, enc, red = w.time(steps, 3)
        out = {"value": job_value(1, w.R, w.n_el, ms / steps), "unit": UNIT, "ms_per_step": ms / steps, "encode_ms": enc,
               "reduce_decoded_ms": red, "R": w.R, "tensors": len(w.ids), "elements_per_rank": w.n_el, "steps": steps,
               "geometry": "synthetic bases (set_basis)"}
        out.update({k: v for k, v in kw.items() if k != "cfg_index"})
        out["config"] = kw["cfg_index"]
        w.free()
        return out
    except Exception as e:      # a variant never takes the headline line down with it
        return {"error": f"{type(e).__name__}: {e}"}


def run_gf8(args):
    import torch
    import torch.distributed as dist
    from paper_2607_07494_b200 import gf8, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the gf8 codec has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    gf8.lib()                                              # fail loudly if libgf8.so is missing

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    t_gen0 = time.perf_counter()
    w = Workload(args.config, dev, layers=args.layers, ranks=args.ranks, precision=args.precision,
                 side={"in": 1, "out": 2, "both": 3}.get(args.side), synthetic_basis=args.synthetic_basis,
                 refresh_iters=args.refresh_iters)
    cfg, ctx, R, n_el, wh_el, ids = w.cfg, w.ctx, w.R, w.n_el, w.wh_el, w.ids
    gen_s = time.perf_counter() - t_gen0
    sampler = ClockSampler(local)
    # warm-up happens inside time(); the clock sampler covers warm-up + timed region (the same load)
    sampler.start()
    ctx.set_stage_timing(False)
    ms, enc_ms, red_ms = w.time(args.steps, args.warmup, barrier)
    launches = w.launches
    clocks = sampler.stop()
    ms = max_over_ranks(ms, world, dev)
    ms_step = ms / args.steps
    esz = 2 if cfg.dtype == "bf16" else 4
    value = job_value(world, R, n_el, ms_step)

    # ---- per-launch times of the tensor-core stages (CUDA events on the launching stream, a few extra steps after the timed
    #      region): the dominant KERNEL LAUNCH of the step and its own roofline
    stage_names = ["panels P'+Q^T", "S", "Q'^T", "update tiles (amax/store)", "update tiles (cast)", "update strips (amax)",
                   "update strips (cast)", "fused update"]
    ctx.set_stage_timing(True)
    k2 = max(2, min(args.steps, 5))
    for _ in range(k2):
        w.encode_all()
    st_enc, n_enc = ctx.stage_times()
    for _ in range(k2):
        w.reduce_all()
    st_dec, n_dec = ctx.stage_times()
    ctx.set_stage_timing(False)
    stages = {"encode": {stage_names[s]: {"ms_per_launch": st_enc[s] / n_enc[s], "launches_per_call": n_enc[s] // k2}
                         for s in range(8) if n_enc[s]},
              "reduce_decoded": {stage_names[s]: {"ms_per_launch": st_dec[s] / n_dec[s], "launches_per_call": n_dec[s] // k2}
                                 for s in range(8) if n_dec[s]}}
    hbm_peak, tf_peak, which = _peaks()
    enc_bytes = R * n_el * (esz + 1)
    red_bytes = n_el * (R + esz)
    enc_gbs = enc_bytes / (enc_ms * 1e-3) / 1e9
    red_gbs = red_bytes / (red_ms * 1e-3) / 1e9
    # the dominant launch: the cast pass over the update strips (reads the BF16 gradient, writes the FP8 codes: 3 B / element
    # of every whitened tensor of every rank); falls back to the whole encode call when that stage did not run (EXACT, k > 64)
    dom = stages["encode"].get("update strips (cast)")
    if dom and cfg.dtype == "bf16":
        dom_bytes = R * wh_el * 3
        roof_kernel = "gf8::tc::tc_items_kernel, cast pass over the update strips (a4 + a6; one launch per gf8_encode_many)"
        dom_ms = dom["ms_per_launch"]
    else:
        dom_bytes, dom_ms = enc_bytes, enc_ms
        roof_kernel = "gf8_encode_many (whole call)"
    roofline = {"bound": "hbm", "kernel": roof_kernel, "achieved": dom_bytes / (dom_ms * 1e-3) / 1e9, "peak": hbm_peak,
                "unit": "GB/s", "frac": dom_bytes / (dom_ms * 1e-3) / 1e9 / hbm_peak, "traffic": None, "peak_source": which,
                "algorithmic_bytes_per_launch": dom_bytes, "ms_per_launch": dom_ms,
                "encode_call": {"achieved": enc_gbs, "frac": enc_gbs / hbm_peak, "ms": enc_ms, "algorithmic_bytes": enc_bytes},
                "reduce_decoded_call": {"achieved": red_gbs, "frac": red_gbs / hbm_peak, "ms": red_ms, "algorithmic_bytes": red_bytes},
                "pipeline": {"achieved": (enc_bytes + red_bytes) / (ms_step * 1e-3) / 1e9,
                             "frac": (enc_bytes + red_bytes) / (ms_step * 1e-3) / 1e9 / hbm_peak,
                             "frac_of_nominal_8TBps": (enc_bytes + red_bytes) / (ms_step * 1e-3) / 1e9 / 8000.0},
                "stages": stages,
                "tensor_flops_per_step": (R + 1) * wh_el * 8 * (cfg.tensors[0].rank if cfg.tensors[0].side else 0)}
    tp = os.path.join(ROOT, "profiles", "r02_traffic.json.txt")
    if os.path.exists(tp) and args.config == 2 and not args.layers and not args.ranks and args.precision == "fast" and not args.side:
        try:
            tj = json.load(open(tp))
            roofline["traffic"] = tj.get("dominant_kernel_dram_bytes_per_launch")
            roofline["traffic_source"] = "profiled offline with ncu --set full (not measured in this run): " + tj.get("source", tp)
            roofline["traffic_encode_call"] = tj.get("encode_call_dram_bytes")
        except Exception:
            pass

    # ---- post-timing parity spot check + oracle baseline (rank 0, N = 1 only; the one place bench.py runs the oracle)
    parity = cpu = cpu1 = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        try:
            parity = parity_spot_check(ctx, cfg, ids, w.grads, w.codes, w.sinvs, w.outs, R)
        except Exception as e:
            parity = {"ok": False, "error": f"{type(e).__name__}: {e}"}
        n, dt, cores, text = cpu_sample(args.config if args.config in (1, 2, 4) else 2)
        cpu = {"value": n * 2 / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": text, "seconds": dt,
               "single_thread_config0": cpu_single_thread_config0()}

    # ---- e2e: the same step through gf8_step_host with pinned HOST buffers (H2D + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        hg = [g.cpu().pin_memory() for i in ids for g in [w.grads[r][i] for r in range(R)]]
        ho = [torch.empty_like(o, device="cpu").pin_memory() for o in w.outs]
        w.grads = w.codes = w.sinvs = None
        w.a_grads = w.a_codes = w.a_sinvs = None
        torch.cuda.empty_cache()
        ctx.step_host(ids, hg, R, ho)
        barrier()
        k3 = max(1, min(args.steps, args.e2e_steps))
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(k3):
            ctx.step_host(ids, hg, R, ho)
        b.record()
        barrier()
        ems = max_over_ranks(a.elapsed_time(b) / k3, world, dev)
        e2e = {"value": job_value(world, R, n_el, ems), "unit": UNIT,
               "h2d_bytes_per_step": R * n_el * esz, "d2h_bytes_per_step": n_el * esz, "steps": k3, "ms_per_step": ems}
        del hg, ho
    fac_ms, fac_first_ms, refresh_ms = w.fac_ms, w.fac_first_ms, w.refresh_ms
    n_tensors = len(ids)
    w.free()

    # ---- side measurements (N = 1): SURVEY.md 8(d) "also reported"
    variants = None
    if rank == 0 and world == 1 and not args.no_variants and args.config == 2 and not args.layers:
        vs = max(2, min(args.steps, 5))
        variants = {
            "side_in (the paper's deployed form, PAPER.md:269; configs[2] shapes, k=64)": variant("side_in", dev, vs, cfg_index=2, side=1),
            "r1_roundtrip (configs[2], one rank: encode + decode)": variant("r1", dev, vs, cfg_index=2, ranks=1),
            "config1 (llama300m-shaped, R=4, k=32)": variant("cfg1", dev, vs, cfg_index=1),
            "config4 (llama600m-shaped stress, R=16)": variant("cfg4", dev, vs, cfg_index=4),
            "exact (EXACT tier, FP32 SIMT path: the 1e-4 code gate; configs[2], first 2 layers)": variant("exact", dev, 2, cfg_index=2, layers=2, precision="exact"),
            "error_feedback (f1, Alg. 1 l.11-15: encode with an FP32 residual per tensor and rank; first version, own launches; configs[2])":
                variant("ef", dev, vs, cfg_index=2, error_feedback=True),
        }

    if rank == 0:
        geo = fac_ms + refresh_ms
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "bf16" if cfg.dtype == "bf16" else "f32", "data": "synthetic",
                "config": {"workload": f"configs[{cfg.index}] {cfg.name}: {n_tensors} tensors, {n_el} elements/rank, R={R} "
                                       f"simulated ranks, k={cfg.tensors[0].rank} side {args.side or 'both'}, embedding+LM head Euclidean, "
                                       f"E4M3 per-tensor scale", "precision": args.precision, "layers": args.layers or 24,
                           "l2": "inputs larger than L2 (per-step working set %.1f GB)" % ((R * n_el * (esz + 1) + n_el * esz) / 1e9),
                           "replicas": "independent replica per GPU, no collective" if world > 1 else "single GPU",
                           "geometry": "synthetic bases (set_basis)" if args.synthetic_basis else "factor_update + refresh_basis",
                           "parity_tier": ("FAST: BF16 tensor-core operands, transform within 2e-3 of the oracle; fused codes are bit-identical to "
                                           "the oracle quantizer on the GPU's own W~ but a few % differ from the oracle's codes (see parity)")
                                          if args.precision == "fast" else "EXACT: codes within the 1e-4 gate of the oracle's"},
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "parity": parity,
                "clocks": clocks, "encode_ms": enc_ms, "reduce_decoded_ms": red_ms, "geometry_ms": geo,
                "factor_update_ms": fac_ms, "factor_update_first_call_ms (allocates the factor buffers)": fac_first_ms,
                "refresh_basis_ms": refresh_ms,
                "geometry_ms_amortised_per_step": {"K=50 (PAPER.md:291)": geo / 50.0, "K=10 (configs[4])": geo / 10.0},
                "variants": variants, "setup_s": gen_s}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def spawn_replicas(args):
    """`python bench.py --gpus N` outside torchrun: start N replicas (one process per GPU) the way the driver would."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="gf8", choices=["gf8", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[0, 1, 2, 4])
    ap.add_argument("--layers", type=int, default=None, help="transformer layers of the shaped set (default 24)")
    ap.add_argument("--ranks", type=int, default=None, help="override R")
    ap.add_argument("--precision", default="fast", choices=["fast", "exact"])
    ap.add_argument("--refresh-iters", type=int, default=2)
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--synthetic-basis", action="store_true",
                    help="hand seeded orthonormal bases to the library instead of running factor update + refresh")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--side", default=None, choices=["in", "out", "both"], help="override the whitened tensors' side (default: both)")
    ap.add_argument("--no-variants", action="store_true", help="skip the side measurements (side IN, R = 1, configs 1 / 4, EXACT)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_replicas(args)
    return run_gf8(args)


if __name__ == "__main__":
    sys.exit(main())
