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


def cpu_sample(cfg_index, seed_rank=0):
    """The bounded oracle sample: layer-0 q, k, v, o matrices of the config (side BOTH, the config's k),
    R = 1: oracle encode (O3 + O4) and reduce_decoded (O5 + O6).  Returns (elements, seconds, cores, text)."""
    import numpy as np
    import torch
    import oracle
    from paper_2607_07494_b200 import synth
    cfg = synth.config(cfg_index, layers=1)
    ts = [t for t in cfg.tensors if t.side == synth.SIDE_BOTH][:4]
    items = []
    for t in ts:
        G = synth.tensor_gradient(cfg, t, "cpu").double().numpy()
        lam = cfg.damping
        bs = []
        for side, d in (("out", t.d_out), ("in", t.d_in)):
            # a synthetic orthonormal basis with the config's power-law Ritz values (the refresh itself is
            # not part of the timed codec step)
            U = synth.rand_orthonormal(d, t.rank, "cpu", cfg.index, t.layer, t.matrix, 41 if side == "in" else 42)
            mu = (np.arange(1, t.rank + 1, dtype=np.float64)) ** -2.0
            tail = float(((np.arange(t.rank + 1, d + 1, dtype=np.float64)) ** -2.0).mean())
            rho, e, eb = oracle.multipliers(mu, d, float(mu.sum() + tail * (d - t.rank)), lam)
            bs.append(oracle.Basis(U.double().numpy(), mu, rho, e, eb))
        items.append((G, bs[0], bs[1]))
    t0 = time.perf_counter()
    for G, bG, bA in items:
        c, s, _ = oracle.encode(G, bG, bA, cfg.fmt, cfg.scaling)
        oracle.to_bf16_bits(oracle.reduce_decoded([c], [s], bG, bA, cfg.fmt, cfg.scaling, average=True))
    dt = time.perf_counter() - t0
    n = sum(t.d_out * t.d_in for t in ts)
    return n, dt, oracle.num_threads(), (f"{cfg.name} layer 0 q,k,v,o ({len(ts)} x {ts[0].d_out}x{ts[0].d_in}, k={ts[0].rank}, "
                                         f"side BOTH), R=1: oracle encode + reduce_decoded, {n} elements")


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

    cfg = synth.config(args.config, layers=args.layers)
    R = args.ranks or cfg.R
    prec = gf8.PREC_FAST if args.precision == "fast" else gf8.PREC_EXACT
    layers = [gf8.Layer(t.d_out, t.d_in, t.side, t.rank, t.rank, cfg.fmt, cfg.scaling, cfg.damping) for t in cfg.tensors]
    ctx = gf8.create(layers, prec)
    ids = list(range(len(layers)))
    n_el = cfg.n_elements
    wh_el = sum(t.d_out * t.d_in for t in cfg.tensors if t.side != synth.SIDE_NONE)

    # ---- geometry state through the library (a1, a2): factor update + basis refresh of every whitened tensor
    torch.cuda.synchronize()
    t_gen0 = time.perf_counter()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    geo_ms = 0.0
    fac_ms = 0.0
    for i, t in enumerate(cfg.tensors):
        if t.side == synth.SIDE_NONE:
            continue
        if args.synthetic_basis:
            # profiling aid: seeded orthonormal bases with the configs' i^-2 Ritz values handed to the library,
            # instead of running a1 + a2 (thousands of small launches) before the timed region
            for side, d in ((gf8.SIDE_IN, t.d_in), (gf8.SIDE_OUT, t.d_out)):
                U = synth.rand_orthonormal(d, t.rank, dev, cfg.index, t.layer, t.matrix, 41 + side).contiguous()
                mu = torch.arange(1, t.rank + 1, device=dev, dtype=torch.float32) ** -2.0
                ctx.set_basis(i, side, U, mu, 1.0 / t.rank / d + cfg.damping)
            continue
        X = synth.tensor_factor_samples(cfg, t, "in", dev)
        D = synth.tensor_factor_samples(cfg, t, "out", dev)
        ctx.set_basis(i, gf8.SIDE_IN, synth.tensor_start_basis(cfg, t, "in", dev))
        ctx.set_basis(i, gf8.SIDE_OUT, synth.tensor_start_basis(cfg, t, "out", dev))
        ev[0].record()
        ctx.factor_update(i, X, D)
        ev[1].record()
        ev[1].synchronize()
        fac_ms += ev[0].elapsed_time(ev[1])
        del X, D
    whitened = [i for i, t in enumerate(cfg.tensors) if t.side != synth.SIDE_NONE]
    if whitened and not args.synthetic_basis:
        ev[0].record()
        ctx.refresh_basis_many(whitened, args.refresh_iters)      # independent factors refresh concurrently
        ev[1].record()
        ev[1].synchronize()
        geo_ms = fac_ms + ev[0].elapsed_time(ev[1])
    # ---- gradients: R simulated ranks resident in HBM (inputs >> L2: 2 B * n_el * R)
    grads = [[None] * len(ids) for _ in range(R)]
    for i, t in enumerate(cfg.tensors):
        G = synth.tensor_gradient(cfg, t, dev)
        for r in range(R):
            grads[r][i] = synth.tensor_rank_gradient(cfg, t, G, r)
        del G
    codes = [[torch.empty((t.d_out, t.d_in), dtype=torch.uint8, device=dev) for t in cfg.tensors] for _ in range(R)]
    sinvs = [[torch.empty((layers[i].n_scales(),), dtype=torch.float32, device=dev) for i in ids] for _ in range(R)]
    outs = [torch.empty((t.d_out, t.d_in), dtype=torch.bfloat16 if cfg.dtype == "bf16" else torch.float32, device=dev)
            for t in cfg.tensors]
    codes_flat = [codes[r][i] for i in ids for r in range(R)]
    sinvs_flat = [sinvs[r][i] for i in ids for r in range(R)]
    # one batched call encodes every (tensor, rank) payload: pointer tables are marshalled once, as a training
    # loop that reuses its gradient buffers would
    dtc = gf8.DT_BF16 if cfg.dtype == "bf16" else gf8.DT_F32
    a_ids_all = gf8.int_array([i for i in ids for _ in range(R)])
    a_ids = gf8.int_array(ids)
    a_grads = gf8.ptr_array([grads[r][i] for i in ids for r in range(R)])
    a_codes, a_sinvs, a_outs = gf8.ptr_array(codes_flat), gf8.ptr_array(sinvs_flat), gf8.ptr_array(outs)
    torch.cuda.synchronize()
    gen_s = time.perf_counter() - t_gen0

    def encode_all():
        ctx.encode_many(a_ids_all, a_grads, a_codes, a_sinvs, dt=dtc)

    def reduce_all():
        ctx.reduce_decoded_many(a_ids, a_codes, a_sinvs, R, a_outs, average=True, dt=dtc)

    def step():
        encode_all()
        reduce_all()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    seg = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    l0 = ctx.launch_count()
    barrier()
    e0.record()
    for s in range(args.steps):
        seg[s][0].record()
        encode_all()
        seg[s][1].record()
        reduce_all()
        seg[s][2].record()
    e1.record()
    barrier()
    ctx.sync_check()
    clocks = sampler.stop()
    launches = ctx.launch_count() - l0
    ms = e0.elapsed_time(e1)
    enc_ms = sum(a.elapsed_time(b) for a, b, _ in seg) / args.steps
    red_ms = sum(b.elapsed_time(c) for _, b, c in seg) / args.steps
    ms = max_over_ranks(ms, world, dev)
    ms_step = ms / args.steps
    esz = 2 if cfg.dtype == "bf16" else 4
    value = job_value(world, R, n_el, ms_step)

    # ---- roofline of the dominant call: encode (3 B/element: 2 read BF16 + 1 write FP8)
    hbm_peak, tf_peak, which = _peaks()
    enc_bytes = R * n_el * (esz + 1)
    red_bytes = n_el * (R + esz)
    enc_gbs = enc_bytes / (enc_ms * 1e-3) / 1e9
    red_gbs = red_bytes / (red_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "gf8::tc::tc_items_kernel — the 5 launches of one gf8_encode_many call over all R ranks (a3-a6; 98 % of "
                          "the call, profiles/r01_launches.md) + the Euclidean tensors' streaming kernels", "achieved": enc_gbs, "peak": hbm_peak,
                "unit": "GB/s", "frac": enc_gbs / hbm_peak, "traffic": None, "peak_source": which,
                "algorithmic_bytes_per_launch": enc_bytes, "ms_per_launch": enc_ms,
                "reduce_decoded": {"achieved": red_gbs, "frac": red_gbs / hbm_peak, "ms": red_ms,
                                   "algorithmic_bytes": red_bytes},
                "pipeline": {"achieved": (enc_bytes + red_bytes) / (ms_step * 1e-3) / 1e9,
                             "frac": (enc_bytes + red_bytes) / (ms_step * 1e-3) / 1e9 / hbm_peak,
                             "frac_of_nominal_8TBps": (enc_bytes + red_bytes) / (ms_step * 1e-3) / 1e9 / 8000.0},
                "tensor_flops_per_step": (R + 1) * wh_el * 8 * (cfg.tensors[0].rank if cfg.tensors[0].side else 0),
                }
    tp = os.path.join(ROOT, "profiles", "r01_traffic.json.txt")
    if os.path.exists(tp):
        try:
            roofline["traffic"] = json.load(open(tp)).get("encode_dram_bytes_per_launch")
        except Exception:
            pass

    # ---- e2e: the same step through gf8_step_host with pinned HOST buffers (H2D + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        del codes, sinvs, codes_flat, sinvs_flat, a_codes, a_sinvs, a_grads
        hg = [g.cpu().pin_memory() for i in ids for g in [grads[r][i] for r in range(R)]]
        ho = [torch.empty_like(o, device="cpu").pin_memory() for o in outs]
        del grads
        torch.cuda.empty_cache()
        ctx.step_host(ids, hg, R, ho)
        barrier()
        k2 = max(1, min(args.steps, args.e2e_steps))
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(k2):
            ctx.step_host(ids, hg, R, ho)
        b.record()
        barrier()
        ems = a.elapsed_time(b) / k2
        ems = max_over_ranks(ems, world, dev)
        e2e = {"value": job_value(world, R, n_el, ems), "unit": UNIT,
               "h2d_bytes_per_step": R * n_el * esz, "d2h_bytes_per_step": n_el * esz, "steps": k2, "ms_per_step": ems}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n, dt, cores, text = cpu_sample(args.config)
        cpu = {"value": n * 2 / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": text, "seconds": dt}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "bf16" if cfg.dtype == "bf16" else "f32", "data": "synthetic",
                "config": {"workload": f"configs[{cfg.index}] {cfg.name}: {len(ids)} tensors, {n_el} elements/rank, R={R} "
                                       f"simulated ranks, k={cfg.tensors[0].rank} side BOTH, embedding+LM head Euclidean, "
                                       f"E4M3 per-tensor scale", "precision": args.precision, "layers": args.layers or 24,
                           "l2": "inputs larger than L2 (per-step working set %.1f GB)" % ((R * n_el * (esz + 1) + n_el * esz) / 1e9),
                           "replicas": "independent replica per GPU, no collective" if world > 1 else "single GPU",
                           "geometry": "synthetic bases (set_basis)" if args.synthetic_basis else "factor_update + refresh_basis"},
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches),
                "clocks": clocks, "encode_ms": enc_ms, "reduce_decoded_ms": red_ms, "geometry_ms": geo_ms, "factor_update_ms": fac_ms,
                "setup_s": gen_s}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


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
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_gf8(args)


if __name__ == "__main__":
    sys.exit(main())
