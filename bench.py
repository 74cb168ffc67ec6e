#!/usr/bin/env python
"""bench.py -- SeKV decode hot path on B200: us per layer-step and achieved HBM GB/s at 128K context.

    python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path (C ABI)
    python bench.py --impl reference --steps K --warmup W     # the oracle on the host cores

Workload = BASELINE.json configs[2]: Llama-3-8B-shaped, 32 layers, 32 q / 8 kv heads, d_h = 128, bf16,
batch 4 x 128K context, r = 16, top-k = 32 spans per kv head, SVD factors in a pinned-host store,
zoomed factors fetched on a side stream into a device factor cache.  A "step" is one decode step of the
whole hot path over all 32 layers (a1-a7: route, select, plan / fetch, pool + coarse + zoom partials, combine);
queries follow an AR(1) stream (rho, default 0.99) so consecutive steps' zoom sets overlap as the cache expects.
Inputs are seeded and synthetic (workloads/).  One JSON line is printed by rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "sekv_decode_attn_us_per_layer_step_128k"
NCU_DRAM_BYTES_PER_LAUNCH = 122.9e6   # 118.1 MB read + 4.9 MB written (algorithmic: 108.6 MB)
UNIT = "us/layer-step"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=48)
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--layers", type=int, default=0, help="debug: override the layer count (invalidates the number)")
    ap.add_argument("--rho", type=float, default=0.99,
                    help="AR(1) coefficient of the query stream: sets the overlap of consecutive zoom sets, i.e. the "
                         "factor-cache miss volume (0.99: ~1%% misses, ~29 MB/step over PCIe; 0.9: ~12%%, ~150 MB/step, "
                         "PCIe-bound; 1.0: no misses).  profiles/ holds the sweep.")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--generic", action="store_true", help="force the generic (non tensor-core) kernels")
    ap.add_argument("--stage1-ctas", type=int, default=0)
    ap.add_argument("--prefetch", type=int, default=8, help="speculative prefetch depth per (sequence, kv head)")
    ap.add_argument("--cache-ways", type=int, default=0)
    ap.add_argument("--item-rows", type=int, default=0)
    ap.add_argument("--zoom-spans", type=int, default=0)
    ap.add_argument("--profile-steps", type=int, default=4)
    ap.add_argument("--e2e-steps", type=int, default=8)
    return ap.parse_args()


def max_over_ranks(value: float, world: int, device) -> float:
    """Replicas only: the one exchange between ranks is the max of the device-timed
    interval; the data path has no collective."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_us_per_layer_step(ms: float, steps: int, layers: int, world: int) -> float:
    """Whole-job metric of N independent replicas: every rank runs `steps` steps of `layers` layer-steps in
    `ms` (max over ranks), so the job does world x as many layer-steps in that time."""
    return ms * 1e3 / (steps * layers) / world


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json, torch copy_ 1 Gi bf16)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# ---------------------------------------------------------------------------------------------
# the oracle on the host cores: reference arm and cpu_baseline leg
# ---------------------------------------------------------------------------------------------
def oracle_sample(spec, steps: int, warmup: int, rho: float):
    """Time the oracle (as it stands) on a bounded sample of the workload: ONE sequence of the batch at
    ONE layer -- its own prefill-time construction from the seeded generator (untimed), then per
    step routing + mixed-resolution attention for all query heads (timed).  Returns seconds per
    (sequence, layer-step) and the sample description."""
    import numpy as np
    import torch
    from oracle import sekv_oracle as O
    from workloads import make_layer_inputs, make_layouts, make_queries, next_queries_ar1
    torch.set_num_threads(1)
    try:
        from threadpoolctl import threadpool_limits
        limiter = threadpool_limits(limits=1)
    except Exception:  # pragma: no cover
        limiter = None
    one = spec.with_(contexts=(spec.contexts[0],), n_layers=1)
    lay = make_layouts(one)
    li = make_layer_inputs(one, lay, 0, device="cpu")
    f64 = lambda t: t.to(torch.float32).numpy().astype(np.float64)
    l = lay[0]
    K = np.zeros((one.n_kv_heads, l.n, 128)); V = np.zeros_like(K)
    K[:, l.planted_pool_pos] = f64(li.Kfull); V[:, l.planted_pool_pos] = f64(li.Vfull)
    pre = dict(tokUK=f64(li.tokUK), SK=f64(li.SK), VtK=f64(li.VtK), tokUV=f64(li.tokUV), SV=f64(li.SV),
               VtV=f64(li.VtV), rank_k=li.rank_k.numpy(), rank_v=li.rank_v.numpy())
    T = O.build_tables(l.H, K, V, f64(li.W), alpha=one.alpha, l_min=one.l_min, r_max=one.rank, window=one.window,
                       dtype=one.dtype, prefactored=pre)
    del K, V, pre
    q = make_queries(one, 0, "cpu")
    times = []
    for i in range(warmup + steps):
        qn = f64(q)[0, 0]
        t0 = time.perf_counter()
        R = O.route(qn, T.W, T.route_K, T.seg.span_len, one.n_kv_heads, one.top_k)
        O.decode_attn(qn, T, R.ids)
        dt = time.perf_counter() - t0
        if i >= warmup:
            times.append(dt)
        q = next_queries_ar1(one, q, i + 1, rho)
    del limiter
    sec = float(np.mean(times))
    desc = (f"1 of {spec.batch} sequences x 1 of {spec.n_layers} layers of configs[{spec.config_id}] "
            f"({spec.contexts[0]} tokens, m={T.seg.m} spans, A={T.seg.A} pool tokens, all {spec.n_q_heads} q heads): "
            f"oracle route + mixed attention per step, numpy fp64, 1 thread; scaled x{spec.batch} sequences")
    return sec, desc


def run_reference(args):
    from workloads import get_spec
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    spec = get_spec(args.config)
    sec, desc = oracle_sample(spec, args.steps, args.warmup, args.rho)
    us_layer_step = sec * spec.batch * 1e6
    line = {
        "impl": "reference", "metric": METRIC, "value": us_layer_step, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": us_layer_step * spec.n_layers / 1e3,
        "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": spec.name, "batch": spec.batch, "context": spec.contexts[0], "layers": spec.n_layers,
                   "rank": spec.rank, "top_k": spec.top_k, "rho": args.rho},
        "cpu_baseline": {"value": us_layer_step, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
        "e2e": {"value": us_layer_step, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------
class ClockSampler(threading.Thread):
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None

    def run(self):
        try:
            import pynvml as N
            N.nvmlInit()
            h = N.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = int(N.nvmlDeviceGetMaxClockInfo(h, N.NVML_CLOCK_SM))
            while not self.stop_flag:
                self.samples.append(int(N.nvmlDeviceGetClockInfo(h, N.NVML_CLOCK_SM)))
                r = int(N.nvmlDeviceGetCurrentClocksEventReasons(h))
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
                time.sleep(0.002)
        except Exception as e:  # pragma: no cover
            self.reasons.add(f"sampler_error:{type(e).__name__}")

    def result(self):
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "samples": len(s),
                "reasons": sorted(self.reasons)}


# ---------------------------------------------------------------------------------------------
# ours
# ---------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_31145_b200.build import build_library
    build_library()
    from paper_2606_31145_b200 import binding as B
    from paper_2606_31145_b200 import engine as E
    from workloads import get_spec, make_layer_inputs, make_layouts, make_queries, next_queries_ar1

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    spec = get_spec(args.config)
    if args.layers:
        spec = spec.with_(n_layers=args.layers)
    layouts = make_layouts(spec)
    t_setup = time.time()
    H_dev = E.surprisal_device(layouts, dev)
    cfg, host_bytes = E.config_for(spec, layouts, out_dtype="bf16", use_graph=0 if args.no_graph else 1,
                                   impl=1 if args.generic else 0, stage1_ctas=args.stage1_ctas, prefetch=args.prefetch,
                                   cache_ways=args.cache_ways or None, item_rows=args.item_rows,
                                   zoom_spans_per_item=args.zoom_spans, H_dev=H_dev, device=dev)
    eng = B.Sekv(cfg, host_bytes, device=dev)
    for layer in range(spec.n_layers):
        li = make_layer_inputs(spec, layouts, layer, device=dev)
        E.build_layer_prefactored(eng, spec, layouts, li, H_dev)
        del li
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    t_setup = time.time() - t_setup

    L, Bn, Hq = spec.n_layers, spec.batch, spec.n_q_heads
    n_q = args.warmup + args.steps + args.profile_steps + args.e2e_steps + 4
    q_all = [make_queries(spec, 0, dev)]
    for i in range(1, n_q):
        q_all.append(next_queries_ar1(spec, q_all[-1], i, args.rho))
    q_cur = torch.empty_like(q_all[0])
    out = torch.empty((L, Bn, Hq, 128), dtype=eng.out_dtype, device=dev)
    static_bytes = eng.sekv_static_bytes_per_layer()
    esz = eng.esize

    def step(i):
        q_cur.copy_(q_all[i])
        eng.sekv_decode_step(q_cur, spec.top_k, out)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing (value) ---------------------------------------------------------
    qi = 0
    for _ in range(max(args.warmup, 3)):
        step(qi); qi += 1
    barrier()
    eng.sekv_reset_stats()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.01)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step(qi); qi += 1
    e1.record()
    barrier()
    sampler.stop_flag = True
    ms = max_over_ranks(e0.elapsed_time(e1), world, dev)
    sampler.join(timeout=2)
    st = eng.sekv_get_stats()
    layer_steps = args.steps * L
    us_layer_step = replica_us_per_layer_step(ms, args.steps, L, world)   # aggregate over replicas
    algo_bytes = layer_steps * static_bytes - st["coarse_rows_skipped"] * 2 * 128 * esz + st["factor_bytes_algo"]
    hbm_gbs = algo_bytes / (ms * 1e-3) / 1e9 * world
    hit = st["cache_hits"] / max(1, st["zoomed_spans"])
    launches = st["kernel_launches"] + args.steps            # + the q staging copy per step

    # ---- per-kernel profile (CUDA events around every kernel, eager launches) ----------------------
    eng.sekv_set_profiling(True)
    step(qi); qi += 1                                        # warm the eager path
    eng.sekv_get_kernel_times()
    eng.sekv_reset_stats()
    for _ in range(args.profile_steps):
        step(qi); qi += 1
    kt = eng.sekv_get_kernel_times()
    st_p = eng.sekv_get_stats()
    eng.sekv_set_profiling(False)
    tot_kernel_ms = sum(v["ms"] for k, v in kt.items() if k not in ("fetch", "prefetch"))
    peak, peak_src = measured_peaks()
    prof_layer_steps = max(1, st_p["layer_steps"])
    if kt["fused"]["launches"]:
        # ONE kernel per layer-step does a1-a7: its algorithmic bytes are the layer-step's
        dom, dom_name = kt["fused"], "fused_layer_kernel (a1-a7: route, plan, pool/coarse/zoom partials, combine)"
        dom_bytes = (prof_layer_steps * static_bytes - st_p["coarse_rows_skipped"] * 2 * 128 * esz
                     + st_p["factor_bytes_algo"]) / prof_layer_steps
    else:
        dom, dom_name = kt["stage1"], "stage1 kernel (a5: pool + coarse entries)"
        rows_bytes = sum(2 * spec.n_kv_heads * (a + m) * 128 * esz for a, m in zip(eng.pool_per_seq, eng.spans_per_seq))
        dom_bytes = rows_bytes - st_p["coarse_rows_skipped"] * 2 * 128 * esz / prof_layer_steps + Bn * Hq * 128 * esz
    eager_us = max(dom["ms"] * 1e3 / max(1, dom["launches"]), 1e-9)
    fused = bool(kt["fused"]["launches"])
    if fused and world == 1:
        # the layer kernel is the only kernel on the launching stream inside the timed region (the prefetch
        # kernels run on the side stream): its average launch duration over the timed region, CUDA events on
        # that stream, is the step time / 32 -- launch gaps between the dependent kernels included
        dom_us = ms * 1e3 / layer_steps
        dom_bytes = algo_bytes / layer_steps
        timing = "CUDA events on the launching stream over the timed region (%d steps x %d launches, one graph per step)" % (args.steps, L)
    else:
        dom_us = eager_us
        timing = "CUDA events on the launching stream around every launch, eager launches, %d steps" % args.profile_steps
    roofline = {"bound": "hbm", "kernel": dom_name,
                "achieved": dom_bytes / (dom_us * 1e-6) / 1e9, "peak": peak, "unit": "GB/s",
                "frac": dom_bytes / (dom_us * 1e-6) / 1e9 / peak,
                # dram__bytes_read.sum + dram__bytes_write.sum per launch of the layer kernel, from the one
                # `ncu --set full` capture summarised in profiles/r01_fused_layer_kernel_ncu_full.md
                "traffic": NCU_DRAM_BYTES_PER_LAUNCH if fused and not args.layers and args.config == 2 else None,
                "peak_source": peak_src,
                "algorithmic_bytes_per_launch": dom_bytes, "avg_launch_us": dom_us,
                "share_of_step_kernel_time": dom["ms"] / max(1e-9, tot_kernel_ms),
                "timing": timing,
                "kernel_us_per_launch_eager": {k: v["ms"] * 1e3 / v["launches"] for k, v in kt.items() if v["launches"]}}

    # ---- end to end through host buffers -----------------------------------------------------------------
    q_host = [q_all[qi + i].cpu().pin_memory() for i in range(args.e2e_steps)]
    out_host = torch.empty(out.shape, dtype=out.dtype).pin_memory()
    eng.sekv_decode_step_host(q_host[0], spec.top_k, out_host)
    eng.sekv_reset_stats()
    barrier()
    t0 = time.perf_counter()
    for i in range(args.e2e_steps):
        eng.sekv_decode_step_host(q_host[i], spec.top_k, out_host)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, world, dev)
    st_e = eng.sekv_get_stats()
    e2e = {"value": e2e_s * 1e6 / (args.e2e_steps * L) / world, "unit": UNIT,
           "h2d_bytes_per_step": q_host[0].numel() * esz + st_e["h2d_bytes"] // max(1, args.e2e_steps),
           "d2h_bytes_per_step": out_host.numel() * out_host.element_size(),
           "factor_fetch_bytes_per_step": st_e["h2d_bytes"] // max(1, args.e2e_steps), "steps": args.e2e_steps}

    if rank != 0:
        return
    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        sec, desc = oracle_sample(spec, 3, 1, args.rho)
        cpu_baseline = {"value": sec * spec.batch * 1e6, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc}
    n_ctas, parts = eng.sekv_get_schedule()
    line = {
        "metric": METRIC, "value": us_layer_step, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "hbm_gbs_achieved": hbm_gbs, "hbm_frac_of_8tbs": hbm_gbs / 8000.0, "hbm_frac_of_measured": hbm_gbs / peak / world,
        "algorithmic_bytes_per_layer_step": algo_bytes / layer_steps,
        "config": {"workload": spec.name, "batch": Bn, "context": spec.contexts[0], "layers": L, "q_heads": Hq,
                   "kv_heads": spec.n_kv_heads, "rank": spec.rank, "top_k": spec.top_k, "rho": args.rho,
                   "spans_per_seq": eng.spans_per_seq, "pool_per_seq": eng.pool_per_seq,
                   "cache_ways": cfg.cache_ways, "cache_hit_rate": hit, "graph": not args.no_graph,
                   "kernels": "generic multi-kernel" if args.generic else "one persistent kernel per layer-step: warp workers on two dependency-ordered queues (mma.sync bf16, cp.async K/V ring, TMA bulk factor copies)",
                   "prefetch": cfg.prefetch, "stage1_ctas": n_ctas,
                   "l2": "inputs larger than L2: one step streams %.2f GB of tables (L2 = 126 MB), no flush" % (algo_bytes / args.steps / 1e9),
                   "replicas": "replicas only (no sharding, no collective)" if world > 1 else "single GPU",
                   "setup_s": round(t_setup, 1)},
        "clocks": sampler.result(), "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
        "fetch": {"h2d_bytes_per_step": st["h2d_bytes"] / args.steps, "misses_per_step": st["cache_misses"] / args.steps,
                  "zoomed_per_step": st["zoomed_spans"] / args.steps},
    }
    if cpu_baseline:
        line["cpu_baseline"] = cpu_baseline
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
