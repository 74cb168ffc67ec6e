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
UNIT = "us/layer-step"
NCU_TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r02_ncu_traffic.json")
KERNEL_SOURCES = ("fused_kernels.cu", "mma_common.cuh", "sekv_internal.cuh")


def kernel_sha256() -> str:
    """Digest of the sources of the layer kernel: the ncu traffic figure is only quoted for the kernel it was
    captured on (profiles/r02_ncu_traffic.json records this digest)."""
    import hashlib
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2606_31145_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def ncu_traffic_per_launch():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the layer kernel from the tracked ncu capture,
    or None when the kernel sources have changed since (a stale figure is not quoted)."""
    try:
        d = json.load(open(NCU_TRAFFIC_JSON))
    except Exception:
        return None, "no tracked ncu capture"
    if d.get("kernel_sha256") != kernel_sha256():
        return None, "stale: kernel sources changed since the capture at %s" % d.get("commit", "?")
    return float(d["dram_bytes_per_launch"]), "profiles/r02_ncu_traffic.json (captured at %s)" % d.get("commit", "?")


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
    ap.add_argument("--e2e-steps", type=int, default=24)
    ap.add_argument("--sweep-steps", type=int, default=10, help="timed steps per rho of the sweep (0 = no sweep)")
    ap.add_argument("--oracle-worker", default="", help=argparse.SUPPRESS)
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
_ORACLE_STATE = {}


def _oracle_head(arg):
    """Pool worker (forked after the tables were built: shares them copy-on-write): the oracle's mixed attention
    for one query head."""
    h, q, ids = arg
    st = _ORACLE_STATE
    out, lse = st["O"].decode_attn(q, st["T"], ids, heads=[h])
    return h, out[h], lse[h]


def oracle_sample(spec, steps: int, warmup: int, rho: float, all_cores: bool = False):
    """Time the oracle (as it stands) on a bounded sample of the workload: ONE sequence of the batch at
    ONE layer -- its own prefill-time construction from the seeded generator (untimed), then per
    step routing + mixed-resolution attention for all query heads (timed), on one thread and, with
    all_cores, with one forked process per query head over all host cores.  Returns a dict with
    seconds per (sequence, layer-step) for both and the sample description."""
    import multiprocessing as mp
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
    qs = []
    for i in range(warmup + steps):
        qs.append(f64(q)[0, 0])
        q = next_queries_ar1(one, q, i + 1, rho)
    times = []
    for i, qn in enumerate(qs):
        t0 = time.perf_counter()
        R = O.route(qn, T.W, T.route_K, T.seg.span_len, one.n_kv_heads, one.top_k)
        ref, _ = O.decode_attn(qn, T, R.ids)
        dt = time.perf_counter() - t0
        if i >= warmup:
            times.append(dt)
    res = {"sec_1": float(np.mean(times)), "cores_all": 1, "sec_all": None}
    if all_cores:
        nproc = os.cpu_count() or 1
        workers = max(1, min(nproc, one.n_q_heads))
        _ORACLE_STATE.update(O=O, T=T)
        tp = []
        with mp.get_context("fork").Pool(workers) as pool:
            for i, qn in enumerate(qs):
                t0 = time.perf_counter()
                R = O.route(qn, T.W, T.route_K, T.seg.span_len, one.n_kv_heads, one.top_k)
                got = pool.map(_oracle_head, [(h, qn, R.ids) for h in range(one.n_q_heads)], chunksize=1)
                dt = time.perf_counter() - t0
                if i >= warmup:
                    tp.append(dt)
                if i == len(qs) - 1:
                    par = np.stack([g[1] for g in sorted(got, key=lambda g: g[0])])
                    assert np.array_equal(par, ref), "the forked oracle must reproduce the single-thread result"
        res.update(sec_all=float(np.mean(tp)), cores_all=workers, nproc=nproc)
    del limiter
    res["desc"] = (f"1 of {spec.batch} sequences x 1 of {spec.n_layers} layers of configs[{spec.config_id}] "
                   f"({spec.contexts[0]} tokens, m={T.seg.m} spans, A={T.seg.A} pool tokens, all {spec.n_q_heads} q heads): "
                   f"oracle route + mixed attention per step, numpy fp64; scaled x{spec.batch} sequences")
    return res


def oracle_sample_subprocess(config: int, steps: int, warmup: int, rho: float):
    """The all-cores leg forks a process pool: it runs in a fresh interpreter that never touched CUDA."""
    import subprocess
    arg = json.dumps({"config": config, "steps": steps, "warmup": warmup, "rho": rho})
    r = subprocess.run([sys.executable, os.path.abspath(__file__), "--oracle-worker", arg], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("oracle worker failed: " + r.stderr[-2000:])
    return json.loads(r.stdout.strip().splitlines()[-1])


def run_reference(args):
    from workloads import get_spec
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    spec = get_spec(args.config)
    res = oracle_sample(spec, args.steps, args.warmup, args.rho)
    sec, desc = res["sec_1"], res["desc"] + "; 1 thread"
    us_layer_step = sec * spec.batch * 1e6
    line = {
        "impl": "reference", "metric": METRIC, "value": us_layer_step, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup,
        # extrapolated like `value`: the arm times 1 sequence x 1 layer per step (see cpu_baseline.sample)
        "ms_per_step": us_layer_step * spec.n_layers / 1e3, "ms_per_step_is": "extrapolated from the sample",
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

    fused, why = eng.sekv_get_path()
    if not args.generic and not fused:
        raise SystemExit("bench.py: the batch does not run on the fused layer kernel: " + why)

    L, Bn, Hq = spec.n_layers, spec.batch, spec.n_q_heads
    out = torch.empty((L, Bn, Hq, 128), dtype=eng.out_dtype, device=dev)
    static_bytes = eng.sekv_static_bytes_per_layer()
    esz = eng.esize
    q_cur = torch.empty((L, Bn, Hq, 128), dtype=eng.st_dtype, device=dev)
    stream_state = {"q": make_queries(spec, 0, dev), "i": 0}

    def next_q(rho):
        """next query of the AR(1) stream (device-side synthesis, outside every timed region)"""
        stream_state["i"] += 1
        stream_state["q"] = next_queries_ar1(spec, stream_state["q"], stream_state["i"], rho)
        return stream_state["q"]

    def step(q):
        q_cur.copy_(q)
        eng.sekv_decode_step(q_cur, spec.top_k, out)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(rho, n_warm, n_steps):
        """n_warm untimed steps of the rho stream (the cache reaches its steady state), then n_steps timed ones:
        device time (CUDA events on the launching stream), statistics of the timed steps only."""
        for _ in range(n_warm):
            step(next_q(rho))
        qs = [next_q(rho) for _ in range(n_steps)]
        barrier()
        eng.sekv_reset_stats()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for q in qs:
            step(q)
        e1.record()
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), world, dev), eng.sekv_get_stats()

    def algo_bytes_of(st, n_layer_steps):
        return n_layer_steps * static_bytes - st["coarse_rows_skipped"] * 2 * 128 * esz + st["factor_bytes_algo"]

    # ---- pinned host -> device bandwidth (what the factor fetch is measured against) -----------------
    pin = torch.empty(256 << 20, dtype=torch.uint8).pin_memory()
    dst = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    best = 0.0
    for _ in range(5):
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(); dst.copy_(pin, non_blocking=True); a1.record(); torch.cuda.synchronize()
        best = max(best, (256 << 20) / (a0.elapsed_time(a1) * 1e-3) / 1e9)
    pcie_h2d_gbs = best
    del pin, dst

    # ---- device-resident timing (value) ---------------------------------------------------------
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.01)
    ms, st = timed(args.rho, max(args.warmup, 3), args.steps)
    sampler.stop_flag = True
    sampler.join(timeout=2)
    layer_steps = args.steps * L
    us_layer_step = replica_us_per_layer_step(ms, args.steps, L, world)   # aggregate over replicas
    algo_bytes = algo_bytes_of(st, layer_steps)
    hbm_gbs = algo_bytes / (ms * 1e-3) / 1e9 * world
    hit = st["cache_hits"] / max(1, st["zoomed_spans"])
    launches = st["kernel_launches"] + args.steps            # + the q staging copy per step

    # ---- end to end through host buffers, same stream, same stationary state --------------------------
    q_host = [next_q(args.rho).cpu().pin_memory() for _ in range(args.e2e_steps)]
    out_host = torch.empty(out.shape, dtype=out.dtype).pin_memory()
    eng.sekv_decode_step_host(q_host[0], spec.top_k, out_host)
    eng.sekv_reset_stats()
    barrier()
    t0 = time.perf_counter()
    for i in range(args.e2e_steps):
        eng.sekv_decode_step_host(q_host[i], spec.top_k, out_host)
    torch.cuda.synchronize()
    e2e_s = max_over_ranks(time.perf_counter() - t0, world, dev)
    st_e = eng.sekv_get_stats()
    fetch_e = (st_e["h2d_bytes"] + st_e["prefetch_h2d_bytes"]) // max(1, args.e2e_steps)
    e2e = {"value": e2e_s * 1e6 / (args.e2e_steps * L) / world, "unit": UNIT,
           "h2d_bytes_per_step": q_host[0].numel() * esz + fetch_e,
           "d2h_bytes_per_step": out_host.numel() * out_host.element_size(),
           "factor_fetch_bytes_per_step": fetch_e, "steps": args.e2e_steps}

    # ---- rho sweep: the miss volume at which the fetch stays hidden ------------------
    sweep = []
    if args.sweep_steps > 0 and world == 1:
        for rho in (1.0, 0.99, 0.9, 0.0):
            ms_r, st_r = timed(rho, 10, args.sweep_steps)
            us_r = ms_r * 1e3 / (args.sweep_steps * L)
            sweep.append({"rho": rho, "value": us_r, "steps": args.sweep_steps,
                          "hit_rate": st_r["cache_hits"] / max(1, st_r["zoomed_spans"]),
                          "demand_h2d_mb_per_step": st_r["h2d_bytes"] / args.sweep_steps / 1e6,
                          "prefetch_h2d_mb_per_step": st_r["prefetch_h2d_bytes"] / args.sweep_steps / 1e6,
                          "pcie_ms_per_step_at_measured_bw": (st_r["h2d_bytes"] + st_r["prefetch_h2d_bytes"]) / args.sweep_steps
                                                             / (pcie_h2d_gbs * 1e9) * 1e3,
                          "ms_per_step": ms_r / args.sweep_steps})
        for e in sweep:
            e["fetch_exposed_us"] = e["value"] - sweep[0]["value"]       # against 100% hits
    value_all_hits = sweep[0]["value"] if sweep else None

    # ---- per-kernel profile (CUDA events around every kernel, eager launches) ----------------------
    eng.sekv_set_profiling(True)
    step(next_q(args.rho))                                   # warm the eager path
    eng.sekv_get_kernel_times()
    eng.sekv_reset_stats()
    for _ in range(args.profile_steps):
        step(next_q(args.rho))
    kt = eng.sekv_get_kernel_times()
    st_p = eng.sekv_get_stats()
    eng.sekv_set_profiling(False)
    tot_kernel_ms = sum(v["ms"] for k, v in kt.items() if k not in ("fetch", "prefetch"))
    peak, peak_src = measured_peaks()
    prof_layer_steps = max(1, st_p["layer_steps"])
    is_fused = bool(kt["fused"]["launches"])
    if is_fused:
        # ONE kernel per layer-step does a1-a7: its algorithmic bytes are the layer-step's
        dom, dom_name = kt["fused"], "fused_layer_kernel (a1-a7: route, plan, pool/coarse/zoom partials, combine)"
        dom_bytes = algo_bytes_of(st_p, prof_layer_steps) / prof_layer_steps
    else:
        dom, dom_name = kt["stage1"], "stage1 kernel (a5: pool + coarse entries)"
        rows_bytes = sum(2 * spec.n_kv_heads * (a + m) * 128 * esz for a, m in zip(eng.pool_per_seq, eng.spans_per_seq))
        dom_bytes = rows_bytes - st_p["coarse_rows_skipped"] * 2 * 128 * esz / prof_layer_steps + Bn * Hq * 128 * esz
    eager_us = max(dom["ms"] * 1e3 / max(1, dom["launches"]), 1e-9)
    if is_fused and world == 1:
        # the layer kernel is the only kernel on the launching stream inside the timed region: its average launch
        # duration over the timed region, CUDA events on that stream, is the step time / layers -- the gaps
        # between the dependent kernels included
        dom_us = ms * 1e3 / layer_steps
        dom_bytes = algo_bytes / layer_steps
        timing = "CUDA events on the launching stream over the timed region (%d steps x %d launches, one graph per step)" % (args.steps, L)
    else:
        dom_us = eager_us
        timing = "CUDA events on the launching stream around every launch, eager launches, %d steps" % args.profile_steps
    traffic, traffic_src = (None, "not quoted for this configuration")
    if is_fused and not args.layers and args.config == 2:
        traffic, traffic_src = ncu_traffic_per_launch()
    roofline = {"bound": "hbm", "kernel": dom_name,
                "achieved": dom_bytes / (dom_us * 1e-6) / 1e9, "peak": peak, "unit": "GB/s",
                "frac": dom_bytes / (dom_us * 1e-6) / 1e9 / peak,
                # dram__bytes_read.sum + dram__bytes_write.sum per launch of the layer kernel from the tracked
                # `ncu --set full` capture (null when the kernel has changed since)
                "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": peak_src,
                "algorithmic_bytes_per_launch": dom_bytes, "avg_launch_us": dom_us,
                "share_of_step_kernel_time": dom["ms"] / max(1e-9, tot_kernel_ms),
                "timing": timing,
                "kernel_us_per_launch_eager": {k: v["ms"] * 1e3 / v["launches"] for k, v in kt.items() if v["launches"]}}

    if rank != 0:
        return
    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        r = oracle_sample_subprocess(args.config, 2, 1, args.rho)
        cpu_baseline = {"value": r["sec_all"] * spec.batch * 1e6, "unit": UNIT, "cores": r["cores_all"], "kind": "oracle",
                        "sample": r["desc"] + "; one forked process per query head over the host cores",
                        "nproc": r.get("nproc"), "value_1_thread": r["sec_1"] * spec.batch * 1e6}
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
                   "path": "fused layer kernel" if fused else "generic multi-kernel path (" + why + ")",
                   "kernels": "generic multi-kernel" if args.generic else "one persistent kernel per layer-step: a team of warps runs route / top-k / cache plan in shared memory, warp workers claim POOL / COARSE / ZOOM / COMBINE items (mma.sync bf16, cp.async K/V ring, TMA bulk copies of factor chunks and routing rows)",
                   "prefetch": cfg.prefetch, "stage1_ctas": n_ctas,
                   "l2": "inputs larger than L2: one step streams %.2f GB of tables (L2 = 126 MB), no flush" % (algo_bytes / args.steps / 1e9),
                   "replicas": "replicas only (no sharding, no collective)" if world > 1 else "single GPU",
                   "setup_s": round(t_setup, 1)},
        "clocks": sampler.result(), "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
        "fetch": {"pcie_h2d_gbs": pcie_h2d_gbs,
                  "demand_h2d_bytes_per_step": st["h2d_bytes"] / args.steps,
                  "prefetch_h2d_bytes_per_step": st["prefetch_h2d_bytes"] / args.steps,
                  "misses_per_step": st["cache_misses"] / args.steps, "zoomed_per_step": st["zoomed_spans"] / args.steps,
                  "value_at_100pct_hits": value_all_hits,
                  "fetch_exposed_us": (us_layer_step - value_all_hits) if value_all_hits is not None else None,
                  "overlap": "demand misses are read by the bulk-copy engine inside the layer kernel; the speculative prefetch of layer l is copied inside layer l+2's kernel, before its dependency wait"},
        "sweep": sweep,
    }
    if cpu_baseline:
        line["cpu_baseline"] = cpu_baseline
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.oracle_worker:
        from workloads import get_spec as _gs
        w = json.loads(a.oracle_worker)
        print(json.dumps(oracle_sample(_gs(w["config"]), w["steps"], w["warmup"], w["rho"], all_cores=True)))
        sys.exit(0)
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
