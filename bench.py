#!/usr/bin/env python
"""bench.py — throughput of the mixed-task vFM forward (fmx_forward_mixed) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload headline|cfg2|cfg3|cfg4|cfg5|sweep5]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...
    python bench.py --impl reference ...        # the fp64 CPU oracle on the host cores

A step is one pass of the whole hot path (S1 task sort .. S6 output scatter) over one synthetic mixed batch.
BASELINE.json's metric is "mixed-task samples/s per B200 and % of bf16 tensor peak vs #co-batched tasks": it is quoted on
configs[4] (the task-count sweep on the cfg2 backbone, batch 512).  The default workload ("headline") is therefore
configs[4] at 92 co-batched tasks, task ids Zipf(0.8); the SAME run also measures the single-task batch and the adapter-free
batch of the same size (`vs_single_task`, `vs_adapter_free`: north_star's "within 10 % of a single-task batch") and the three
other full-size configs (`per_config`: cfg2 / cfg3 / cfg4 with value, ms_per_step, % of peak and per-GEMM-family TFLOP/s).
Rank 0 prints ONE JSON line.

  value      whole-job samples/s, inputs resident in HBM, CUDA events around every step on the launching stream, L2 flushed
             (256 MB memset) between steps outside the events.  The step is the C-ABI call fmx_forward_mixed on a non-default
             stream; the call is identical every step, so the library replays its cached CUDA graph (--no-graph: plain
             launches).  `no_graph` gives the same K steps as plain kernel launches right after.
  breakdown  a third pass of K steps, plain launches with CUDA events around EVERY kernel launch (on the launching stream):
             per-family launches and ms per step, plus `ms_per_step` of that pass - the family times are parts of it, so
             their sum is <= it.
  roofline   the tcgen05 pair GEMM (all four projection families), from the SAME pass as `breakdown`: algorithmic FLOPs per
             launch / average launch duration.  avg_launch_ms x launches_per_step = the GEMM families' ms in `breakdown`.
             `peak` is MEASURED_PEAKS.json's burst bf16 figure unless the SM clock sampled during the pass sat at the
             sustained level (then the sustained figure); both fractions are printed.
  e2e        the same metric through fmx_forward_mixed_host: pinned HOST inputs -> device, forward, outputs -> HOST, inside the
             timed region (wall clock around the synchronous calls).
  cpu_baseline  the oracle (numpy fp64, as it stands) on a bounded sample of the same workload.

Multi-GPU is replicas only: every rank runs the same batch shape on its own GPU, no data-path collective;
value = units of all ranks / max-over-ranks time; scaling "weak".
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "mixed-task samples/s per B200 and % of bf16 tensor peak vs #co-batched tasks"
GEMM_FAMILIES = ("gemm_qkv", "gemm_o", "gemm_ffn_in", "gemm_ffn_out")
HEADLINE = dict(tasks=92, dist="zipf0.8")
WORKLOAD_NAMES = {
    "headline": "configs[4]: task-count/skew sweep on the cfg2 backbone (24L d1024 FFN4096 ReLU RMSNorm, T5-large-encoder-shaped), "
                "batch 512 x 64 tokens, 92 co-batched tasks (every task present), LoRA rank {4,8,16,32,64} per task on q/k/v/o, "
                "forecast (flatten->96) / mean-pool heads alternating, task ids Zipf(0.8)",
    "cfg2": "configs[1]: T5-large-encoder-shaped time-series backbone (24L d1024 FFN4096 ReLU RMSNorm), batch 256 x 64 tokens, "
            "10 tasks, rank-8 LoRA on q/k/v/o, forecast (flatten->96) or mean-pool heads, task ids Zipf(1.1)",
    "cfg3": "configs[2]: ViT-L/14-shaped vision backbone, batch 128 x 257 tokens, 32 tasks, rank 8/16 LoRA on q/k/v/o, CLS heads",
    "cfg4": "configs[3]: decoder-only LM prefill (28L d1536 GQA 12/2 SwiGLU 8960 RoPE causal), batch 64, lengths U[64,1024], "
            "92 tasks, LoRA rank {4..64} on 7 targets, last-token heads, task ids Zipf(1.0)",
    "cfg5": "configs[4]: task-count/skew sweep point on the cfg2 backbone, batch 512",
}


def gemm_traffic(workload):
    """DRAM bytes per launch of the pair GEMM (dram__bytes_read.sum + dram__bytes_write.sum averaged over the GEMM launches of
    one layer, from the committed `ncu --set full` capture summary profiles/gemm_traffic.csv), or None for a workload without one."""
    p = os.path.join(ROOT, "profiles", "gemm_traffic.csv")
    if not os.path.exists(p):
        return None
    for line in open(p):
        f = line.strip().split(",")
        if len(f) >= 3 and f[0] == workload:
            return float(f[2])
    return None


def peaks():
    """Measured roofline denominators (driver-written), else the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(source="measured", hbm_gbs=float(d["hbm_gbs"]), bf16_tflops=float(d["bf16_tflops"]),
                    bf16_tflops_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    sustained_sm_mhz=(d.get("clocks_under_load") or {}).get("sm_mhz_median"))
    return dict(source="fallback (B200_PROFILING.md)", hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, sustained_sm_mhz=None)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (profiling recipe)."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "20"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None
        self.t0 = self.t1 = None

    def start(self):
        self.t0 = time.time()

    def stop(self):
        self.t1 = time.time()

    def result(self):
        import datetime
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        inside, allr = [], []
        for r in rows:
            if len(r) < 8:
                continue
            try:
                ts = datetime.datetime.strptime(r[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                rec = (ts, float(r[1]), float(r[2]), float(r[3]), r[4:8])
            except ValueError:
                continue
            allr.append(rec)
            if self.t0 - 0.01 <= ts <= self.t1 + 0.01:
                inside.append(rec)
        use = inside or allr
        if not use:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(x[1] for x in use)
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = [n for k, n in enumerate(names) if any(x[4][k].strip().lower().startswith("active") for x in use)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": use[0][2], "power_w_max": max(x[3] for x in use), "samples": len(use),
                "samples_in_timed_region": len(inside), "reasons": reasons}


def build_workload(args):
    from fmx_workloads import make_workload
    if args.workload == "headline":
        return make_workload("cfg5", n_tasks=HEADLINE["tasks"], dist=HEADLINE["dist"])
    if args.workload == "cfg5":
        return make_workload("cfg5", n_tasks=args.tasks, dist=args.dist, adapters=not args.no_adapters, mlp_hidden=args.mlp_hidden, enc_channels=args.enc_channels,
                             rel_bias=args.rel_bias)
    if args.workload == "decode":                       # (the reference arm on this workload times the cfg4 prefill oracle)
        return make_workload("cfg4")
    return make_workload(args.workload, mlp_hidden=args.mlp_hidden, enc_channels=args.enc_channels, rel_bias=args.rel_bias)


# ------------------------------------------------------------------------------------- the oracle legs
def oracle_time(wl, idx, get=None, warm=True):
    """Seconds the oracle (as it stands) takes for requests idx; weights widened to fp64 beforehand."""
    from oracle import from_workload as G
    from oracle.vfm_forward import forward_requests
    get = get or G.make_get(wl, max_cached_bytes=12 << 30)
    if warm:
        for name in wl.backbone_tensor_names():
            get(name)
        for t in sorted({int(wl.task_ids[i]) for i in idx}):
            for name in wl.task_tensor_names(t):
                get(name)
    inputs = G.request_inputs(wl, idx)
    bb, tasks = G.bb_dict(wl), G.task_dicts(wl)
    t0 = time.perf_counter()
    out = forward_requests(bb, get, tasks, [int(wl.task_ids[i]) for i in idx], inputs)
    return time.perf_counter() - t0, out


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 0) for p in threadpool_info() if p.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return os.cpu_count()


def run_reference(args):
    """--impl reference: the oracle on the host cores; each step = a bounded sample of the workload."""
    from paper_2606_09643_b200 import replicas
    rank, _, world = replicas.env_world()
    if rank != 0:
        return 0
    wl = build_workload(args)
    n = min(args.ref_sample, wl.n_req)
    times = []
    from oracle import from_workload as G
    get = G.make_get(wl, max_cached_bytes=12 << 30)
    for s in range(args.warmup + args.steps):
        idx = [(s * n + j) % wl.n_req for j in range(n)]
        dt, _ = oracle_time(wl, idx, get=get, warm=True)
        if s >= args.warmup:
            times.append(dt)
    total = sum(times)
    v = n * len(times) / total
    line = {"metric": METRIC, "value": v, "unit": "samples/s", "impl": "reference", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAMES.get(args.workload, args.workload), "sample": f"{n} requests per step"},
            "cpu_baseline": {"value": v, "unit": "samples/s", "cores": blas_threads(), "kind": "oracle",
                             "sample": f"{n} of {wl.n_req} requests per step, {len(times)} timed steps, weights widened to fp64 outside the clock"},
            "e2e": {"value": v, "unit": "samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------- the CUDA arm
def bfq_host_cost(wl):
    """S0: the host-side BFQ batch builder on a backlog shaped like the workload (its task-id mix and lengths, weights 1..3):
    enqueue (Eq. 1-2 tags), next_batch (order by S, extend to B_max) and complete (Eq. 3 retag), timed through the C ABI
    from Python, so the figure includes ~1 us of ctypes per enqueue.  Paper: 0.35 ms per request on its host."""
    import numpy as np
    from paper_2606_09643_b200.binding import Bfq
    B, T = wl.n_req, len(wl.tasks)
    rounds = 8
    q = Bfq(T, B, [1.0 + 0.04 * b for b in range(B)])
    for t in range(T):
        q.set_task(t, 1.0 + (t % 3))
    ids = np.tile(np.asarray(wl.task_ids, dtype=np.int64), rounds)
    lens = np.tile(np.asarray(wl.lengths, dtype=np.int64), rounds)
    t0 = time.perf_counter()
    for i in range(len(ids)):
        q.enqueue(int(ids[i]), i, int(lens[i]), 0.001 * i)
    t1 = time.perf_counter()
    served = 0
    for r in range(rounds):
        b_ids, _, _ = q.next_batch(10.0 + r, B)
        q.complete(1.0 + 0.04 * len(b_ids))
        served += len(b_ids)
    t2 = time.perf_counter()
    return {"us_per_request": round((t2 - t0) * 1e6 / max(served, 1), 3), "enqueue_us_per_request": round((t1 - t0) * 1e6 / len(ids), 3),
            "batch_build_us_per_batch": round((t2 - t1) * 1e6 / rounds, 1), "requests": int(served), "batch": B, "tasks": T,
            "how": "fmx_bfq_enqueue / next_batch / complete through ctypes on the host; paper: 350 us per request (P:L418, its host)"}


def timed_steps(sess, torch, steps, flush):
    """K steps, each bracketed by its own CUDA events on the launching stream; L2 flushed between
    steps outside the events.  Returns total ms."""
    e0 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    e1 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    for i in range(steps):
        if flush is not None:
            flush.zero_()
        e0[i].record()
        sess.forward()
        e1[i].record()
    torch.cuda.synchronize()
    return sum(a.elapsed_time(b) for a, b in zip(e0, e1))


def measure(args, wl, rank, local_rank, world, full=True, steps=None, weights_from=None, label=None):
    """Everything runs on one non-default stream: fmx_forward_mixed replays its cached CUDA graph there (FMX_OPT_GRAPH)."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libfmx has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    with torch.cuda.stream(torch.cuda.Stream(torch.device("cuda", local_rank))):
        return _measure(args, wl, rank, local_rank, world, full, steps or args.steps, weights_from, label or args.workload)


def _measure(args, wl, rank, local_rank, world, full, steps, weights_from, label):
    """One workload.  full = the headline treatment (e2e, BFQ cost, task lifecycle, oracle baseline); otherwise the three timed
    passes only.  Returns (line, session) - the session keeps the device weights alive for a run that shares the backbone."""
    import numpy as np
    import torch
    from paper_2606_09643_b200 import accounting, replicas
    from paper_2606_09643_b200.session import Session

    dev = torch.device("cuda", local_rank)
    pk = peaks()
    sess = Session(wl, device=local_rank, weights_from=weights_from)
    for kv in args.opt:
        name, val = kv.split("=")
        sess.fmx.set_option(name, int(val))
    sess.upload_inputs()
    fl = accounting.flops(wl)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if not args.no_flush else None
    B = wl.n_req
    warm = max(args.warmup, 3)

    sampler = ClockSampler(local_rank) if rank == 0 else None
    sess.fmx.set_option("graph", 0 if args.no_graph else 1)
    for _ in range(warm):
        if flush is not None:
            flush.zero_()
        sess.forward()
    torch.cuda.synchronize()
    launches_per_step = sess.fmx.last_launch_count()

    # ---- pass 1, the timed region: exactly K steps through fmx_forward_mixed (graph replay: the call is identical every step)
    replicas.barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    replays0 = sess.fmx.graph_replays()
    ms_total = timed_steps(sess, torch, steps, flush)
    torch.cuda.synchronize()
    replicas.barrier()
    graph_steps = sess.fmx.graph_replays() - replays0
    ms_max = replicas.max_over_ranks(ms_total, dev if world > 1 else None)
    value = replicas.whole_job_throughput(B, steps, ms_max, world)

    # ---- pass 2: the same K steps as plain kernel launches (what a serving loop whose batch changes every step gets)
    sess.fmx.set_option("graph", 0)
    sess.forward()
    ms_plain = timed_steps(sess, torch, steps, flush)
    ms_plain_max = replicas.max_over_ranks(ms_plain, dev if world > 1 else None)

    # ---- pass 3: K steps, plain launches, CUDA events around EVERY launch: breakdown by family + the GEMM roofline
    breakdown, roof, ms_prof = {}, None, 0.0
    if not args.no_kernel_events:
        sess.fmx.profile_select(None)
        sess.fmx.profile_enable(True)
        ms_prof = timed_steps(sess, torch, steps, flush)
        torch.cuda.synchronize()
        fam = sess.fmx.profile_read()
        sess.fmx.profile_enable(False)
        breakdown = {k: {"launches_per_step": n // steps, "ms_per_step": round(ms / steps, 4)} for k, (n, ms) in fam.items() if n}
    if sampler:
        sampler.stop()
    clocks = sampler.result() if sampler else None
    sess.fmx.set_option("graph", 0 if args.no_graph else 1)

    # ---- roofline of the dominant kernel (tcgen05 pair GEMM, all four projection families), from pass 3 ----
    if breakdown:
        n_l = sum(fam[f][0] for f in GEMM_FAMILIES)
        ms_g = sum(fam[f][1] for f in GEMM_FAMILIES)
        fused = "lora_shrink" not in breakdown      # the LoRA shrink ran as work items of the GEMM launches (no shrink family)
        fam_fl = {f: fl["families"][f] + (fl["shrink_families"][f] if fused else 0.0) for f in GEMM_FAMILIES}
        fl_g = sum(fam_fl.values())                                     # per forward
        avg_ms = ms_g / max(n_l, 1)
        flops_per_launch = fl_g / accounting.gemm_launches_per_forward(wl)
        achieved = flops_per_launch / (avg_ms * 1e-3) / 1e12
        # which measured peak applies: the burst figure, unless the SM clock during these passes sat at the level the
        # driver recorded for its 4-second sustained matmul (MEASURED_PEAKS.json clocks_under_load)
        sm = (clocks or {}).get("sm_mhz")
        sus = pk.get("sustained_sm_mhz")
        at_sustained = bool(sm and sus and sm <= 1.10 * sus)
        peak = pk["bf16_tflops_sustained"] if at_sustained else pk["bf16_tflops"]
        roof = {"kernel": "fmx::pair_gemm_kernel<256> (tcgen05 cta_group::2 / TMEM / TMA, fused LoRA expand)", "bound": "tensor",
                "achieved": round(achieved, 2), "peak": peak, "unit": "TFLOP/s", "frac": round(achieved / peak, 4),
                "peak_kind": f"{pk['source']} {'sustained' if at_sustained else 'burst'} bf16 (median SM clock in the passes {sm} MHz; "
                             f"the driver's sustained matmul ran at {sus} MHz)",
                "frac_of_burst_peak": round(achieved / pk["bf16_tflops"], 4),
                "frac_of_sustained_peak": round(achieved / pk["bf16_tflops_sustained"], 4),
                "traffic": gemm_traffic(label), "traffic_unit": "DRAM bytes per launch (ncu --set full, cold cache; profiles/gemm_traffic.csv)",
                "flops_per_launch": flops_per_launch, "avg_launch_ms": round(avg_ms, 5), "launches_per_step": n_l // steps,
                "gemm_ms_per_step": round(ms_g / steps, 4), "share_of_step": round(ms_g / ms_prof, 4),
                "timed_in": "the `breakdown` pass (plain launches, events around every launch; `breakdown.ms_per_step` is that pass's step time)",
                "fused_lora_shrink": fused,
                "per_family_tflops": {f: round(fam_fl[f] * steps / (fam[f][1] * 1e-3) / 1e12, 1) for f in GEMM_FAMILIES if fam[f][1] > 0}}
        other = sum(v["ms_per_step"] for k, v in breakdown.items() if k not in GEMM_FAMILIES)
        breakdown = {"ms_per_step": round(ms_prof / steps, 4), "sum_of_families_ms": round(ms_g / steps + other, 4), "families": breakdown}

    tf = fl["total"] * world * steps / (ms_max * 1e-3) / 1e12
    line = {"metric": METRIC, "value": round(value, 2), "unit": "samples/s", "n_gpus": world, "steps": steps,
            "warmup": warm, "ms_per_step": round(ms_max / steps, 4), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAMES.get(label, label), "requests": B, "tokens": wl.n_tokens,
                       "tasks": len(wl.tasks), "tasks_in_batch": int(len(set(wl.task_ids.tolist()))), "dist": wl.notes.get("dist"),
                       "l2": "flushed (256 MB memset) between steps, outside the per-step events" if flush is not None else "no flush",
                       "accumulate": "fp32 (TMEM), fp32 residual stream", "replicas": world, **({"options": args.opt} if args.opt else {}),
                       **({"mlp_heads_hidden": args.mlp_hidden} if args.mlp_hidden else {}), **({"input_encoder_channels": args.enc_channels} if args.enc_channels else {}),
                       "launch": f"CUDA graph replay inside fmx_forward_mixed on {graph_steps} of {steps} timed steps" if graph_steps else "plain kernel launches"},
            "no_graph": {"value": round(replicas.whole_job_throughput(B, steps, ms_plain_max, world), 2), "ms_per_step": round(ms_plain_max / steps, 4),
                         "what": "the same K steps as plain kernel launches (FMX_OPT_GRAPH off), timed the same way"},
            "pct_bf16_tensor_peak": {"of_burst": round(100 * tf / pk["bf16_tflops"], 2), "of_sustained": round(100 * tf / pk["bf16_tflops_sustained"], 2),
                                     "achieved_tflops": round(tf, 1), "algorithmic_tflop_per_step": round(fl["total"] / 1e12, 4), "peaks": pk["source"]},
            "gpu_launches": launches_per_step * steps, "launches_per_step": launches_per_step,
            "clocks": clocks, "roofline": roof, "breakdown": breakdown}
    if not full:
        return line, sess

    # ---- e2e through the host-buffer entry point ----
    packed = wl.packed_inputs()
    host_in = torch.from_numpy(packed.view(np.int16) if packed.dtype == np.uint16 else packed).pin_memory()
    ids = np.array([sess.task_ids_of[int(t)] for t in wl.task_ids], dtype=np.int32)
    off = sess.fmx.output_layout(ids)
    host_out = torch.empty(int(off[-1]), dtype=torch.float32).pin_memory()
    sess.ensure_host_workspace(packed.nbytes, int(off[-1]))
    stream = torch.cuda.current_stream().cuda_stream
    e2e_steps = max(3, min(steps, 20))
    for _ in range(2):
        sess.fmx.forward_mixed_host(sess.bb, host_in.data_ptr(), packed.nbytes, ids, wl.lengths, host_out.data_ptr(), sess.ws_ptr,
                                    sess.ws_bytes, stream)
    replicas.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        if flush is not None:
            flush.zero_()
        sess.fmx.forward_mixed_host(sess.bb, host_in.data_ptr(), packed.nbytes, ids, wl.lengths, host_out.data_ptr(), sess.ws_ptr,
                                    sess.ws_bytes, stream)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_ms_max = replicas.max_over_ranks(e2e_s * 1e3, dev if world > 1 else None)
    line["e2e"] = {"value": round(replicas.whole_job_throughput(B, e2e_steps, e2e_ms_max, world), 2), "unit": "samples/s",
                   "h2d_bytes_per_step": int(packed.nbytes + 8 * B), "d2h_bytes_per_step": int(off[-1]) * 4, "steps": e2e_steps,
                   "includes": "pinned host -> device copy of the packed inputs, ids / lengths upload, forward, device -> host copy of all outputs, "
                               "stream synchronise; L2 flush memset between steps"}
    if rank == 0:
        line["bfq"] = bfq_host_cost(wl)
        # R2 lifecycle decoupling: take one task off the live context and put it back (the backbone and the other tasks stay)
        un_ms, reg_ms = sess.task_lifecycle_ms(len(wl.tasks) - 1)
        reg_busy_ms, fwd_ms, _ = sess.register_while_serving_ms(len(wl.tasks) - 1, n_forwards=5)
        un_busy_ms, fwd2_ms = sess.unregister_while_serving_ms(len(wl.tasks) - 1, n_forwards=5)
        line["task_lifecycle"] = {"unregister_ms": round(un_ms, 3), "register_ms": round(reg_ms, 3), "task": len(wl.tasks) - 1,
                                  "register_ms_with_5_forwards_queued": round(reg_busy_ms, 3), "those_5_forwards_ms": round(fwd_ms, 2),
                                  "unregister_ms_with_5_forwards_queued": round(un_busy_ms, 3), "those_forwards_ms": round(fwd2_ms, 2),
                                  "how": "fmx_unregister_task / fmx_register_task on the live context, tensors already on the device; neither "
                                         "synchronises the device; paper: 25 ms task load vs 5737 ms backbone load for MOMENT-Large on its T4 host (P:L387)"}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n = min(args.cpu_sample, B)
        idx = list(range(n))
        dt, ref = oracle_time(wl, idx)
        # the same requests through the CUDA path: parity of the timed sample, reported not asserted
        y = sess.forward_numpy()
        mx = max(float(np.abs(y[i] - r).max()) for i, r in zip(idx, ref))
        line["cpu_baseline"] = {"value": round(n / dt, 4), "unit": "samples/s", "cores": blas_threads(), "kind": "oracle",
                                "sample": f"first {n} of {B} requests, one by one in numpy fp64 ({dt:.1f} s; weights widened before the clock)",
                                "max_abs_vs_cuda": mx}
    return line, sess


def measure_decode(sess, wl, steps=16, warm=3):
    """NEXT-3: token decode with a KV cache on the decoder backbone, every request of the batch advancing one
    token per iteration (mixed tasks, segmented LoRA).  Prefill of the prompts (cut so that the cache has room), then `steps`
    timed iterations with CUDA events; the step's greedy tokens feed the next step on the device.  A decode iteration is
    bound by HBM: it reads every backbone / LM-head weight once plus the cached k / v of every sequence."""
    import numpy as np
    import torch
    bb = wl.bb
    B = wl.n_req
    room = steps + warm + 4
    lens = np.minimum(wl.lengths, bb.max_seq - room).astype(np.int32)
    toks = np.concatenate([wl.request_input(i)[:lens[i]] for i in range(B)]).astype(np.int32)
    sess.enable_decode(n_slots=B, max_req=B)
    slots = np.arange(B, dtype=np.int32)
    sess.prefill(toks, wl.task_ids, lens, slots, with_heads=False)
    pos = lens.copy()
    ptr = sess.next_dev.data_ptr()
    for _ in range(warm):
        sess.decode_step(ptr, wl.task_ids, slots, pos, want_scores=False, sync=False)
        pos += 1
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kv_rows = 0
    e0.record()
    for _ in range(steps):
        sess.decode_step(ptr, wl.task_ids, slots, pos, want_scores=False, sync=False)
        kv_rows += int(pos.sum()) + B
        pos += 1
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    launches = sess.fmx.last_launch_count()
    sess.fmx.profile_select(None)
    sess.fmx.profile_enable(True)
    for _ in range(2):
        sess.decode_step(ptr, wl.task_ids, slots, pos, want_scores=False, sync=False)
        pos += 1
    fam = sess.fmx.profile_read()
    sess.fmx.profile_enable(False)
    families = {k: {"launches_per_step": n // 2, "ms_per_step": round(t / 2, 4)} for k, (n, t) in fam.items() if n}
    per_layer = 2 * (bb.d_model * (bb.d_q + 2 * bb.d_kv) + bb.d_q * bb.d_model + (3 if bb.act == "swiglu" else 2) * bb.d_model * bb.d_ffn)
    weight_bytes = bb.n_layers * per_layer + 2 * bb.vocab * bb.d_model          # backbone matrices + LM head, bf16
    kv_bytes = kv_rows / steps * bb.n_layers * 2 * bb.d_kv * 2
    from fmx_workloads.spec import target_dims
    adapter_bytes = 0                                                            # A and B of every adapter of the DISTINCT tasks in the batch, once
    for t in sorted(set(int(x) for x in wl.task_ids)):
        for ad in wl.tasks[t].adapters:
            d_in, d_out = target_dims(bb, ad.target)
            adapter_bytes += bb.n_layers * 2 * ad.rank * (d_in + d_out)
    pk = peaks()
    total = weight_bytes + kv_bytes + adapter_bytes
    gbs = total / (ms * 1e-3) / 1e9
    return {"what": "fmx_decode_step: one new token for each of the batch's sequences per iteration, KV cache, mixed tasks, greedy tokens fed back on the device",
            "requests": B, "tokens_per_s": round(B / (ms * 1e-3), 1), "ms_per_step": round(ms, 4), "steps": steps, "launches_per_step": launches,
            "mean_cached_tokens": round(kv_rows / steps / B, 1), "distinct_tasks": len(set(int(x) for x in wl.task_ids)), "families": families,
            "roofline": {"bound": "hbm", "achieved": round(gbs, 1), "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": round(gbs / pk["hbm_gbs"], 4),
                         "bytes_per_step": int(total),
                         "bytes": {"backbone_and_lm_head": int(weight_bytes), "kv_cache": int(kv_bytes), "lora_adapters": int(adapter_bytes)},
                         "note": "algorithmic bytes = every backbone and LM-head weight once + the cached k / v rows read + the LoRA matrices of the "
                                 "distinct tasks in the batch once (unpadded ranks).  The iteration is bound by kernel count and dependent memory "
                                 "latency (17 launches per layer), not by bandwidth; families are timed with plain launches and an event pair per "
                                 "launch, so their sum exceeds the graph-replayed iteration"}}


def light(line):
    """The per-config / reference summary of a measured line."""
    r = line["roofline"] or {}
    return {"workload": line["config"]["workload"], "requests": line["config"]["requests"], "tokens": line["config"]["tokens"],
            "tasks_in_batch": line["config"]["tasks_in_batch"], "value": line["value"], "unit": "samples/s", "ms_per_step": line["ms_per_step"],
            "steps": line["steps"], "no_graph_ms_per_step": line["no_graph"]["ms_per_step"],
            "pct_of_burst": line["pct_bf16_tensor_peak"]["of_burst"], "pct_of_sustained": line["pct_bf16_tensor_peak"]["of_sustained"],
            "achieved_tflops": line["pct_bf16_tensor_peak"]["achieved_tflops"],
            "gemm_tflops": r.get("achieved"), "gemm_frac_of_burst": r.get("frac_of_burst_peak"), "per_family_tflops": r.get("per_family_tflops"),
            "family_ms_per_step": {k: v["ms_per_step"] for k, v in (line["breakdown"] or {}).get("families", {}).items()},
            "sm_mhz": (line["clocks"] or {}).get("sm_mhz"), "clock_reasons": (line["clocks"] or {}).get("reasons")}


def run_headline(args, rank, local_rank, world):
    """The default run: BASELINE.json's metric on its own configuration (configs[4], 92 co-batched tasks) plus, in the same
    process, its two reference batches (single task / adapter-free, same size, same backbone weights on the device) and the
    other full-size configs."""
    from fmx_workloads import make_workload
    short = max(5, min(args.steps, 10))
    wl = make_workload("cfg5", n_tasks=HEADLINE["tasks"], dist=HEADLINE["dist"])
    line, sess = measure(args, wl, rank, local_rank, world, full=True, label="headline")
    refs = {}
    for key, kw in (("single_task", dict(n_tasks=1, dist="uniform")), ("adapter_free", dict(n_tasks=1, dist="uniform", adapters=False))):
        l2, s2 = measure(args, make_workload("cfg5", **kw), rank, local_rank, world, full=False, weights_from=sess, label=f"cfg5 {key}")
        refs[key] = light(l2)
        s2.fmx.destroy()
    sess.fmx.destroy()
    del sess
    line["vs_single_task"] = round(line["value"] / refs["single_task"]["value"], 4)
    line["vs_adapter_free"] = round(line["value"] / refs["adapter_free"]["value"], 4)
    line["references"] = {**refs, "note": "same batch size (512) and backbone weights; single_task: all requests on one task with a rank-16 LoRA "
                                           "on q/k/v/o and a forecast head (reading 19); adapter_free: one head-only task.  north_star target: "
                                           "vs_single_task >= 0.90"}
    per = {}
    if world > 1:
        line["config"]["per_config"] = "skipped under torchrun (N > 1): the scaling run needs the headline only; run N = 1 for the other configs"
    elif not args.no_per_config:
        for cfg, st in (("cfg2", short), ("cfg3", short), ("cfg4", max(3, short // 2))):
            wl2 = make_workload(cfg)
            l2, s2 = measure(args, wl2, rank, local_rank, world, full=False, steps=st, label=cfg)
            per[cfg] = light(l2)
            if cfg == "cfg4" and rank == 0:
                per[cfg]["decode"] = measure_decode(s2, wl2)
            s2.fmx.destroy()
            del s2
    line["per_config"] = per
    return line


def run_decode(args, rank, local_rank, world):
    """NEXT-3 only: decode iterations on the cfg4 backbone (64 sequences, 92 tasks); the line's value is tokens per second."""
    import torch
    from fmx_workloads import make_workload
    from paper_2606_09643_b200.session import Session
    torch.cuda.set_device(local_rank)
    wl = make_workload("cfg4")
    with torch.cuda.stream(torch.cuda.Stream(torch.device("cuda", local_rank))):
        sess = Session(wl, device=local_rank)
        for k, v in (o.split("=") for o in args.opt):
            sess.fmx.set_option(k, int(v))
        d = measure_decode(sess, wl, steps=args.steps, warm=max(3, args.warmup))
        sess.fmx.destroy()
    return {"metric": "decode tokens per second, mixed-task batch", "value": d["tokens_per_s"], "unit": "tokens/s", "n_gpus": 1, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": d["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16", "data": "synthetic", "config": {"workload": "cfg4 decode: 64 sequences, 92 registered tasks, prompts cut to leave room in the cache",
                                                             "options": args.opt}, "gpu_launches": d["launches_per_step"] * args.steps,
            "roofline": d["roofline"], "decode": d}


def run_sweep5(args, rank, local_rank, world):
    """BASELINE.json configs[4] in full: T x distribution -> samples/s, ratio to the single-task batch and to the adapter-free one."""
    from fmx_workloads import make_workload
    rows, ref, keep, last = [], {}, None, None
    for T, dist, ad in [(1, "uniform", True), (1, "uniform", False)] + [(T, d, True) for T in (4, 16, 48, 92)
                                                                         for d in ("uniform", "zipf0.8", "zipf1.5")]:
        wl = make_workload("cfg5", n_tasks=T, dist=dist, adapters=ad)
        line, sess = measure(args, wl, rank, local_rank, world, full=False, weights_from=keep, label=f"cfg5 T={T} {dist}")
        if keep is None:
            keep = sess                       # later points reuse the backbone weights on the device
        else:
            sess.fmx.destroy()
        key = "single_task" if (T == 1 and ad) else ("adapter_free" if T == 1 else None)
        if key:
            ref[key] = line["value"]
        rows.append({"tasks": T, "dist": dist, "adapters": ad, "samples_per_s": line["value"], "ms_per_step": line["ms_per_step"],
                     "no_graph_ms_per_step": line["no_graph"]["ms_per_step"],
                     "pct_peak_burst": line["pct_bf16_tensor_peak"]["of_burst"],
                     "vs_single_task": round(line["value"] / ref["single_task"], 4) if "single_task" in ref else None,
                     "vs_adapter_free": round(line["value"] / ref["adapter_free"], 4) if "adapter_free" in ref else None,
                     "gemm_frac_of_burst": line["roofline"]["frac_of_burst_peak"] if line["roofline"] else None})
        last = line
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    if rank == 0:
        json.dump(rows, open(os.path.join(ROOT, "gpurun_out", "sweep5.json"), "w"), indent=1)
    last["config"]["workload"] = "configs[4] sweep; this line = T=92, Zipf(1.5); full table in `sweep` (also written to gpurun_out/sweep5.json)"
    last["sweep"] = rows
    return last


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="fmx", choices=["fmx", "reference"])
    ap.add_argument("--workload", default="headline", choices=["headline", "cfg2", "cfg3", "cfg4", "cfg5", "sweep5", "decode"],
                    help="headline (default): configs[4] at 92 tasks + its single-task / adapter-free references + per_config cfg2 / cfg3 / cfg4")
    ap.add_argument("--no-per-config", action="store_true", help="headline: skip the cfg2 / cfg3 / cfg4 lines")
    ap.add_argument("--tasks", type=int, default=92, help="cfg5: number of co-batched tasks")
    ap.add_argument("--dist", default="zipf0.8", choices=["uniform", "zipf0.8", "zipf1.5"])
    ap.add_argument("--no-adapters", action="store_true", help="cfg5: head-only tasks (adapter-free reference)")
    ap.add_argument("--enc-channels", type=int, default=0, help="NEXT-1 variant: every other task brings this many input channels and a channel combiner (cfg2 / cfg5)")
    ap.add_argument("--mlp-hidden", type=int, default=0, help="NEXT-1 variant: pooled heads become MLP decoder heads of this hidden width")
    ap.add_argument("--rel-bias", action="store_true", help="NEXT-4 variant: the backbone carries a T5-style relative-position bias (32 buckets, max distance 128)")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="fmx_set_option experiment knob (csrc/fmx_internal.h), e.g. --opt attention_impl=3; recorded in config.options")
    ap.add_argument("--no-flush", action="store_true")
    ap.add_argument("--no-graph", action="store_true", help="plain kernel launches in the timed region (FMX_OPT_GRAPH off)")
    ap.add_argument("--no-kernel-events", action="store_true", help="no per-GEMM events inside the timed region (no roofline)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample", type=int, default=24, help="requests the oracle is timed on (cpu_baseline)")
    ap.add_argument("--ref-sample", type=int, default=4, help="--impl reference: requests per step")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    from paper_2606_09643_b200 import replicas
    rank, local_rank, world = replicas.init()
    if world != args.gpus and rank == 0:
        sys.stderr.write(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; launch N>1 with torch.distributed.run\n")
    if args.workload == "sweep5":
        line = run_sweep5(args, rank, local_rank, world)
    elif args.workload == "headline":
        line = run_headline(args, rank, local_rank, world)
    elif args.workload == "decode":
        line = run_decode(args, rank, local_rank, world)
    else:
        wl = build_workload(args)
        line, sess = measure(args, wl, rank, local_rank, world)
        if args.workload == "cfg4" and rank == 0:
            line["decode"] = measure_decode(sess, wl)
        sess.fmx.destroy()
    if rank == 0:
        print(json.dumps(line))
    replicas.finalize()
    return 0


if __name__ == "__main__":
    sys.exit(main())
