#!/usr/bin/env python
"""bench.py -- NACL encoding-phase eviction throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

`--gpus N` with N > 1 and no torchrun environment re-launches itself under torch.distributed.run with N ranks.

One *step* = one pass of the whole hot path over one batch
of synthetic prompts: every layer of the workload is evicted once through the C ABI
(`nacl_evict`, include/nacl_evict.h).  Default workload: BASELINE.json configs[3] -- the L=32k
configuration the metric is quoted on (Mistral-7B-shaped GQA, batch 4, 32 layers).  Each layer has
its own K/V/Q and output buffers (16 GiB of K/V in total), so every timed call reads inputs that
are cold in the 126 MB L2.

Prints ONE JSON line (rank 0).  `value` = KV GB/s = algorithmic bytes / device time, with
algorithmic bytes per layer = B*Hkv*d*e*(L + 4C): K read once for scoring + C rows of K and of V
read and written (BASELINE.json north star).

Multi-GPU (torchrun): the path shards over independent batch elements with no data-path
collective; every rank evicts its own batch of prompts ("weak" scaling),
`value` = bytes of all ranks / max-over-ranks device time.

`--impl reference`: there is no reference implementation to install (the reference is a paper);
per the task's tier framing this arm times the fp64 CPU oracle (oracle/) on the host cores,
each step a bounded sample (one layer) of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

from paper_2408_03675_b200 import CONFIGS  # noqa: E402
from paper_2408_03675_b200 import dist as nacl_dist  # noqa: E402
from paper_2408_03675_b200.inputs import make_layer_inputs  # noqa: E402

METRIC = "eviction throughput per layer at L=32k (KV GB/s)"
UNIT = "GB/s"


def load_peaks() -> dict:
    """Measured roofline denominators (driver-written); the profiling guide's fallback otherwise."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        p["source"] = "measured (MEASURED_PEAKS.json)"
        return p
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0,
            "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """Samples SM clock / throttle reasons with nvidia-smi while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines: list[str] = []
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        if self.thread is not None:
            self.thread.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ workload
def workload_desc(cfg, layers, world) -> dict:
    Bp, Br = cfg.budgets()
    return {
        "workload": cfg.name, "layers": layers, "batch_per_gpu": cfg.batch, "global_batch": cfg.batch * world,
        "L": cfg.L, "Hq": cfg.Hq, "Hkv": cfg.Hkv, "head_dim": cfg.d, "P": cfg.P, "budget_proxy": Bp, "budget_random": Br,
        "n_sink": cfg.n_sink, "n_recent": cfg.n_recent, "heavy_hitter_rate": cfg.hh_rate, "alpha": cfg.hh_alpha,
        "parallelism": f"batch-sharded x{world}, no collective", "l2": "inputs_exceed_l2 (distinct K/V per layer)",
        "alg_bytes_per_layer": cfg.alg_bytes_per_layer(),
    }


def stage_alg_bytes(cfg) -> dict:
    """Algorithmic HBM bytes one launch of each kernel has to move."""
    kv_head = cfg.batch * cfg.Hkv
    k_bytes = kv_head * cfg.L * cfg.d * cfg.elem_bytes
    imp_bytes = kv_head * cfg.L * 4
    return {
        "score_stats": k_bytes,                      # K streamed once
        "score_combine": 0,
        "score_colsum": k_bytes + imp_bytes,         # K streamed again (L2 hits show up as traffic < this) + imp written
        "score_fused": k_bytes + imp_bytes,          # both sweeps in one launch: K once
        "gumbel_keys": 2 * imp_bytes,
        "select": 2 * imp_bytes + kv_head * cfg.C * 4,
        "gather": 4 * kv_head * cfg.C * cfg.d * cfg.elem_bytes + kv_head * cfg.C * 4,
    }


def load_traffic(cfg_name: str, kernel: str):
    """dram bytes (read + write) per launch of `kernel` from the committed ncu --set full summary
    (profiles/traffic.csv: workload,kernel,dram_bytes_per_launch,source), if one exists."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    found = None
    try:
        with open(path) as f:
            for line in f:
                c = [x.strip() for x in line.split(",")]
                if len(c) >= 3 and c[0] == cfg_name and c[1] == kernel:
                    found = int(float(c[2]))  # later lines are later captures
    except (OSError, ValueError):
        pass
    return found


def run_ours(args) -> dict:
    from paper_2408_03675_b200 import binding  # raises when libnacl_evict.so cannot be built/loaded: no fallback

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device for --impl ours (there is no CPU fallback)")
    if int(os.environ.get("WORLD_SIZE", 1)) > 1:
        # the benchmark (not the library) wants NCCL's communicator line ("... nranks N ...") in its log: the driver reads it
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    rank, local_rank, world = nacl_dist.init()
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    cfg = CONFIGS[args.config]
    layers = args.layers or cfg.layers
    Bp, Br = cfg.budgets()
    C = Bp + Br
    tdt = torch.float32 if cfg.dtype == "f32" else torch.bfloat16
    rank_cfg = cfg.scaled(config_id=cfg.config_id + 10 * rank)  # every rank evicts its own batch of prompts

    data = []
    for l in range(layers):
        K, V, Q, _ = make_layer_inputs(rank_cfg, layer=l, device=dev)
        oK = torch.empty((cfg.batch, cfg.Hkv, C, cfg.d), dtype=tdt, device=dev)
        oV = torch.empty_like(oK)
        oi = torch.empty((cfg.batch, cfg.Hkv, C), dtype=torch.int32, device=dev)
        data.append((K, V, Q, oK, oV, oi))
    wss = []
    for _ in range(2):  # neighbouring calls of a batch run on two streams: two workspaces
        w = torch.empty(binding.nacl_workspace_bytes(cfg.batch, cfg.L, cfg.Hq, cfg.Hkv, cfg.d, cfg.P) + 256, dtype=torch.uint8, device=dev)
        wss.append(w[(-w.data_ptr()) % 256:])
    ws = wss[0]
    stream = torch.cuda.current_stream(dev)

    def step():  # one C-ABI call per layer, one after the other on one stream
        for l, (K, V, Q, oK, oV, oi) in enumerate(data):
            binding.nacl_evict_ex(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(l), l,
                                  out_K=oK, out_V=oV, out_idx=oi, workspace=ws, stream=stream, flags=args.nacl_flags)

    def batch_calls(extra=None):
        return [dict(K=K, V=V, Qproxy=Q, budget_proxy=Bp, budget_random=Br, n_sink=cfg.n_sink, n_recent=cfg.n_recent,
                     seed=cfg.layer_seed(l), layer=l, out_K=oK, out_V=oV, out_idx=oi, workspace=wss[l & 1], stream=stream,
                     flags=args.nacl_flags, **(extra(l) if extra else {}))
                for l, (K, V, Q, oK, oV, oi) in enumerate(data)]

    def batch_step():  # the step's layers as ONE nacl_evict_batch call: independent calls alternating between two streams
        binding.nacl_evict_batch(batch_calls())

    def timed(n_steps: int) -> float:
        nacl_dist.barrier(dev)
        torch.cuda.synchronize(dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(n_steps):
            step()
        e1.record(stream)
        torch.cuda.synchronize(dev)
        nacl_dist.barrier(dev)
        return nacl_dist.max_over_ranks(e0.elapsed_time(e1), dev)

    for _ in range(max(args.warmup, 3)):
        step()
    # The timed step is ONE CUDA-graph launch of the step's calls (the library only enqueues: every call is capturable with
    # a caller workspace); the same calls launched one by one from Python are timed beside it (ms_per_step_eager).
    eager_step = step
    for _ in range(max(args.warmup, 3)):
        batch_step()
    graph = None
    if args.no_batch:
        batch_step = eager_step
    if not args.no_graph:
        cap = torch.cuda.Stream(dev)
        cap.wait_stream(stream)
        with torch.cuda.stream(cap):
            graph = torch.cuda.CUDAGraph()
            outer_stream, stream = stream, cap
            with torch.cuda.graph(graph, stream=cap):
                batch_step()
            stream = outer_stream
        stream.wait_stream(cap)
        torch.cuda.synchronize(dev)

        def step():
            graph.replay()

        for _ in range(max(args.warmup, 3)):
            step()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    if graph is None:
        step = batch_step
    ms_total = timed(args.steps)
    # what the timed configuration left in one layer's outputs, for the self-check below (outside the timed region)
    chk_l = layers - 1
    chk_snap = [t.clone() for t in data[chk_l][3:6]]
    step = batch_step
    ms_total_batch_eager = timed(args.steps) if graph is not None else ms_total
    step = eager_step
    ms_total_eager = timed(args.steps)
    # the timed region again (the same calls, without the graph: events cannot be captured) with per-kernel events
    # (include/nacl_evict.h nacl_profile_*), for `kernels`, `gpu_launches` and the roofline
    binding.nacl_profile_enable(True)
    binding.nacl_profile_read(reset=True)
    step = batch_step
    ms_total_prof = timed(args.steps)
    stages = binding.nacl_profile_read(reset=True)
    # ... and of one nacl_evict_ex call per layer on one stream (fused scoring launch, select with fused gather)
    step = eager_step
    step()
    binding.nacl_profile_read(reset=True)
    timed(max(1, args.steps // 4))
    stages_one = binding.nacl_profile_read(reset=True)
    binding.nacl_profile_enable(False)
    clocks = sampler.stop() if rank == 0 else None

    # the same step with the row log-sum-exps supplied (as a prefill attention kernel has them):
    # one logit sweep instead of two.  Reported beside the headline, never instead of it.
    lses = []
    for l, (K, V, Q, oK, oV, oi) in enumerate(data):
        r = binding.nacl_evict_ex(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(l), l, out_K=oK, out_V=oV,
                                  out_idx=oi, workspace=ws, stream=stream, want_lse=True)
        lses.append(r["lse"])
    main_step = step

    def step_lse():
        if args.no_batch:
            for l, (K, V, Q, oK, oV, oi) in enumerate(data):
                binding.nacl_evict_ex(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(l), l,
                                      out_K=oK, out_V=oV, out_idx=oi, workspace=ws, stream=stream, lse_in=lses[l])
        else:
            binding.nacl_evict_batch(batch_calls(lambda l: {"lse_in": lses[l]}))

    step = step_lse
    step()
    ms_lse = timed(args.steps) / args.steps
    # ... and the producer of those statistics when the prefill kernel does not hand them out: nacl_proxy_lse (the statistics
    # sweep alone), one call per layer on one stream
    lse_tmp = torch.empty_like(lses[0])

    def step_plse():
        for l, (K, V, Q, oK, oV, oi) in enumerate(data):
            binding.nacl_proxy_lse(K, Q, out=lse_tmp, workspace=ws, stream=stream)

    step = step_plse
    step()
    ms_plse = timed(max(1, args.steps // 4)) / max(1, args.steps // 4)
    step = main_step

    # self-check: the outputs the TIMED configuration (graph replay of the batch call) produced for one layer equal, bit for
    # bit, those of a fresh single nacl_evict_ex call on the same inputs (its own outputs, the library's workspace)
    K, V, Q = data[chk_l][:3]
    fresh = binding.nacl_evict_ex(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(chk_l), chk_l, stream=stream)
    torch.cuda.synchronize(dev)
    self_ok = (torch.equal(chk_snap[2], fresh["out_idx"]) and torch.equal(chk_snap[0].view(torch.uint8), fresh["out_K"].view(torch.uint8))
               and torch.equal(chk_snap[1].view(torch.uint8), fresh["out_V"].view(torch.uint8)))
    self_ok = self_ok and int(fresh["out_idx"].min()) >= 0 and int(fresh["out_idx"].max()) < cfg.L
    del fresh, chk_snap

    ms_per_step = ms_total / args.steps
    alg_bytes_step = cfg.alg_bytes_per_layer() * layers * world
    value = alg_bytes_step / (ms_per_step * 1e-3) / 1e9
    peaks = load_peaks()

    # ---- roofline of the dominant kernel
    sab = stage_alg_bytes(cfg)
    if stages.get("gather", (0, 0))[1] == 0:  # the cluster select kernel also moves the kept rows (steps a4-a7 in one launch)
        sab["select"] += sab["gather"]
    sab_one = stage_alg_bytes(cfg)
    if stages_one.get("gather", (0, 0))[1] == 0:
        sab_one["select"] += sab_one["gather"]
    stage_rows = {}
    for name, (ms, n) in stages.items():
        if n == 0:
            continue
        avg_us = ms / n * 1e3
        stage_rows[name] = {"launches": n, "avg_us": round(avg_us, 2), "share": None,
                            "alg_GBps": round(sab.get(name, 0) / (avg_us * 1e-6) / 1e9, 1)}
    tot = sum(r["avg_us"] * r["launches"] for r in stage_rows.values()) or 1.0
    for r in stage_rows.values():
        r["share"] = round(r["avg_us"] * r["launches"] / tot, 4)
    one_rows = {name: {"launches": n, "avg_us": round(ms / n * 1e3, 2),
                       "alg_GBps": round(sab_one.get(name, 0) / (ms / n * 1e-3) / 1e9, 1)}
                for name, (ms, n) in stages_one.items() if n}
    # The dominant kernel is the SCORING (steps a1-a3): two launches (statistics sweep, column-sum sweep) in the timed
    # configuration, one fused launch in the single-call form.  Its algorithmic bytes count K ONCE (the second read is meant
    # to come from L2) plus the importance written.  `achieved` takes the fused launch ALONE on the GPU
    # (kernels_one_call_per_layer); the timed configuration's two sweeps run beside the other stream's selection and gather
    # and share the SMs with them: their event-to-event durations are given under `timed_form`, marked contended.
    score_alg = sab["score_fused"]
    score_names = [n for n in ("score_stats", "score_combine", "score_colsum", "score_fused") if n in stage_rows]
    roofline = None
    iso = one_rows.get("score_fused") or None
    if iso is None and one_rows:  # CUDA-core path: the three scoring launches of the single-call form, added up
        us = sum(one_rows[n]["avg_us"] for n in ("score_stats", "score_combine", "score_colsum") if n in one_rows)
        iso = {"avg_us": us, "alg_GBps": round(score_alg / (us * 1e-6) / 1e9, 1)} if us > 0 else None
    if iso:
        ach = iso["alg_GBps"]
        t_form_us = sum(stage_rows[n]["avg_us"] for n in score_names)
        roofline = {"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": round(ach / peaks["hbm_gbs"], 4),
                    "kernel": "score_fused" if "score_fused" in one_rows else "score_stats+score_combine+score_colsum",
                    "avg_us": iso["avg_us"], "alg_bytes_per_launch": score_alg,
                    "timing": "isolated: the scoring launch alone on the GPU, one nacl_evict_ex call per layer, CUDA events on its stream",
                    "timed_form": {"kernels": score_names, "avg_us_sum": round(t_form_us, 2), "contended": not args.no_batch,
                                   "alg_GBps": round(score_alg / (t_form_us * 1e-6) / 1e9, 1) if t_form_us > 0 else None,
                                   "frac": round(score_alg / (t_form_us * 1e-6) / 1e9 / peaks["hbm_gbs"], 4) if t_form_us > 0 else None,
                                   "note": "durations of the timed configuration's scoring launches; with two streams they overlap the "
                                           "other layer's selection / gather on the same SMs"}}
        if cfg.dtype == "bf16" and "score_fused" in one_rows:
            flop = 2.0 * cfg.batch * cfg.Hq * cfg.P * cfg.L * cfg.d * 2
            tf = flop / (iso["avg_us"] * 1e-6) / 1e12
            sus = peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"])
            roofline["tensor"] = {"achieved": round(tf, 1), "unit": "TFLOP/s", "alg_flop_per_launch": flop,
                                  "peak_burst": peaks["bf16_tflops"], "frac_of_burst": round(tf / peaks["bf16_tflops"], 4),
                                  "peak_sustained": sus, "frac_of_sustained": round(tf / sus, 4)}
            exps = 2.0 * cfg.batch * cfg.Hq * cfg.P * cfg.L
            roofline["exp"] = {"exps_per_launch": exps, "achieved_Gexp_per_s": round(exps / (iso["avg_us"] * 1e-6) / 1e9, 1),
                               "mufu_peak_Gexp_per_s": round(16 * 148 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e9, 1),
                               "note": "MUFU.EX2 alone: 16/clk/SM; the kernel splits the exponentials between MUFU and the FMA pipe"}
        roofline.update({"traffic": load_traffic(cfg.name, roofline["kernel"]), "peak_source": peaks["source"]})
    # call-level DRAM traffic of the TIMED configuration: sum of dram__bytes (ncu --set full, profiles/traffic.csv, rows named
    # "<kernel>@batch") over a layer's launches / the algorithmic bytes of a layer
    traffic_call = None
    per_kernel = {n: load_traffic(cfg.name, n + ("@batch" if not args.no_batch else "")) for n in stage_rows}
    if per_kernel and all(v is not None for v in per_kernel.values()):
        tot_b = sum(per_kernel.values())
        traffic_call = {"dram_bytes_per_layer": tot_b, "ratio_to_algorithmic": round(tot_b / cfg.alg_bytes_per_layer(), 3),
                        "kernels": per_kernel, "source": "profiles/traffic.csv (ncu --set full, one launch each, cold cache)"}

    # ---- end to end through the host entry point: pinned host buffers, H2D + D2H inside the timed region
    e2e = run_e2e(binding, cfg, layers, data, Bp, Br, dev, args, world)

    out = {
        "metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": round(ms_per_step, 4), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic (seeded N(0,1) Q/K/V + planted heavy hitters, DESIGN.md section 4)",
        "config": workload_desc(cfg, layers, world),
        "us_per_layer": round(ms_per_step * 1e3 / layers, 2),
        "prompt_tokens_per_s": round(cfg.batch * cfg.L * layers * world / (ms_per_step * 1e-3), 1),
        "evicted_token_slots_per_s": round(cfg.batch * cfg.Hkv * (cfg.L - C) * layers * world / (ms_per_step * 1e-3), 1),
        "hbm_frac_of_measured": round(value / world / peaks["hbm_gbs"], 4),
        "hbm_frac_of_nominal_8TBps": round(value / world / 8000.0, 4),
        "clocks": clocks, "e2e": e2e,
        # counted by the library itself: kernel launches recorded by the per-stage events over the same args.steps steps
        # counted by the library itself: kernel launches recorded by the per-stage events over the same args.steps steps
        "gpu_launches": int(sum(n for _, n in stages.values())),
        "roofline": roofline, "kernels": stage_rows,
        "kernels_note": ("durations between per-kernel events in the timed configuration; with two streams the kernels of "
                         "neighbouring layers run at the same time and share the SMs, so the durations add up to more than the "
                         "step; kernels_one_call_per_layer has every kernel alone on the GPU") if not args.no_batch else None,
        "kernels_one_call_per_layer": one_rows,
        "traffic_call": traffic_call,
        "self_check": "ok" if self_ok else "MISMATCH",
        "self_check_note": f"layer {chk_l}: out_idx / out_K / out_V of the timed configuration == a fresh nacl_evict_ex call, bitwise",
        "ms_per_step_batch_without_graph": round(ms_total_batch_eager / args.steps, 4),
        "ms_per_step_eager": round(ms_total_eager / args.steps, 4),
        "ms_per_step_with_kernel_events": round(ms_total_prof / args.steps, 4),
        "lse_in_variant": {"what": "nacl_evict_ex with lse_in (row log-sum-exps supplied, single logit sweep; SURVEY.md 8(f) f1)",
                           "ms_per_step": round(ms_lse, 4), "us_per_layer": round(ms_lse * 1e3 / layers, 2),
                           "proxy_lse_us_per_layer": round(ms_plse * 1e3 / layers, 2),
                           "value": round(alg_bytes_step / (ms_lse * 1e-3) / 1e9, 2), "unit": UNIT,
                           "hbm_frac_of_measured": round(alg_bytes_step / world / (ms_lse * 1e-3) / 1e9 / peaks["hbm_gbs"], 4)},
        "library": os.path.relpath(binding.library_path(), ROOT),
    }
    out["launch"] = ("one nacl_evict_batch call per step (the layers alternate between two streams)" if not args.no_batch
                               else "one nacl_evict_ex call per layer on one stream") + (", as one CUDA-graph launch" if graph is not None else "")
    if rank == 0 and world == 1 and not args.no_other_workloads:
        del data, lses
        torch.cuda.empty_cache()
        out["other_workloads"] = {CONFIGS[c].name: run_other(binding, CONFIGS[c], dev, peaks) for c in sorted(CONFIGS) if c != args.config}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = run_cpu_sample(cfg, max_seconds=15.0, max_layers=10)
    else:
        out["cpu_baseline"] = None
    nacl_dist.finalize()
    return out if rank == 0 else {}


def run_other(binding, cfg, dev, peaks, steps: int = 3, max_sets: int = 8) -> dict:
    """The same measurement (device time between CUDA events, distinct K/V per call so that every call is cold in L2)
    for one of the other BASELINE.json workloads, short: `max_sets` layers (the workload's own if fewer: the remaining
    calls rotate over the sets, at least 8 of them for the single-layer configs)."""
    Bp, Br = cfg.budgets()
    C = Bp + Br
    tdt = torch.float32 if cfg.dtype == "f32" else torch.bfloat16
    n_sets = max_sets
    data = []
    for l in range(n_sets):
        K, V, Q, _ = make_layer_inputs(cfg, layer=l % cfg.layers if cfg.layers > 1 else 0, device=dev) if cfg.layers > 1 else \
            make_layer_inputs(cfg.scaled(config_id=cfg.config_id + 100 * l), layer=0, device=dev)
        oK = torch.empty((cfg.batch, cfg.Hkv, C, cfg.d), dtype=tdt, device=dev)
        data.append((K, V, Q, oK, torch.empty_like(oK), torch.empty((cfg.batch, cfg.Hkv, C), dtype=torch.int32, device=dev)))
    ws = torch.empty(binding.nacl_workspace_bytes(cfg.batch, cfg.L, cfg.Hq, cfg.Hkv, cfg.d, cfg.P) + 256, dtype=torch.uint8, device=dev)
    ws = ws[(-ws.data_ptr()) % 256:]
    stream = torch.cuda.current_stream(dev)

    ws2 = torch.empty_like(ws)

    def step():
        for l, (K, V, Q, oK, oV, oi) in enumerate(data):
            binding.nacl_evict_ex(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(l), l, out_K=oK, out_V=oV, out_idx=oi,
                                  workspace=ws, stream=stream)

    def batch_step():
        binding.nacl_evict_batch([dict(K=K, V=V, Qproxy=Q, budget_proxy=Bp, budget_random=Br, n_sink=cfg.n_sink, n_recent=cfg.n_recent,
                                       seed=cfg.layer_seed(l), layer=l, out_K=oK, out_V=oV, out_idx=oi,
                                       workspace=ws if l % 2 == 0 else ws2, stream=stream)
                                  for l, (K, V, Q, oK, oV, oi) in enumerate(data)])

    def timed(fn):
        for _ in range(3):
            fn()
        torch.cuda.synchronize(dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize(dev)
        return e0.elapsed_time(e1) * 1e3 / (steps * n_sets)

    us_single = timed(step)
    us = timed(batch_step)
    binding.nacl_profile_enable(True)
    binding.nacl_profile_read(reset=True)
    step()
    torch.cuda.synchronize(dev)
    stages = binding.nacl_profile_read(reset=True)
    binding.nacl_profile_enable(False)
    gbs = cfg.alg_bytes_per_layer() / (us * 1e-6) / 1e9
    return {"us_per_layer": round(us, 2), "us_per_layer_one_call_per_layer": round(us_single, 2), "value": round(gbs, 2), "unit": UNIT,
            "hbm_frac_of_measured": round(gbs / peaks["hbm_gbs"], 4),
            "alg_bytes_per_layer": cfg.alg_bytes_per_layer(), "distinct_input_sets": n_sets, "dtype": cfg.dtype,
            "kernels_us": {k: round(ms / n * 1e3, 2) for k, (ms, n) in stages.items() if n},
            "dram_bytes": {k: load_traffic(cfg.name, k) for k in ("score_stats", "score_colsum", "select")}}


def run_e2e(binding, cfg, layers, data, Bp, Br, dev, args, world) -> dict:
    """The same metric through `nacl_evict_host_batch` (HOST buffers in, HOST buffers out): every layer's
    K/V/Q is copied from pinned host memory and its compacted K/V + index list is copied back, all
    inside the timed region.  Host copies of the first `n_sets` layers are rotated over the layers."""
    C = Bp + Br
    n_sets = min(layers, 4)
    host = []
    for l in range(n_sets):
        K, V, Q = data[l][0], data[l][1], data[l][2]
        hK, hV, hQ = K.cpu().pin_memory(), V.cpu().pin_memory(), Q.cpu().pin_memory()
        hoK = torch.empty((cfg.batch, cfg.Hkv, C, cfg.d), dtype=K.dtype, pin_memory=True)
        hoV = torch.empty_like(hoK, pin_memory=True)
        hoi = torch.empty((cfg.batch, cfg.Hkv, C), dtype=torch.int32, pin_memory=True)
        host.append((hK, hV, hQ, hoK, hoV, hoi))
    h2d = sum(t.numel() * t.element_size() for t in host[0][:3])
    d2h = sum(t.numel() * t.element_size() for t in host[0][3:])

    sets = [host[l % n_sets] for l in range(layers)]

    def step():
        # one call for the step's layers: two staging slots, the copies of a layer overlap the next layer's
        binding.nacl_evict_host_batch([h[0] for h in sets], [h[1] for h in sets], [h[2] for h in sets], Bp, Br, cfg.n_sink,
                                      cfg.n_recent, [cfg.layer_seed(l) for l in range(layers)], list(range(layers)),
                                      [h[3] for h in sets], [h[4] for h in sets], [h[5] for h in sets], device=dev.index)

    step()  # warm-up: staging buffers are allocated on first use
    n_steps = max(1, min(args.steps, 2))
    nacl_dist.barrier(dev)
    torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    for _ in range(n_steps):
        step()
    torch.cuda.synchronize(dev)
    dt = time.perf_counter() - t0
    nacl_dist.barrier(dev)
    dt = nacl_dist.max_over_ranks(dt, dev)
    val = cfg.alg_bytes_per_layer() * layers * world * n_steps / dt / 1e9
    return {"value": round(val, 3), "unit": UNIT, "h2d_bytes_per_step": h2d * layers, "d2h_bytes_per_step": d2h * layers,
            "steps": n_steps, "ms_per_step": round(dt / n_steps * 1e3, 3), "api": "nacl_evict_host_batch (pinned host buffers, one call per step)",
            "host_sets_rotated": n_sets, "timer": "host wall clock around synchronous calls, max over ranks"}


def run_cpu_sample(cfg, max_seconds: float, max_layers: int, layer0: int = 0) -> dict:
    """Times the fp64 oracle as it stands on the host cores over whole layers of the workload until
    `max_seconds` of CPU work or `max_layers` layers."""
    import oracle

    Bp, Br = cfg.budgets()
    n, spent = 0, 0.0
    while n < max_layers and spent < max_seconds:
        K, V, Q, _ = make_layer_inputs(cfg, layer=layer0 + n, device="cpu")
        t0 = time.perf_counter()
        oracle.evict(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(layer0 + n), layer0 + n)
        spent += time.perf_counter() - t0
        n += 1
    val = cfg.alg_bytes_per_layer() * n / spent / 1e9
    return {"value": round(val, 5), "unit": UNIT, "cores": oracle.threads(), "kind": "oracle",
            "sample": f"{n} whole layer(s) of {cfg.name} (layers {layer0}..{layer0 + n - 1}), {spent:.1f} s of oracle time",
            "s_per_layer": round(spent / n, 3)}


def run_reference(args) -> dict:
    """`--impl reference`: the oracle on the host cores; one step = one whole layer of the workload."""
    rank, _, world = nacl_dist.env_world()
    if rank != 0:
        return {}
    import oracle

    cfg = CONFIGS[args.config]
    Bp, Br = cfg.budgets()
    # torchrun pins OMP_NUM_THREADS=1 for its workers; the oracle arm is rank 0 alone and takes the host cores it may use
    nthreads = len(os.sched_getaffinity(0)) if world > 1 and hasattr(os, "sched_getaffinity") else 0
    steps, warmup = max(1, min(args.steps, 4)), max(0, min(args.warmup, 1))
    inputs = [make_layer_inputs(cfg, layer=l, device="cpu") for l in range(max(steps, 1))]
    for w in range(warmup):
        K, V, Q, _ = inputs[0]
        oracle.evict(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(0), 0, nthreads=nthreads)
    t0 = time.perf_counter()
    for l in range(steps):
        K, V, Q, _ = inputs[l]
        oracle.evict(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(l), l, nthreads=nthreads)
    dt = time.perf_counter() - t0
    val = cfg.alg_bytes_per_layer() * steps / dt / 1e9
    desc = workload_desc(cfg, cfg.layers, 1)
    sample = f"each step = one whole layer of {cfg.name}; {steps} step(s), {dt:.1f} s"
    return {
        "impl": "reference", "metric": METRIC, "value": round(val, 5), "unit": UNIT, "n_gpus": world, "steps": steps,
        "warmup": warmup, "ms_per_step": round(dt / steps * 1e3, 2), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic (same seeded generator as the CUDA arm)", "config": desc,
        "cpu_baseline": {"value": round(val, 5), "unit": UNIT, "cores": oracle.threads(nthreads), "kind": "oracle", "sample": sample},
        "e2e": {"value": round(val, 5), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "note": "fp64 CPU oracle (oracle/), rank 0 only; the reference is a paper with no code",
    }


def spawn_ranks(n: int) -> int:
    """`python bench.py --gpus N` without a torchrun environment: re-launch this command line under
    torch.distributed.run with N ranks on this node (one per GPU), exactly as the driver does."""
    import socket

    if "--impl" not in sys.argv or sys.argv[sys.argv.index("--impl") + 1] != "reference":
        if not torch.cuda.is_available() or torch.cuda.device_count() < n:
            raise SystemExit(f"bench.py --gpus {n}: needs {n} CUDA devices, found "
                             f"{torch.cuda.device_count() if torch.cuda.is_available() else 0} (there is no CPU fallback)")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=4, choices=sorted(CONFIGS))
    ap.add_argument("--layers", type=int, default=0, help="override the number of layers per step (0 = the workload's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-graph", action="store_true", help="time the step's calls launched one by one instead of one CUDA-graph launch")
    ap.add_argument("--no-batch", action="store_true", help="one nacl_evict_ex call per layer on one stream instead of one nacl_evict_batch call per step")
    ap.add_argument("--nacl-flags", type=lambda v: int(v, 0), default=0,
                    help="NACL_FLAG_* bits for the timed calls (profiling: 0x200 = the two scoring sweeps as two launches)")
    ap.add_argument("--no-other-workloads", action="store_true", help="skip the short runs of the other BASELINE.json configs")
    args = ap.parse_args()
    if args.gpus > 1 and "RANK" not in os.environ:
        return spawn_ranks(args.gpus)
    if args.gpus > 1 and int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus} was launched with WORLD_SIZE={os.environ.get('WORLD_SIZE')}")
    out = run_reference(args) if args.impl == "reference" else run_ours(args)
    if out:
        print(json.dumps(out), flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
