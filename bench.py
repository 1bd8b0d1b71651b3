#!/usr/bin/env python
"""bench.py -- decode tokens/s at 128K context for the SparDA decode hot path on B200 (libsparda).

Contract (driver):  python bench.py --gpus N --steps K --warmup W [--impl reference]
One JSON line on stdout (rank 0).  A "step" is one decode step of the whole hot path over one batch:
32 Forecast selections (a1+a2), 31 UVA gathers from pinned host memory (a3), the event hand-off (a4) and 32
block-sparse GQA attentions (a5/a6) -- Algorithm 2 lines 4-7 for 32 layers.

Workload at N=1: BASELINE.json configs[2] ("32-layer lookahead decode pipeline at 128K", batch 4), the
configuration the metric "decode tok/s at 128K" is quoted on that fits one GPU box (16 GiB of pinned host
KV).  configs[3] (batch 32, 137 GB pinned) is reachable with --workload cfg4 [--batch B] and aliases the
host cache onto fewer resident layers when the box cannot pin that much.

N > 1: every rank runs the same per-GPU workload on its own sequences (batch shards, no collective on the data
path -- SURVEY 8(e)); value = tokens all ranks decoded / max-over-ranks device time.  Under torchrun the ranks
come from the environment; a plain `python bench.py --gpus N` spawns them itself and exits non-zero if the box
has fewer than N GPUs.

Everything the line reports is measured in this run.  The only numbers that are not -- DRAM traffic and executed
instructions per launch, which need ncu -- are read from the committed profiles/r2_ncu_metrics.csv and carry the
file's content hash (`traffic_src`); a kernel without an entry there reports null.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import socket
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "decode_tokens_per_s_128k"
UNIT = "tok/s"
NCU_METRICS = os.path.join(ROOT, "profiles", "r2_ncu_metrics.csv")
STANDIN_BYTES = 474 * 10**6    # bf16 weights of one 8B decoder layer minus the attention: the labelled stand-in
ALL_SECTIONS = ("kernels", "prefill", "reuse", "standin", "gather", "floor", "append")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="sparda", choices=["sparda", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=["cfg3", "cfg4"])
    ap.add_argument("--batch", type=int, default=0, help="override the workload's batch (cfg4 sweep: 8/16/32)")
    ap.add_argument("--layers", type=int, default=0, help="override the layer count (debug; invalid as a bench value)")
    ap.add_argument("--gather-ctas", type=int, default=0)
    ap.add_argument("--gather-mode", default="tma", choices=["tma", "ldg"])
    ap.add_argument("--host-gib", type=float, default=0.0, help="cap on pinned host KV per rank (GiB); 0 = auto")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sections", default="all",
                    help="comma list of the extra sections measured after the headline step: " + ",".join(ALL_SECTIONS) + " (all | none)")
    ap.add_argument("--section", default="all", choices=["all", "kernels"],
                    help="kernels: ONLY the per-kernel sections, no pipeline (the command the ncu captures in profiles/ run)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the cpu_baseline sample")
    a = ap.parse_args()
    a.sections = set(ALL_SECTIONS) if a.sections == "all" else set(s for s in a.sections.split(",") if s and s != "none")
    bad = a.sections - set(ALL_SECTIONS)
    if bad:
        ap.error(f"unknown sections {sorted(bad)}")
    return a


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": d.get("bf16_tflops"),
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained"), "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback (B200_PROFILING.md)"}


def load_ncu_metrics():
    """profiles/r2_ncu_metrics.csv: `key,metric,value` rows extracted from the committed ncu captures (the commands are
    in profiles/r2_ncu_summary.md).  Returns ({key: {metric: value}}, 'path@sha1[:12]')."""
    if not os.path.exists(NCU_METRICS):
        return {}, None
    raw = open(NCU_METRICS, "rb").read()
    out = {}
    for line in raw.decode().splitlines():
        line = line.split("#")[0].strip()
        if not line or line.startswith("key,"):
            continue
        key, metric, value = [x.strip() for x in line.split(",")[:3]]
        out.setdefault(key, {})[metric] = float(value)
    return out, f"profiles/{os.path.basename(NCU_METRICS)}@{hashlib.sha1(raw).hexdigest()[:12]}"


def workload_config(args):
    from paper_2606_04511_b200 import synth
    cfg = synth.CFG3_128K if args.workload == "cfg3" else synth.CFG4_128K
    if args.batch:
        cfg = cfg.with_(batch=args.batch)
    if args.layers:
        cfg = cfg.with_(n_layers=args.layers)
    return cfg


def config_dict(cfg, world):
    """The workload, identically for both arms (the driver compares the two dicts)."""
    return {"workload": cfg.name, "batch_per_gpu": cfg.batch, "global_batch": cfg.batch * world, "context": cfg.context,
            "layers": cfg.n_layers, "q_heads": cfg.n_q_heads, "kv_heads": cfg.n_kv_heads, "head_dim": cfg.head_dim,
            "block": cfg.block_size, "topk": cfg.topk, "parallelism": f"batch shards x{world}, no collective",
            "fresh_fetch_fraction": 1.0,
            "l2": f"inputs larger than L2: {(cfg.kpool_bytes_per_layer * cfg.n_layers + cfg.gather_bytes_per_layer * (cfg.n_layers - 1)) / 2**20:.0f} MiB touched per step"}


# ------------------------------------------------------------------------------------------------
# clocks: nvidia-smi sampled DURING the timed region
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, gpu_id: str):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", gpu_id, f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "50"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(",") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, smax, power, reasons = [], [], [], set()
        for r in rows:
            try:
                sm.append(float(r[0])), smax.append(float(r[1])), power.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(self.NAMES, r[3:7]):
                if v.strip().lower() == "active":
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "reasons": sorted(reasons), "samples": len(sm)}


def numa_info(torch, local):
    """Where the pinned KV lives relative to the GPU: the GPU's NUMA node from sysfs, the node of the CPU this
    process allocates (first-touches) on, and the CPU affinity.  Best effort: None where the box does not say."""
    out = {"gpu_numa_node": None, "alloc_cpu": None, "alloc_numa_node": None, "numa_nodes": None,
           "affinity_cpus": len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else None}
    try:
        props = torch.cuda.get_device_properties(local)
        bdf = f"{props.pci_domain_id:04x}:{props.pci_bus_id:02x}:{props.pci_device_id:02x}.0"
        out["gpu_numa_node"] = int(open(f"/sys/bus/pci/devices/{bdf}/numa_node").read())
    except Exception:
        pass
    try:
        cpu = int(open("/proc/self/stat").read().rsplit(")", 1)[1].split()[36])
        out["alloc_cpu"] = cpu
        nodes = sorted(d for d in os.listdir("/sys/devices/system/node") if d.startswith("node") and d[4:].isdigit())
        out["numa_nodes"] = len(nodes)
        for nd in nodes:
            for part in open(f"/sys/devices/system/node/{nd}/cpulist").read().strip().split(","):
                lo, _, hi = part.partition("-")
                if int(lo) <= cpu <= int(hi or lo):
                    out["alloc_numa_node"] = int(nd[4:])
    except Exception:
        pass
    out["policy"] = "default (first touch by the allocating thread; no explicit binding)"
    return out


# ------------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline and --impl reference).  The only place bench.py touches oracle/.
# ------------------------------------------------------------------------------------------------
def _oracle_layer_step(oracle, lay, prev_F, k, layer0):
    """One layer of Algorithm 2 lines 4-7 on the CPU oracle: select, gather, attention."""
    ids, _ = oracle.forecast_select(prev_F, lay["kpool"], k)
    if layer0:
        oracle.sparse_attn(lay["Q"], lay["kv"], ids, pool_is_indexed=True)
    else:
        pool = oracle.gather(lay["kv"], ids)
        oracle.sparse_attn(lay["Q"], pool, ids)


def _oracle_sample_layers(cfg, n, device="cpu"):
    """n layers of oracle inputs (uint16 bit arrays), generated with the shared seeded generator; the pooled
    keys come from the oracle's own pooling (o1), outside the timed region (a0 is a pre-condition)."""
    import numpy as np
    import torch
    from oracle import sparda_oracle as oracle
    from paper_2606_04511_b200 import synth
    out = []
    for l in range(n):
        L = synth.decode_layer(cfg, l, device=device)
        bits = {key: L[key].cpu().contiguous().view(torch.int16).numpy().view(np.uint16) for key in ("kv", "F", "Q", "F0cur")}
        bits["kpool"] = oracle.pool_keys(bits["kv"])
        out.append(bits)
    return out


def cpu_baseline(cfg, layers_bits, target_s):
    """Oracle timed on this box's host cores on a bounded sample: whole layers of the decode step, as many as
    fit in ~target_s seconds, scaled to the full layer count; plus the same two layer-steps single-threaded."""
    from oracle import sparda_oracle as oracle
    cores = oracle.threads()

    def run(max_steps, budget):
        t0 = time.perf_counter()
        done = 0
        while done < max_steps:
            l = done % cfg.n_layers
            lay = layers_bits[l % len(layers_bits)]
            prev = layers_bits[(l - 1) % len(layers_bits)]
            _oracle_layer_step(oracle, lay, lay["F0cur"] if l == 0 else prev["F"], cfg.topk, layer0=(l == 0))
            done += 1
            if time.perf_counter() - t0 >= budget:
                break
        return done, time.perf_counter() - t0

    done, el = run(10**6, target_s)
    per_step_s = el * cfg.n_layers / done
    oracle.set_threads(1)
    d1, e1 = run(2, 1e9)                                       # layer 0 + one gathered layer, one thread
    oracle.set_threads(cores)
    per_step_1 = e1 * cfg.n_layers / d1
    return {"value": cfg.batch / per_step_s, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{done} layer-steps (select+gather+attention, batch {cfg.batch}, 128K) in {el:.2f} s, scaled to {cfg.n_layers} layers",
            "seconds_per_decode_step": per_step_s,
            "single_thread": {"value": cfg.batch / per_step_1, "unit": UNIT, "cores": 1, "seconds_per_decode_step": per_step_1,
                              "sample": f"{d1} layer-steps in {e1:.2f} s, scaled to {cfg.n_layers} layers"}}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = workload_config(args)
    from oracle import sparda_oracle as oracle
    oracle.build()
    n_sample = 2                                            # layer 0 (indexed cache) + one gathered layer per step
    layers_bits = _oracle_sample_layers(cfg, n_sample)
    times = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        for l in range(n_sample):
            _oracle_layer_step(oracle, layers_bits[l], layers_bits[0]["F0cur"] if l == 0 else layers_bits[l - 1]["F"],
                               cfg.topk, layer0=(l == 0))
        if it >= args.warmup:
            times.append(time.perf_counter() - t0)
    per_step_s = statistics.mean(times) * cfg.n_layers / n_sample
    val = cfg.batch / per_step_s
    sample = f"each step = {n_sample} of {cfg.n_layers} layer-steps (layer 0 + one gathered layer) of the oracle, scaled to {cfg.n_layers}"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": per_step_s * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(cfg, 1),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
# the CUDA arm: helpers
# ------------------------------------------------------------------------------------------------
def graph_time(torch, fn, n_sets, reps=10, best_of=3, flush=None):
    """Seconds per launch of fn(i, stream): reps passes over n_sets rotating buffer sets captured once into a CUDA graph
    (the launches of these short kernels would otherwise be paced by the Python caller, not by the GPU) and replayed
    between two events on the replaying stream; best of `best_of` replays.  flush(): called before every timed replay,
    outside the events (an L2 flush for shapes whose rotation does not exceed L2)."""
    st = torch.cuda.current_stream()
    for i in range(2 * n_sets):
        fn(i % n_sets, st)
    torch.cuda.synchronize()
    graph, cap = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.graph(graph, stream=cap):
        for i in range(reps * n_sets):
            fn(i % n_sets, torch.cuda.current_stream())
    graph.replay()
    torch.cuda.synchronize()
    best = float("inf")
    for _ in range(best_of):
        if flush is not None:
            flush()
            torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        graph.replay()
        e1.record(st)
        e1.synchronize()
        best = min(best, e0.elapsed_time(e1) * 1e-3 / (reps * n_sets))
    del graph
    return best


def isolated_time(torch, fn, n_sets, n=64):
    """Seconds for ONE launch of fn(i, stream) as the decode step runs it: between two events of its own on the launching
    stream, without programmatic dependent launch (the caller's context has no_pdl = 1), on the next of n_sets rotating buffer
    sets (cold HBM), nothing of the same kind in flight before or behind it.  Median of n.  This is what one launch costs;
    graph_time() beside it is the steady-state PERIOD of back-to-back launches, in which PDL hides each launch's gap, prologue
    and first loads behind its predecessor's tail -- a pattern the step does not have."""
    st = torch.cuda.current_stream()
    for i in range(n_sets):
        fn(i, st)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
    for i, (e0, e1) in enumerate(ev):
        # a 150 us spin (no memory traffic) in front of the bracket: by the time the GPU reaches e0 the launch and e1 are already
        # queued, so the bracket holds the GPU's time for the launch (kernel boundary included), not this Python loop's pace
        torch.cuda._sleep(300_000)
        e0.record(st)
        fn(i % n_sets, st)
        e1.record(st)
        if i % 8 == 7:
            torch.cuda.synchronize()
    torch.cuda.synchronize()
    ts = sorted(e0.elapsed_time(e1) for e0, e1 in ev)
    return ts[len(ts) // 2] * 1e-3


def kernel_entry(name, shape, t, nbytes, peak, ncu, key, ncu_src, **extra):
    m = ncu.get(key, {})
    traffic = (m.get("dram__bytes_read.sum", 0.0) + m.get("dram__bytes_write.sum", 0.0)) if "dram__bytes_read.sum" in m else None
    e = {"kernel": name, "shape": shape, "bound": "hbm", "us": round(t * 1e6, 3), "bytes": int(nbytes),
         "achieved": round(nbytes / t / 1e9, 1), "peak": peak, "unit": "GB/s", "frac": round(nbytes / t / 1e9 / peak, 4),
         "frac_of_8tbs": round(nbytes / t / 1e9 / 8000.0, 4), "traffic": traffic, "traffic_src": ncu_src if traffic is not None else None}
    e.update(extra)
    return e


def measure_h2d_ceiling(torch, host_chunks):
    """cudaMemcpyAsync pinned host -> device ceiling on this box: the denominator of the gather's roofline.
    Copies whole pinned layer buffers (>= 256 MiB each) back to back, best of 5 passes, CUDA events."""
    dev = torch.empty_like(host_chunks[0], device="cuda")
    nbytes = sum(h.numel() * h.element_size() for h in host_chunks)
    best = 0.0
    for _ in range(5):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for h in host_chunks:
            dev.copy_(h, non_blocking=True)
        e1.record()
        e1.synchronize()
        best = max(best, nbytes / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    return best


# ------------------------------------------------------------------------------------------------
# per-kernel sections
# ------------------------------------------------------------------------------------------------
def bench_kernels(torch, binding, peaks, ncu, ncu_src, batch):
    """Per-kernel HBM rooflines at one batch of the BASELINE.json configs[3] shape (R = 2 * batch rows, 2048 blocks,
    top-64, D = 128).  Batch 32 is where the ideal times (5 us select, 20 us attention) stand clear of the launch
    floor; batch 4 is configs[2]'s per-layer shape, launch-latency-sized, reported beside the floor.
    Cold HBM: each launch works on the next of several buffer sets, together >= 1 GiB (8 x the 126 MB L2); launches are
    replayed from a CUDA graph."""
    from paper_2606_04511_b200 import synth
    cfg = synth.CFG4_128K.with_(batch=batch)
    R, Nb, k, D = cfg.rows, cfg.n_blocks, cfg.topk, cfg.head_dim
    ctx = binding.Sparda.from_config(cfg)
    g = torch.Generator(device="cuda").manual_seed(40 + batch)
    tag = f"b{batch}"
    kp_bytes, pool_bytes = cfg.kpool_bytes_per_layer, cfg.gather_bytes_per_layer
    NS_SEL = max(4, -(-(1 << 30) // kp_bytes))
    NS_SEL = min(NS_SEL, 64)
    NS_ATT = min(max(4, -(-(1 << 30) // pool_bytes)), 64)
    Fs = [torch.randn((R, D), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16) for _ in range(8)]
    ids = torch.empty((R, k), dtype=torch.int32, device="cuda")
    kpools = [torch.randn((R, Nb, D), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16) for _ in range(NS_SEL)]
    t_sel = graph_time(torch, lambda i, s: ctx.forecast_select(Fs[i % 8], kpools[i], Nb, k, ids, stream=s), NS_SEL, reps=max(2, 160 // NS_SEL))
    cs_sel = ctx.select_cluster
    ctx_iso = binding.Sparda.from_config(cfg, no_pdl=1)      # plain launches: one launch in isolation (see isolated_time)
    t_sel_iso = isolated_time(torch, lambda i, s: ctx_iso.forecast_select(Fs[i % 8], kpools[i], Nb, k, ids, stream=s), NS_SEL)
    NS_PAIR = min(NS_SEL, max(2, -(-(256 << 20) // kp_bytes)))   # pooled-key sets kept for the pair: >= 256 MiB (2 x L2) of rotation
    kpools = kpools[:NS_PAIR]
    pools = []
    for _ in range(NS_ATT):
        p = torch.empty((R, k, 2, 64, D), dtype=torch.bfloat16, device="cuda")
        p.copy_(torch.randn(p.shape, generator=g, device="cuda", dtype=torch.float32))
        pools.append(p)
    Q = torch.randn((cfg.batch, cfg.n_q_heads, D), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16)
    O = torch.empty_like(Q)
    ids_att = torch.arange(k, dtype=torch.int32, device="cuda").repeat(R, 1).contiguous()
    t_att = graph_time(torch, lambda i, s: ctx.sparse_decode(Q, pools[i], ids_att, k, O, stream=s), NS_ATT, reps=max(2, 80 // NS_ATT))
    cl_att = ctx.attn_cluster
    t_att_iso = isolated_time(torch, lambda i, s: ctx_iso.sparse_decode(Q, pools[i], ids_att, k, O, stream=s), NS_ATT)

    def pair(i, s):   # one layer's select + attention back to back on one stream, no PDL: the metric's "select+attn"
        ctx_iso.forecast_select(Fs[i % 8], kpools[i % NS_PAIR], Nb, k, ids, stream=s)
        ctx_iso.sparse_decode(Q, pools[i], ids_att, k, O, stream=s)
    t_pair = isolated_time(torch, pair, NS_ATT)
    # what the bracket itself costs: nothing between the two events, and one empty kernel (the launch floor inside the same bracket)
    t_br0 = isolated_time(torch, lambda i, s: None, 1)
    t_br1 = isolated_time(torch, lambda i, s: ctx_iso.probe_launch(0, stream=s), 1)
    ctx_iso.close()
    del kpools
    # the tcgen05 "swap-AB" experiment (cfg.attn_impl = 1) on the same pools: a measured comparison, not the product path
    ctx5 = binding.Sparda.from_config(cfg, attn_impl=1)
    t_att5 = graph_time(torch, lambda i, s: ctx5.sparse_decode(Q, pools[i], ids_att, k, O, stream=s), NS_ATT, reps=max(2, 80 // NS_ATT))
    ctx5.close()
    del pools
    sel_bytes = kp_bytes + R * D * 2 + R * k * 4
    att_bytes = pool_bytes + 2 * cfg.batch * cfg.n_q_heads * D * 2 + R * k * 4
    hbm = peaks["hbm_gbs"]
    iso = lambda t, b: {"us_isolated": round(t * 1e6, 3), "frac_isolated": round(b / t / 1e9 / hbm, 4),
                        "isolated": "one launch between two events behind a 150 us spin kernel, no PDL, cold buffers, median of 64; `us` / `frac` are the PDL back-to-back period"}
    out = [kernel_entry("forecast_select_kernel<128,false>", f"batch {batch}: R={R}, {Nb} blocks, top-{k}; cold HBM, graph replay", t_sel, sel_bytes,
                        hbm, ncu, f"select_{tag}", ncu_src, cluster=cs_sel, **iso(t_sel_iso, sel_bytes)),
           kernel_entry("sparse_decode_kernel<128>", f"batch {batch}: R={R}, top-{k} x 32 KiB; cold HBM, graph replay", t_att, att_bytes,
                        hbm, ncu, f"attn_{tag}", ncu_src, cluster=cl_att, ctas_per_row=ctx.attn_splits(k), **iso(t_att_iso, att_bytes)),
           {"kernel": "pair: forecast_select + sparse_decode", "shape": f"batch {batch}: one layer's select then attention on one stream, no PDL, cold HBM; "
            "one pair between two events, median of 64", "bound": "hbm", "us_isolated": round(t_pair * 1e6, 3), "bytes": int(sel_bytes + att_bytes),
            "achieved": round((sel_bytes + att_bytes) / t_pair / 1e9, 1), "peak": hbm, "unit": "GB/s",
            "frac_isolated": round((sel_bytes + att_bytes) / t_pair / 1e9 / hbm, 4), "frac_of_8tbs": round((sel_bytes + att_bytes) / t_pair / 1e9 / 8000.0, 4),
            "tag": f"pair_{tag}", "bracket_empty_us": round(t_br0 * 1e6, 3), "bracket_null_kernel_us": round(t_br1 * 1e6, 3)},
           kernel_entry("sparse_decode_tc5_kernel (experiment)", f"batch {batch}: same shape, tcgen05 swap-AB form (attn_impl=1); not the default", t_att5,
                        att_bytes, hbm, ncu, f"attn_tc5_{tag}", ncu_src, cluster=cl_att)]
    if batch == 32:
        # f3: the paper's geometry -- (32,16) compressed-key grid (4 keys per block), max-pool to blocks, budget 96 = 1 + 32 + 63
        NS_G = 8
        grids = [torch.randn((R, 4 * Nb, D), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16) for _ in range(NS_G)]
        ids96 = torch.empty((R, 96), dtype=torch.int32, device="cuda")
        ctx96 = binding.Sparda(cfg.batch, cfg.n_q_heads, cfg.n_kv_heads, D, Nb, 96)
        t_grid = graph_time(torch, lambda i, s: ctx96.forecast_select_grid(Fs[i % 8], grids[i], Nb, 96, ids96, n_init=1, n_local=32, stream=s), NS_G, reps=10)
        grid_bytes = R * (4 * Nb - 1) * D * 2 + R * D * 2 + R * 96 * 4
        out.append(kernel_entry("forecast_select_kernel<128,grid>", "f3 (reading q19, unpinned): batch 32, 4 keys per block, top-96 = 1 + 32 + 63; cold HBM",
                                t_grid, grid_bytes, hbm, ncu, "grid_b32", ncu_src, cluster=ctx96.select_cluster))
        ctx96.close()
        del grids
        # A4: the Forecast projection GEMV (Eq.3), 8B shape: hidden 4096 -> 2 x 128; bound by streaming W_F (2 MiB) once
        hidden = 4096
        NS_W = 64
        Ws = [torch.randn((hidden, cfg.n_kv_heads * D), generator=g, device="cuda").to(torch.bfloat16) for _ in range(NS_W)]
        X = torch.randn((cfg.batch, hidden), generator=g, device="cuda").to(torch.bfloat16)
        Fo = torch.empty((R, D), dtype=torch.bfloat16, device="cuda")
        t_fp = graph_time(torch, lambda i, s: ctx.forecast_project(X, Ws[i], hidden, Fo, stream=s), NS_W, reps=3)
        fp_bytes = hidden * cfg.n_kv_heads * D * 2 + cfg.batch * hidden * 2 + R * D * 2
        out.append(kernel_entry("forecast_project_kernel", "A4 (Eq.3): batch 32, hidden 4096 -> 2 x 128; W_F rotated over 128 MiB", t_fp, fp_bytes,
                                hbm, ncu, "project_b32", ncu_src))
        del Ws
    ctx.close()
    torch.cuda.empty_cache()
    return out


def bench_floor(torch, binding):
    """Launch floor beside the launch-latency-sized shapes: per-launch time of back-to-back probe kernels
    replayed from a CUDA graph -- an empty kernel, an empty kernel with the select launch shape, and 148 CTAs doing one
    dependent DRAM load each."""
    from paper_2606_04511_b200 import synth
    ctx = binding.Sparda.from_config(synth.CFG1_TINY)
    buf = torch.zeros(1 << 28, dtype=torch.int32, device="cuda")   # 1 GiB: the touched locations are cold every launch
    nb = buf.numel() * 4
    out = {}
    for name, kind in (("empty_1x32_us", 0), ("empty_select_shape_us", 1)):
        out[name] = round(graph_time(torch, lambda i, s: ctx.probe_launch(kind, stream=s), 1, reps=200) * 1e6, 3)
    views = [buf[i * 4096:] for i in range(192)]                   # 16 KiB apart: a different DRAM line per launch and CTA
    scrub = torch.empty(1 << 27, dtype=torch.int32, device="cuda")  # 512 MiB written before each replay: the lines are cold
    out["one_dram_load_148_ctas_us"] = round(graph_time(torch, lambda i, s: ctx.probe_launch(2, views[i], nb - 192 * 16384, stream=s), 192, reps=1,
                                                        flush=lambda: scrub.fill_(1)) * 1e6, 3)
    out["note"] = "back-to-back launches in one graph: per-launch period, not latency"
    del scrub
    ctx.close()
    del buf
    torch.cuda.empty_cache()
    return out


def bench_prefill(torch, binding, peaks_all, ncu, ncu_src):
    """BASELINE.json configs[4]: chunked-prefill Forecast selection (a7) at T = 32768, 2 groups, 512 pooled keys, top-64,
    in 2048-row chunks (16 launches per pass) and as one launch, plus the per-head softmax comparison selector (a7',
    G = 16 heads per group) on the same shapes: the analog of the paper's 'selection cost cut up to 2.50x'."""
    from paper_2606_04511_b200 import synth
    cfg = synth.CFG5_PREFILL
    P = synth.prefill_inputs(cfg, device="cuda")
    T, Nb, k, Hkv, D = cfg.seq_len, cfg.n_blocks, cfg.topk, cfg.n_kv_heads, cfg.head_dim
    ctx = binding.Sparda(1, cfg.n_q_heads, Hkv, D, Nb, k)
    kpool = torch.empty((Hkv, Nb, D), dtype=torch.bfloat16, device="cuda")
    ctx.pool_keys(P["kv"], Hkv, Nb, kpool)
    ids = torch.empty((Hkv, T, k), dtype=torch.int32, device="cuda")
    part = torch.empty((Hkv, cfg.chunk, k), dtype=torch.int32, device="cuda")

    def chunked(fn, src, s):
        for r0 in range(0, T, cfg.chunk):
            fn(src, kpool, T, Nb, r0, cfg.chunk, k, part, stream=s)

    n0 = ctx.launch_count
    t_one = graph_time(torch, lambda i, s: ctx.prefill_select(P["F"], kpool, T, Nb, 0, T, k, ids, stream=s), 1, reps=10)
    t_chunk = graph_time(torch, lambda i, s: chunked(ctx.prefill_select, P["F"], s), 1, reps=5)
    t_base = graph_time(torch, lambda i, s: chunked(ctx.prefill_select_baseline, P["Q"], s), 1, reps=2)
    launches = ctx.launch_count - n0
    ncand = sum(min(Nb, (i + 1) // 64) for i in range(T))        # causal contraction: row i meets min(Nb, (i+1)//64) pooled keys
    flops = 2.0 * Hkv * ncand * D
    bf16_peak = peaks_all.get("bf16_tflops_sustained") or peaks_all.get("bf16_tflops") or 1400.0
    ranked_rows = Hkv * sum(1 for i in range(T) if (i + 1) // 64 > k)
    inst = ncu.get("prefill_one", {}).get("smsp__inst_executed.sum")
    inst_c = ncu.get("prefill_chunked_pass", {}).get("smsp__inst_executed.sum")
    alu_peak = 148 * 4 * 1.965                                     # G warp-instr/s: 148 SMs x 4 schedulers x 1 per clock x 1.965 GHz
    out = {
        "shape": f"{cfg.name}: T={T}, {Hkv} groups, {Nb} pooled keys, top-{k}, {cfg.chunk}-row chunks",
        "forecast_us_chunked": round(t_chunk * 1e6, 2), "forecast_us_one_launch": round(t_one * 1e6, 2),
        "baseline_selector_us_chunked": round(t_base * 1e6, 2), "baseline_over_forecast": round(t_base / t_chunk, 2),
        "tok_s_selection_only": round(T / t_chunk), "gpu_launches": launches, "ns_per_ranked_row": round(t_chunk * 1e9 / ranked_rows, 3),
        "tensor": {"kernel": "prefill_select_kernel<128,false>", "bound": "tensor", "achieved": round(flops / t_chunk / 1e12, 2), "peak": bf16_peak,
                   "unit": "TFLOP/s", "frac": round(flops / t_chunk / 1e12 / bf16_peak, 4), "flops": flops,
                   "note": "the contraction is ~1% of the kernel; the fused exact per-row top-k (plain ALU) is the cost"},
        "alu": {"kernel": "prefill_select_kernel<128,false,false> (one launch)", "bound": "alu", "us": round(t_one * 1e6, 2),
                "warp_instructions": inst, "achieved": round(inst / t_one / 1e9, 1) if inst else None, "peak": round(alu_peak, 1),
                "unit": "G warp-instr/s", "frac": round(inst / t_one / 1e9 / alu_peak, 4) if inst else None,
                "traffic_src": ncu_src if inst else None},
        "alu_chunked": {"kernel": "prefill_select_kernel<128,false,true> (16 chunk launches, replicated 32-row tiles)", "bound": "alu",
                        "us": round(t_chunk * 1e6, 2), "warp_instructions": inst_c, "achieved": round(inst_c / t_chunk / 1e9, 1) if inst_c else None,
                        "peak": round(alu_peak, 1), "unit": "G warp-instr/s", "frac": round(inst_c / t_chunk / 1e9 / alu_peak, 4) if inst_c else None,
                        "traffic_src": ncu_src if inst_c else None},
    }
    ctx.close()
    return out


def bench_append(torch, binding):
    """f2 (Alg.2 lines 2-3): one token appended per launch to a device-resident cache and to a pinned host cache written
    through UVA, batch-32 rows (R = 64, D = 128), 64 consecutive positions (one of them completes a block), replayed from
    a CUDA graph.  4 KiB of K/V + 64 KiB of fp32 running sums per launch: launch-latency-sized."""
    from paper_2606_04511_b200 import synth
    cfg = synth.CFG4_128K.with_(n_blocks=64)
    R, Nb, D = cfg.rows, cfg.n_blocks, cfg.head_dim
    ctx = binding.Sparda.from_config(cfg)
    g = torch.Generator(device="cuda").manual_seed(12)
    kn = torch.randn((64, R, D), generator=g, device="cuda").to(torch.bfloat16)
    vn = torch.randn((64, R, D), generator=g, device="cuda").to(torch.bfloat16)
    kpool = torch.zeros((R, Nb, D), dtype=torch.bfloat16, device="cuda")
    out = {}
    for where in ("device", "host_uva"):
        kv = torch.zeros((R, Nb, 2, 64, D), dtype=torch.bfloat16, device="cuda") if where == "device" else \
            torch.zeros((R, Nb, 2, 64, D), dtype=torch.bfloat16).pin_memory()
        ksum = torch.zeros((R, D), dtype=torch.float32, device="cuda")
        for t in range(64):
            ctx.append_kv(kn[t], vn[t], 64 + t, kv, Nb, ksum, kpool)
        torch.cuda.synchronize()
        graph, cap = torch.cuda.CUDAGraph(), torch.cuda.Stream()
        with torch.cuda.graph(graph, stream=cap):
            for t in range(64):
                ctx.append_kv(kn[t], vn[t], 128 + t, kv, Nb, ksum, kpool, stream=torch.cuda.current_stream())
        graph.replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(5):
            graph.replay()
        e1.record()
        e1.synchronize()
        out[f"us_per_append_{where}"] = round(e0.elapsed_time(e1) * 1e3 / (5 * 64), 3)
        del graph, kv
    out["shape"] = f"append_kv_kernel<128>, R = {R} rows (batch 32), one token per launch, 64 launches per graph"
    out["bytes_per_launch"] = R * D * 2 * 2 + 2 * R * D * 4
    ctx.close()
    return out


def bench_reuse(torch, binding, ctx, cfg, dev_layers, F0, cs, ps, steps, standin_bytes=0):
    """SURVEY 8(f) f1 / 8(d) "gather hidden": the same 32-layer decode step with the previous step's blocks kept per
    layer, so only newly selected blocks cross the host link.  The Forecast alternates between F_A and
    F_B = bf16(F_A + alpha * N(0,1)) from step to step; alpha sets how much the selection drifts, the fresh-fetch
    fraction rho is MEASURED (blocks fetched / blocks selected, from the plan kernel's counters).  alpha = 0 gives
    rho = 0: the compute-only floor of the step; exposed gather time = step(rho) - step(0).
    standin_bytes > 0: a labelled stand-in kernel (NOT part of the method) streams that many bytes of weights on the
    compute stream after every attention -- the rest of an 8B decoder layer -- so that 'gather hidden behind the next
    layer's compute' is measured."""
    R, k, Nb, D, NL = cfg.rows, cfg.topk, cfg.n_blocks, cfg.head_dim, cfg.n_layers
    g = torch.Generator(device="cuda").manual_seed(777)
    # two views of the same layers that differ only in the Forecast they point to: the step alternates between them, so
    # no copy of F sits in the timed region (F is an input of the path, produced by the model's projections)
    layers = [[], []]
    for l, d in enumerate(dev_layers):
        e = dict(d)
        if l:
            e["pool"] = torch.zeros((R, k, 2, cfg.block_size, D), dtype=torch.bfloat16, device="cuda")
            e["slot_ids"] = torch.full((R, k), -1, dtype=torch.int32, device="cuda")
            e["fetch"] = torch.full((R, k), -1, dtype=torch.int32, device="cuda")
            e["n_fetch"] = torch.zeros((R,), dtype=torch.int32, device="cuda")
        layers[0].append(e)
        layers[1].append({**e, "F": d["F"].clone()})
    arrs = [ctx.make_cached_layers(layers[0]), ctx.make_cached_layers(layers[1])]
    F0s = [F0, F0.clone()]
    noise = [torch.randn(d["F"].shape, generator=g, device="cuda") for d in dev_layers]
    noise0 = torch.randn(F0.shape, generator=g, device="cuda")
    weights = None
    if standin_bytes:
        weights = torch.empty(standin_bytes // 2, dtype=torch.bfloat16, device="cuda").fill_(1.0)
        ctx.set_layer_standin(weights, standin_bytes)

    def one(which):
        ctx.decode_step_cached(arrs[which], F0s[which], Nb, k, cs, ps, binding.STEP_OVERLAP)

    out = []
    for alpha in (0.0, 0.05, 0.1, 0.2, 0.3, 0.4, 0.8, 1e9):
        for l, e in enumerate(layers[1]):                    # F_B = bf16(F_A + alpha * N(0, 1))
            e["F"].copy_((dev_layers[l]["F"].float() + alpha * noise[l]).to(torch.bfloat16))
        F0s[1].copy_((F0.float() + alpha * noise0).to(torch.bfloat16))
        for e in layers[0][1:]:
            e["slot_ids"].fill_(-1)
        torch.cuda.synchronize()
        for i in range(4):
            one(i & 1)
        torch.cuda.synchronize()
        fetched = 0
        for i in range(2):                                   # periodic state: count one A step and one B step
            one(i & 1)
            torch.cuda.synchronize()
            fetched += sum(int(e["n_fetch"].sum().item()) for e in layers[0][1:])
        rho = fetched / (2.0 * (NL - 1) * R * k)
        n = max(4, steps - steps % 2)
        torch.cuda.synchronize()
        # one A step and one B step captured into a CUDA graph (three streams and their events): the ~200 enqueue calls of a
        # step would otherwise pace this compute-sized step from the host
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=cs):
            for i in range(2):
                ctx.decode_step_cached(arrs[i], F0s[i], Nb, k, cs, ps, binding.STEP_OVERLAP)
        graph.replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(cs):
            e0.record(cs)
            for i in range(n // 2):
                graph.replay()
            e1.record(cs)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / n
        del graph
        out.append({"alpha": alpha if alpha < 1e8 else "independent", "rho": round(rho, 4), "ms_per_step": round(ms, 4),
                    "tok_s": round(cfg.batch / (ms * 1e-3), 1), "link_mib_per_step": round(rho * (NL - 1) * cfg.gather_bytes_per_layer / 2**20, 1)})
    # Alg.2 l.1 inside the step (Eq.3): every layer hands X and W_F instead of a ready F, the projection kernel runs
    # on the select chain in front of the select that reads F.  Same X every step: rho = 0, so this is the floor + l.1
    proj_ms = None
    if ctx.cfg.hidden:
        hidden = ctx.cfg.hidden
        X = torch.randn((cfg.batch, hidden), generator=g, device="cuda").to(torch.bfloat16)
        wl = []
        for l, e in enumerate(layers[0]):
            w = {**e, "F": e["F"].clone(), "X": X, "WF": (torch.randn((hidden, cfg.n_kv_heads * D), generator=g, device="cuda") / hidden ** 0.5).to(torch.bfloat16)}
            if l == 0:
                w["WFcur"] = (torch.randn((hidden, cfg.n_kv_heads * D), generator=g, device="cuda") / hidden ** 0.5).to(torch.bfloat16)
            wl.append(w)
        arr_p = ctx.make_cached_layers(wl)
        F0p = F0.clone()
        for e in layers[0][1:]:
            e["slot_ids"].fill_(-1)
        for _ in range(3):
            ctx.decode_step_cached(arr_p, F0p, Nb, k, cs, ps, binding.STEP_OVERLAP)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=cs):
            for i in range(2):
                ctx.decode_step_cached(arr_p, F0p, Nb, k, cs, ps, binding.STEP_OVERLAP)
        graph.replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n = max(4, steps - steps % 2)
        with torch.cuda.stream(cs):
            e0.record(cs)
            for i in range(n // 2):
                graph.replay()
            e1.record(cs)
        torch.cuda.synchronize()
        proj_ms = round(e0.elapsed_time(e1) / n, 4)
        del graph, wl, arr_p
    floor = out[0]["ms_per_step"]
    for o in out:
        o["gather_exposed_us_per_layer"] = round(max(0.0, (o["ms_per_step"] - floor) * 1e3 / (NL - 1)), 2)
    hidden_up_to = max([o["rho"] for o in out if o["gather_exposed_us_per_layer"] <= 0.05 * floor * 1e3 / (NL - 1)] or [0.0])
    if standin_bytes:
        ctx.set_layer_standin(None, 0)
    del layers, arrs, weights
    torch.cuda.empty_cache()
    return {"shape": f"{cfg.name}, per-layer persistent pools, steps alternate between F_A and F_A + alpha*N(0,1); CUDA-graph replay",
            "standin_bytes_per_layer": standin_bytes,
            "standin": "NOT part of the method: a kernel streaming 474 MB of weights after every attention" if standin_bytes else None,
            "compute_floor_ms_per_step": floor, "us_per_layer_at_floor": round(floor * 1e3 / NL, 2),
            "compute_floor_with_in_step_projection_ms": proj_ms,
            "rho_hidden_up_to": hidden_up_to, "sweep": out}


def bench_chain_under_load(torch, binding):
    """What a kernel boundary costs on the select chain when the GPU is busy (the reason for the select -> gather doorbell of
    sparda_decode_step): batch-4 shapes of configs[2], the kernels of the chain replayed from a CUDA graph (16 per graph,
    rotating cold buffers) alone and while the labelled layer stand-in (NOT part of the method) saturates HBM on another
    stream.  Stand-alone launches: the two-kernel chain here is stream-ordered, without the doorbell."""
    from paper_2606_04511_b200 import synth
    cfg = synth.CFG4_128K.with_(batch=4)
    R, Nb, k, D = cfg.rows, cfg.n_blocks, cfg.topk, cfg.head_dim
    g = torch.Generator(device="cuda").manual_seed(91)
    ctx = binding.Sparda.from_config(cfg)
    NS = 16
    kpools = [torch.randn((R, Nb, D), generator=g, device="cuda").to(torch.bfloat16) for _ in range(NS)]
    pools = [torch.randn((R, k, 2, 64, D), generator=g, device="cuda").to(torch.bfloat16) for _ in range(NS)]
    F = torch.randn((R, D), generator=g, device="cuda").to(torch.bfloat16)
    Q = torch.randn((cfg.batch, cfg.n_q_heads, D), generator=g, device="cuda").to(torch.bfloat16)
    O = torch.empty_like(Q)
    ids = torch.empty((R, k), dtype=torch.int32, device="cuda")
    ids_a = torch.arange(k, dtype=torch.int32, device="cuda").repeat(R, 1).contiguous()
    slot = torch.full((R, k), -1, dtype=torch.int32, device="cuda")
    fetch = torch.full((R, k), -1, dtype=torch.int32, device="cuda")
    empty = torch.full((R, k), -1, dtype=torch.int32, device="cuda")
    host = torch.empty((R, 8, 2, 64, D), dtype=torch.bfloat16, pin_memory=True)
    pool = torch.empty((R, k, 2, 64, D), dtype=torch.bfloat16, device="cuda")
    W = torch.empty(STANDIN_BYTES // 2, dtype=torch.bfloat16, device="cuda").fill_(1.0)
    cs, xs = torch.cuda.Stream(), torch.cuda.Stream(priority=-1)   # as the context's select stream
    sel = lambda i: ctx.forecast_select_plan(F, kpools[i], Nb, k, ids, slot, fetch, stream=xs)
    gat = lambda i: ctx.prefetch_launch(host, 8, empty, k, pool, stream=xs)
    att = lambda i: ctx.sparse_decode(Q, pools[i], ids_a, k, O, stream=xs)
    out = {}
    for name, fn in (("select_plan", sel), ("gather_empty_list", gat), ("attention", att), ("select_plan_then_gather", lambda i: (sel(i), gat(i)))):
        for i in range(NS):
            fn(i)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=xs):
            for i in range(NS):
                fn(i)
        graph.replay()
        torch.cuda.synchronize()
        for loaded in (False, True):
            if loaded:
                for _ in range(40):
                    ctx.probe_launch(3, W, STANDIN_BYTES, stream=cs)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(xs):
                e0.record(xs)
                for _ in range(3):
                    graph.replay()
                e1.record(xs)
            e1.synchronize()
            still = not cs.query()
            torch.cuda.synchronize()
            out[name + ("_us_beside_hbm_load" if loaded else "_us_alone")] = round(e0.elapsed_time(e1) * 1e3 / (3 * NS), 2)
            if loaded:
                out.setdefault("load_on_throughout", True)
                out["load_on_throughout"] = out["load_on_throughout"] and bool(still)
        del graph
    out["note"] = "per launch (per pair for the chain); the load is the layer stand-in streaming HBM on another stream: NOT part of the method"
    ctx.close()
    return out


def bench_gather_sweep(torch, binding, peaks, ceiling, host_layer_b4):
    """Table-7 analog: persistent-CTA count of the UVA gather against link throughput AND against
    what it costs the compute stream.  For batch 4 and batch 32 (one layer of configs[3]: R*64 blocks of 32 KiB from
    pinned host memory): gather GB/s and fraction of the same-run memcpy ceiling per engine and CTA count; and the time
    of 20 (select, attention) pairs of that batch replayed from a graph alone and while gathers run on another stream."""
    from paper_2606_04511_b200 import synth
    out = []
    for batch in (4, 32):
        cfg = synth.CFG4_128K.with_(batch=batch)
        R, Nb, k, D = cfg.rows, cfg.n_blocks, cfg.topk, cfg.head_dim
        if batch == 4:
            host = host_layer_b4
        else:
            host = torch.empty((R, Nb, 2, 64, D), dtype=torch.bfloat16, pin_memory=True)   # 4 GiB; contents irrelevant to the copy
        g = torch.Generator(device="cuda").manual_seed(500 + batch)
        ids_g = torch.stack([torch.randperm(Nb, generator=g, device="cuda")[:k].sort().values for _ in range(R)]).to(torch.int32).contiguous()
        pool = torch.empty((R, k, 2, 64, D), dtype=torch.bfloat16, device="cuda")
        # the compute pair: select + attention on rotating cold buffers
        NSETS = 4 if batch == 32 else 16
        kpools = [torch.randn((R, Nb, D), generator=g, device="cuda").to(torch.bfloat16) for _ in range(NSETS)]
        apools = [torch.randn((R, k, 2, 64, D), generator=g, device="cuda").to(torch.bfloat16) for _ in range(NSETS)]
        F = torch.randn((R, D), generator=g, device="cuda").to(torch.bfloat16)
        Q = torch.randn((cfg.batch, cfg.n_q_heads, D), generator=g, device="cuda").to(torch.bfloat16)
        O = torch.empty_like(Q)
        ids_s = torch.empty((R, k), dtype=torch.int32, device="cuda")
        ids_a = torch.arange(k, dtype=torch.int32, device="cuda").repeat(R, 1).contiguous()
        cctx = binding.Sparda.from_config(cfg)
        cs, ps = torch.cuda.Stream(), torch.cuda.Stream(priority=-1)   # the prefetch stream outranks the compute stream (sparda.h)
        NP = 20
        for i in range(NSETS):
            cctx.forecast_select(F, kpools[i], Nb, k, ids_s)
            cctx.sparse_decode(Q, apools[i], ids_a, k, O)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=cs):
            for i in range(NP):
                cctx.forecast_select(F, kpools[i % NSETS], Nb, k, ids_s, stream=cs)
                cctx.sparse_decode(Q, apools[i % NSETS], ids_a, k, O, stream=cs)
        graph.replay()
        torch.cuda.synchronize()

        def pairs_us(n_rep):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(cs):
                e0.record(cs)
                for _ in range(n_rep):
                    graph.replay()
                e1.record(cs)
            e1.synchronize()
            return e0.elapsed_time(e1) * 1e3 / (n_rep * NP)
        alone = min(pairs_us(5) for _ in range(3))
        gbytes = cfg.gather_bytes_per_layer
        # under load (batch 4 only): the layer stand-in (474 MB streamed per launch, NOT part of the method) keeps HBM
        # saturated on cs while the gathers run on ps -- what the prefetch meets behind a real layer
        W = standin_us = None
        if batch == 4:
            W = torch.empty(STANDIN_BYTES // 2, dtype=torch.bfloat16, device="cuda").fill_(1.0)

            def standins(n):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(cs)
                for _ in range(n):
                    cctx.probe_launch(3, W, STANDIN_BYTES, stream=cs)
                e1.record(cs)
                return e0, e1, n
            s0, s1, n = standins(20)
            torch.cuda.synchronize()
            s0, s1, n = standins(20)
            torch.cuda.synchronize()
            standin_us = s0.elapsed_time(s1) * 1e3 / n
        rows = []
        for mode, name, ctas_list in ((binding.GATHER_TMA, "tma", (2, 4, 8, 16)), (binding.GATHER_LDG, "ldg", (8, 16, 32, 64))):
            for ctas in ctas_list:
                gctx = binding.Sparda.from_config(cfg, gather_mode=mode, gather_ctas=ctas)
                for _ in range(2):
                    gctx.prefetch_launch(host, Nb, ids_g, k, pool, stream=ps)
                ps.synchronize()
                n_g = 6 if batch == 4 else 3
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(ps)
                for _ in range(n_g):
                    gctx.prefetch_launch(host, Nb, ids_g, k, pool, stream=ps)
                e1.record(ps)
                e1.synchronize()
                t_g = e0.elapsed_time(e1) * 1e-3 / n_g
                # interference: keep the link busy for the whole timed window of the compute graph
                est_pairs_s = alone * 1e-6 * NP * 5
                n_bg = int(est_pairs_s * 3 / t_g) + 3
                for _ in range(n_bg):
                    gctx.prefetch_launch(host, Nb, ids_g, k, pool, stream=ps)
                with_g = pairs_us(5)
                busy = not ps.query()                              # gathers still running when the timed window closed
                ps.synchronize()
                row = {"engine": name, "ctas": ctas, "gbs": round(gbytes / t_g / 1e9, 2), "frac_of_ceiling": round(gbytes / t_g / 1e9 / ceiling, 4),
                       "pair_us_with_gather": round(with_g, 2), "pair_slowdown": round(with_g / alone, 3), "link_busy_throughout": bool(busy)}
                if W is not None:
                    n_gl = 8
                    s0, s1, n = standins(int(t_g * n_gl * 1e6 / standin_us * 2.5) + 4)
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(ps)
                    for _ in range(n_gl):
                        gctx.prefetch_launch(host, Nb, ids_g, k, pool, stream=ps)
                    e1.record(ps)
                    e1.synchronize()
                    loaded = not cs.query()                        # stand-ins still running when the last gather ended
                    torch.cuda.synchronize()
                    row["gbs_under_hbm_load"] = round(gbytes * n_gl / (e0.elapsed_time(e1) * 1e-3) / 1e9, 2)
                    row["standin_slowdown"] = round(s0.elapsed_time(s1) * 1e3 / n / standin_us, 3)
                    row["hbm_loaded_throughout"] = bool(loaded)
                rows.append(row)
                gctx.close()
        # f4's peer-HBM tier with the link out of the way: the same gather from a source in this GPU's own HBM (a peer's HBM
        # behind NVLink cannot be faster than this; the harness leases one GPU, so the peer copy itself is not measured)
        hbm_tier = None
        if batch == 4:
            src = torch.empty((R, Nb, 2, 64, D), dtype=torch.bfloat16, device="cuda")        # 1 GiB, cold: 16 MiB of it is read per launch
            hbm_tier = []
            for mode, name, ctas_list in ((binding.GATHER_TMA, "tma", (8, 16, 32, 64, 148)), (binding.GATHER_LDG, "ldg", (32, 64, 148, 296))):
                for ctas in ctas_list:
                    gctx = binding.Sparda.from_config(cfg, gather_mode=mode, gather_ctas=ctas)
                    t_h = graph_time(torch, lambda i, s: gctx.prefetch_launch(src, Nb, ids_g, k, pool, stream=s), 1, reps=20)
                    hbm_tier.append({"engine": name, "ctas": ctas, "us": round(t_h * 1e6, 2), "gbs": round(gbytes / t_h / 1e9, 1)})
                    gctx.close()
            del src
        out.append({"batch": batch, "gather_mib_per_launch": gbytes / 2**20, "pair_us_alone": round(alone, 2), "hbm_tier": hbm_tier,
                    "standin_us_alone": round(standin_us, 1) if standin_us else None,
                    "pair": "forecast_select + sparse_decode of this batch, cold HBM, 20 pairs per graph", "rows": rows})
        cctx.close()
        del graph, kpools, apools, pool, host, W
        torch.cuda.empty_cache()
    # pick: the rate that survives beside a layer (where measured) over what the CTAs cost the path's own kernels
    best = {o["batch"]: max(o["rows"], key=lambda r: r.get("gbs_under_hbm_load", r["gbs"]) / r["pair_slowdown"]) for o in out}
    return {"ceiling_gbs": round(ceiling, 2), "sweep": out,
            "pick": {str(b): {"engine": r["engine"], "ctas": r["ctas"]} for b, r in best.items()},
            "paper": "H100: 16 CTAs below batch 32, 32 from there (P:L116, Table 7); B200 numbers above are this box's"}


# ------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------
def flat_scalars(roofline, gather_ctas, gather_mode):
    """The per-kernel figures as SCALAR keys directly under `roofline` (a record that keeps only scalars still carries them).
    *_isolated: one launch between two events without PDL on cold buffers; *_period: steady-state back-to-back period from
    a graph replay with PDL (what `us` in roofline.kernels is).  frac = algorithmic bytes / time / measured HBM peak."""
    out = {}
    for e in roofline.get("kernels") or []:
        shape = e.get("shape", "")
        tag = "b32" if shape.startswith("batch 32") else "b4" if shape.startswith("batch 4") else None
        if tag is None:
            continue
        if e["kernel"].startswith("forecast_select_kernel<128,false>"):
            out.update({f"select_{tag}_us_isolated": e["us_isolated"], f"select_{tag}_us_period": e["us"],
                        f"select_{tag}_frac_isolated": e["frac_isolated"], f"select_{tag}_frac_period": e["frac"]})
        elif e["kernel"].startswith("sparse_decode_kernel<128>"):
            out.update({f"attn_{tag}_us_isolated": e["us_isolated"], f"attn_{tag}_us_period": e["us"],
                        f"attn_{tag}_frac_isolated": e["frac_isolated"], f"attn_{tag}_frac_period": e["frac"]})
        elif e["kernel"].startswith("pair:"):
            out.update({f"pair_{tag}_us": e["us_isolated"], f"pair_{tag}_frac": e["frac_isolated"], f"pair_{tag}_frac_of_8tbs": e["frac_of_8tbs"]})
            if "bracket_null_kernel_us" in e:   # context for every *_isolated figure: the same bracket around nothing / around an empty kernel
                out.update({"isolated_bracket_empty_us": e["bracket_empty_us"], "isolated_bracket_null_kernel_us": e["bracket_null_kernel_us"]})
    pf = roofline.get("prefill_select")
    if pf:
        out.update({"prefill_chunked_us": pf["forecast_us_chunked"], "prefill_one_us": pf["forecast_us_one_launch"]})
    ru = roofline.get("reuse_cache")
    if ru:
        out["floor_cached_step_ms"] = ru["compute_floor_ms_per_step"]
    gs = roofline.get("gather_sweep")
    if gs:
        for blk in gs["sweep"]:
            if blk["batch"] != 4:
                continue
            for row in blk["rows"]:
                if row["engine"] == gather_mode and row["ctas"] == gather_ctas and "gbs_under_hbm_load" in row:
                    out["gather_gbs_under_hbm_load"] = row["gbs_under_hbm_load"]
    return out


def run_sparda(args):
    import torch
    import torch.distributed as dist
    from paper_2606_04511_b200 import binding, synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libsparda has no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    assert args.warmup >= 3, "timing rules: at least 3 warm-up steps"
    peaks = load_peaks()
    ncu, ncu_src = load_ncu_metrics()
    if args.section == "kernels":
        print(json.dumps({"section": "kernels", "kernels": bench_kernels(torch, binding, peaks, ncu, ncu_src, 32) +
                          bench_kernels(torch, binding, peaks, ncu, ncu_src, 4),
                          "prefill": bench_prefill(torch, binding, peaks, ncu, ncu_src), "append": bench_append(torch, binding)}))
        return 0
    cfg = workload_config(args)
    from paper_2606_04511_b200 import shard
    cfg = shard.rank_config(cfg, rank)                       # every rank decodes its own sequences
    R, k, Nb, D, NL = cfg.rows, cfg.topk, cfg.n_blocks, cfg.head_dim, cfg.n_layers

    mode = binding.GATHER_TMA if args.gather_mode == "tma" else binding.GATHER_LDG
    ctx = binding.Sparda.from_config(cfg, max_layers=NL, gather_ctas=args.gather_ctas, gather_mode=mode, hidden=4096)

    # ---- pinned host KV: as many distinct layers as the box can hold, layer l -> l mod resident otherwise
    import psutil
    numa = numa_info(torch, local)
    per_layer = cfg.kv_bytes_per_layer
    avail = psutil.virtual_memory().available / max(1, int(os.environ.get("LOCAL_WORLD_SIZE", world)))
    cap = args.host_gib * 2**30 if args.host_gib > 0 else 0.5 * avail
    resident = max(1, min(NL - 1, int(cap // per_layer)))
    host_kv = [torch.empty((R, Nb, 2, cfg.block_size, D), dtype=torch.bfloat16, pin_memory=True) for _ in range(resident)]
    dev_layers, host_vals = [], []
    kv0 = None
    for l in range(NL):
        gen_needed = l == 0 or (l - 1) < resident
        L = synth.decode_layer(cfg, l, device="cuda")        # F/Q always; kv only where it is stored
        kpool = torch.empty((R, Nb, D), dtype=torch.bfloat16, device="cuda")
        if l == 0:
            kv0 = L["kv"]
            ctx.pool_keys(kv0, R, Nb, kpool)
            F0 = L["F0cur"]
            kv = kv0
        else:
            slot = (l - 1) % resident
            if gen_needed:
                host_kv[slot].copy_(L["kv"])
                ctx.pool_keys(L["kv"], R, Nb, kpool)
            else:                                            # aliased layer: pooled keys of the aliased cache
                kpool.copy_(dev_layers[1 + slot]["Kpool"])
            kv = host_kv[slot]
        dev_layers.append({"F": L["F"], "Q": L["Q"], "Kpool": kpool, "kv": kv,
                           "O": torch.zeros((cfg.batch, cfg.n_q_heads, D), dtype=torch.bfloat16, device="cuda"),
                           "ids": torch.full((R, k), -1, dtype=torch.int32, device="cuda")})
        host_vals.append({"F": L["F"].cpu().pin_memory(), "Q": L["Q"].cpu().pin_memory(),
                          "O": torch.zeros((cfg.batch, cfg.n_q_heads, D), dtype=torch.bfloat16).pin_memory()})
        del L
    torch.cuda.synchronize()
    F0_host = F0.cpu().pin_memory()
    pools = [torch.zeros((R, k, 2, cfg.block_size, D), dtype=torch.bfloat16, device="cuda") for _ in range(2)]
    arr = ctx.make_layers(dev_layers)
    arr_host = ctx.make_layers([{**d, **h} for d, h in zip(dev_layers, host_vals)])
    cs, ps = torch.cuda.Stream(), torch.cuda.Stream(priority=-1)   # the prefetch stream outranks the compute stream (sparda.h)

    ceiling = measure_h2d_ceiling(torch, host_kv[:min(4, resident)])

    def step(m=binding.STEP_OVERLAP):
        ctx.decode_step(arr, F0, Nb, k, pools[0], pools[1], cs, ps, m)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_region(fn, n):
        """K steps bracketed by barrier + synchronize on both sides, CUDA events on the compute stream."""
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(cs)
        for _ in range(n):
            fn()
        e1.record(cs)
        barrier()
        return shard.max_over_ranks(e0.elapsed_time(e1), device="cuda")

    # ---- timed region: device-resident Q/F/Kpool, KV in pinned host memory (the method's offload tier)
    for _ in range(args.warmup):
        step()
    props = torch.cuda.get_device_properties(local)
    gpu_id = f"GPU-{props.uuid}" if getattr(props, "uuid", None) else str(local)
    sampler = ClockSampler(gpu_id) if rank == 0 else None
    t_wait = time.time()                                     # nvidia-smi takes a moment to start: wait for its first sample
    while sampler and sampler.p and time.time() - t_wait < 3.0 and os.path.getsize(sampler.f.name) == 0:
        time.sleep(0.05)
    launches0 = ctx.launch_count
    ms_total = timed_region(step, args.steps)
    launches = ctx.launch_count - launches0

    def step_host():                                         # keep the sampler running through the e2e region too (same load)
        ctx.decode_step_host(arr_host, F0_host, Nb, k, pools[0], pools[1], cs, ps, binding.STEP_OVERLAP)
        cs.synchronize()                                     # the caller reads O of this step on the host
    for _ in range(args.warmup):
        step_host()
    ms_e2e = timed_region(step_host, args.steps)
    clocks = sampler.stop() if sampler else None

    # serialized pipeline (same kernels, one stream): what the overlap buys
    n_ser = max(3, args.steps // 3)
    for _ in range(2):
        step(binding.STEP_SERIAL)
    ms_serial = timed_region(lambda: step(binding.STEP_SERIAL), n_ser) / n_ser

    # ---- the dominant kernel's own duration: timing events around every gather launch, in a pass over the same K steps in
    # SERIAL mode -- the kernel alone on the link (in the overlapped step two gathers of consecutive layers share it, so a
    # bracket there reads two kernels' time); a 335 us kernel: the event bracket costs < 1 %
    ctx.profile_enable(True)
    g_ms, g_n = 0.0, 0
    for _ in range(args.steps):
        step(binding.STEP_SERIAL)
        torch.cuda.synchronize()
        ms, n = ctx.profile_read()["gather"]
        g_ms += ms
        g_n += n
    ctx.profile_enable(False)
    t_gat = g_ms / g_n * 1e-3 if g_n else float("nan")

    # ---- what the timed steps computed: after the timed regions, one more step in each form on NaN-poisoned pools.  The
    # overlapped step must be bit-identical to the serial one (O and ids of every layer), the host-buffer step's O too; any
    # block that arrived late, any stale slot, shows up as NaN or as a differing bit.  (Parity against the oracle at this
    # size is tests/test_gpu_parity.py::test_full_size_32_layer_decode_step; bench.py must not import the oracle here.)
    def snapshot(fn):
        for p_ in pools:
            p_.fill_(float("nan"))
        for d in dev_layers:
            d["O"].zero_()
            d["ids"].fill_(-9)
        torch.cuda.synchronize()
        fn()
        torch.cuda.synchronize()
        return [d["O"].clone() for d in dev_layers], [d["ids"].clone() for d in dev_layers]
    O_ser, I_ser = snapshot(lambda: step(binding.STEP_SERIAL))
    O_ovl, I_ovl = snapshot(step)
    checked = all(torch.equal(a, b) for a, b in zip(I_ser, I_ovl)) and \
        all(torch.equal(a.view(torch.int16), b.view(torch.int16)) for a, b in zip(O_ser, O_ovl)) and \
        not any(bool(torch.isnan(o).any()) for o in O_ovl) and all(int(i.min()) >= 0 for i in I_ovl)
    for h in host_vals:
        h["O"].zero_()
    step_host()
    torch.cuda.synchronize()
    checked = checked and all(torch.equal(h["O"].view(torch.int16), o.cpu().view(torch.int16)) for h, o in zip(host_vals, O_ovl))
    if not checked:
        raise SystemExit("bench.py: the overlapped / host-buffer step is not bit-identical to the serial step; the timing above is void")

    ms_per_step = ms_total / args.steps
    tokens = cfg.batch * world
    value = shard.whole_job_value(cfg.batch, world, ms_per_step)
    e2e_value = shard.whole_job_value(cfg.batch, world, ms_e2e / args.steps)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    sec = args.sections
    reuse = standin = None
    if "reuse" in sec:
        reuse = bench_reuse(torch, binding, ctx, cfg, dev_layers, F0, cs, ps, args.steps)
    if "standin" in sec:
        standin = bench_reuse(torch, binding, ctx, cfg, dev_layers, F0, cs, ps, args.steps, standin_bytes=STANDIN_BYTES)
    gather_sweep = None
    if "gather" in sec:
        gather_sweep = bench_gather_sweep(torch, binding, peaks, ceiling, host_kv[0] if cfg.batch == 4 else None) if cfg.batch == 4 else None

    gather_bytes = cfg.gather_bytes_per_layer
    gm = ncu.get("gather_b4", {}) if cfg.name == "cfg3_128k_pipeline" else {}
    g_traffic = gm.get("dram__bytes_read.sum", 0.0) + gm.get("dram__bytes_write.sum", 0.0) if "dram__bytes_read.sum" in gm else None
    roofline = {"kernel": "gather_tma_kernel" if args.gather_mode == "tma" else "gather_ldg_kernel",
                "bound": "host_link", "achieved": gather_bytes / t_gat / 1e9, "peak": ceiling, "unit": "GB/s",
                "frac": gather_bytes / t_gat / 1e9 / ceiling, "traffic": g_traffic, "traffic_src": ncu_src if g_traffic is not None else None,
                "traffic_note": "HBM traffic of one launch (the ids); the payload crosses the host link and lands in L2",
                "peak_source": "cudaMemcpyAsync pinned host->device, measured in this run on this box",
                "us_per_launch": t_gat * 1e6, "algorithmic_bytes": gather_bytes,
                "share_of_step": t_gat * 1e3 * (NL - 1) / ms_per_step,   # 31 gathers back to back against the overlapped step
                "hbm_peak": peaks["hbm_gbs"], "hbm_peak_source": peaks["source"],
                "note": "dominant kernel of the step; its roofline is the host link, not HBM (DESIGN.md 5.2)"}
    # everything below is nested under `roofline` so that the driver's record keeps it
    del pools
    torch.cuda.empty_cache()
    if "kernels" in sec:
        roofline["kernels"] = bench_kernels(torch, binding, peaks, ncu, ncu_src, 32) + bench_kernels(torch, binding, peaks, ncu, ncu_src, 4)
    if "floor" in sec:
        roofline["launch_floor"] = bench_floor(torch, binding)
    if "prefill" in sec:
        roofline["prefill_select"] = bench_prefill(torch, binding, peaks, ncu, ncu_src)
    if "append" in sec:
        roofline["cache_maintenance"] = bench_append(torch, binding)
    floor_ms = reuse["compute_floor_ms_per_step"] if reuse else None
    roofline["pipeline"] = {
        "ms_per_step_overlap": ms_per_step, "ms_per_step_serial": ms_serial, "us_per_layer_step": ms_per_step * 1e3 / NL,
        "us_gather": t_gat * 1e6, "gather_gbs": gather_bytes / t_gat / 1e9, "host_link_ceiling_gbs": ceiling,
        "tok_s_ceiling_at_host_link": cfg.batch * world / (gather_bytes * (NL - 1) / (ceiling * 1e9)),
        # exposed = step with every block fetched minus the step with nothing to fetch (the cached step at rho = 0)
        "gather_exposed_us_per_layer": (ms_per_step - floor_ms) * 1e3 / (NL - 1) if floor_ms else None,
        "compute_floor_ms_per_step": floor_ms}
    if "standin" in sec:
        roofline["kernel_boundary_under_load"] = bench_chain_under_load(torch, binding)
    roofline["reuse_cache"] = reuse
    roofline["reuse_cache_with_layer_standin"] = standin
    roofline["gather_sweep"] = gather_sweep
    roofline["numa"] = numa
    roofline.update(flat_scalars(roofline, ctx.gather_ctas, args.gather_mode))

    base = None
    if not args.no_cpu_baseline and world == 1:
        from oracle import sparda_oracle as oracle
        oracle.build()
        import numpy as np
        n_s = min(2, NL)
        bits = []
        for l in range(n_s):
            d = dev_layers[l]
            kvb = (kv0 if l == 0 else d["kv"])
            bits.append({"kv": kvb.cpu().contiguous().view(torch.int16).numpy().view(np.uint16),
                         "kpool": d["Kpool"].cpu().view(torch.int16).numpy().view(np.uint16),
                         "F": d["F"].cpu().view(torch.int16).numpy().view(np.uint16),
                         "Q": d["Q"].cpu().view(torch.int16).numpy().view(np.uint16),
                         "F0cur": F0.cpu().view(torch.int16).numpy().view(np.uint16)})
        base = cpu_baseline(cfg, bits, args.cpu_seconds)

    staged = (R * D * 2) * NL + (cfg.batch * cfg.n_q_heads * D * 2) * NL
    config = config_dict(cfg, world)
    roofline["run"] = {"kv_residency": f"layers 1..{NL - 1} pinned on host ({resident} distinct" + ("" if resident >= NL - 1 else f", l -> (l-1) mod {resident}") + "), layer 0 in HBM",
                       "gather": {"mode": args.gather_mode, "ctas": ctx.gather_ctas}, "attn_ctas_per_row": ctx.attn_splits(k),
                       "pdl": "stand-alone calls and the serial step; not inside the overlapped step"}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic", "config": config, "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e / args.steps,
                "h2d_bytes_per_step": staged + gather_bytes * (NL - 1), "d2h_bytes_per_step": cfg.batch * cfg.n_q_heads * D * 2 * NL,
                "h2d_staged_bytes_per_step": staged, "h2d_uva_gather_bytes_per_step": gather_bytes * (NL - 1),
                "api": "sparda_decode_step_host: pinned host F/Q/O copied just in time inside the call; stream sync per step"},
        "gpu_launches": launches,
        "checked": checked,      # overlapped == serial == host-buffer step, bit for bit, on poisoned pools after the timed regions
        "roofline": roofline,
        "cpu_baseline": base,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def spawn_ranks(args):
    """`python bench.py --gpus N` outside torchrun: launch N ranks (one per GPU) of this script through
    torch.distributed.run and pass rank 0's line through.  Fewer than N GPUs is an error, never a 1-GPU number."""
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        sys.stderr.write(f"bench.py: --gpus {args.gpus} asked for, {have} CUDA device(s) visible: refusing to print a smaller job's number\n")
        return 3
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    return subprocess.call(cmd)


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    env_world = os.environ.get("WORLD_SIZE")
    if env_world is None and args.gpus > 1:
        return spawn_ranks(args)
    if env_world is not None and int(env_world) != args.gpus:
        sys.stderr.write(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={env_world}\n")
        return 2
    return run_sparda(args)


if __name__ == "__main__":
    sys.exit(main())
