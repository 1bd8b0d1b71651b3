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

N > 1 (torchrun): every rank runs the same per-GPU workload on its own sequences (batch shards, no
collective on the data path -- SURVEY 8(e)); value = tokens all ranks decoded / max-over-ranks device time.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
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
    ap.add_argument("--no-kernels", action="store_true", help="skip the batch-32 per-kernel HBM roofline section")
    ap.add_argument("--section", default="all", choices=["all", "kernels"],
                    help="kernels: only the per-kernel sections (batch-32 select / attention, prefill selection); used for ncu captures")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the cpu_baseline sample")
    return ap.parse_args()


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": d.get("bf16_tflops"),
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained"), "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1700.0, "bf16_tflops_sustained": 1400.0, "source": "fallback (B200_PROFILING.md)"}


def workload_config(args):
    from paper_2606_04511_b200 import synth
    cfg = synth.CFG3_128K if args.workload == "cfg3" else synth.CFG4_128K
    if args.batch:
        cfg = cfg.with_(batch=args.batch)
    if args.layers:
        cfg = cfg.with_(n_layers=args.layers)
    return cfg


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
    fit in ~target_s seconds, scaled to the full layer count."""
    from oracle import sparda_oracle as oracle
    t0 = time.perf_counter()
    done = 0
    while done < 4 * cfg.n_layers:                          # whole layer-steps until ~target_s of CPU time
        l = done % cfg.n_layers
        lay = layers_bits[l % len(layers_bits)]
        prev = layers_bits[(l - 1) % len(layers_bits)]
        _oracle_layer_step(oracle, lay, lay["F0cur"] if l == 0 else prev["F"], cfg.topk, layer0=(l == 0))
        done += 1
        if time.perf_counter() - t0 >= target_s:
            break
    el = time.perf_counter() - t0
    per_step_s = el * cfg.n_layers / done
    return {"value": cfg.batch / per_step_s, "unit": UNIT, "cores": oracle.threads(), "kind": "oracle",
            "sample": f"{done} layer-steps (select + gather + sparse attention, batch {cfg.batch}, 128K, "
                      f"{cfg.n_layers} per decode step) in {el:.2f} s, scaled to one {cfg.n_layers}-layer step",
            "seconds_per_decode_step": per_step_s}


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
    sample = (f"each step = {n_sample} of {cfg.n_layers} layer-steps (layer 0 + one gathered layer) of the oracle at batch "
              f"{cfg.batch}, 128K, scaled to {cfg.n_layers} layers")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": per_step_s * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "batch": cfg.batch, "context": cfg.context, "layers": cfg.n_layers,
                       "topk": cfg.topk, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------
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


def bench_kernels_b32(torch, binding, peaks, args):
    """Per-kernel HBM rooflines at the batch-32 shape of BASELINE.json configs[3] (R = 64 rows, 2048 blocks,
    top-64, D = 128), where the ideal times (5 us select, 20 us attention) stand clear of the launch floor
    (SURVEY 8(d)).  Cold HBM: each launch works on the next of NSETS buffer sets, together larger than L2."""
    from paper_2606_04511_b200 import synth
    cfg = synth.CFG4_128K
    R, Nb, k, D = cfg.rows, cfg.n_blocks, cfg.topk, cfg.head_dim
    ctx = binding.Sparda.from_config(cfg)
    g = torch.Generator(device="cuda").manual_seed(40)
    NS_SEL, NS_ATT = 8, 4                                    # 8 x 32 MiB Kpool, 4 x 128 MiB pool: each ring > 126 MB L2
    kpools = [torch.randn((R, Nb, D), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16) for _ in range(NS_SEL)]
    Fs = [torch.randn((R, D), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16) for _ in range(NS_SEL)]
    pools = []
    for _ in range(NS_ATT):
        p = torch.empty((R, k, 2, 64, D), dtype=torch.bfloat16, device="cuda")
        p.copy_(torch.randn(p.shape, generator=g, device="cuda", dtype=torch.float32))
        pools.append(p)
    Q = torch.randn((cfg.batch, cfg.n_q_heads, D), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16)
    O = torch.empty_like(Q)
    ids = torch.empty((R, k), dtype=torch.int32, device="cuda")
    ids_att = torch.arange(k, dtype=torch.int32, device="cuda").repeat(R, 1).contiguous()
    st = torch.cuda.current_stream()

    def timed(fn, n_sets, reps=10):
        """reps passes over the n_sets buffer sets, captured once into a CUDA graph (the launches of these short kernels
        would otherwise be paced by the Python caller, not by the GPU) and replayed between two events."""
        for i in range(2 * n_sets):
            fn(i % n_sets, st)
        torch.cuda.synchronize()
        graph, cap = torch.cuda.CUDAGraph(), torch.cuda.Stream()
        with torch.cuda.graph(graph, stream=cap):
            for i in range(reps * n_sets):
                fn(i % n_sets, torch.cuda.current_stream())
        graph.replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        graph.replay()
        e1.record(st)
        e1.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / (reps * n_sets)

    t_sel = timed(lambda i, s: ctx.forecast_select(Fs[i], kpools[i], Nb, k, ids, stream=s), NS_SEL)
    t_att = timed(lambda i, s: ctx.sparse_decode(Q, pools[i], ids_att, k, O, stream=s), NS_ATT)
    sel_bytes = cfg.kpool_bytes_per_layer + R * D * 2 + R * k * 4
    att_bytes = cfg.gather_bytes_per_layer + 2 * cfg.batch * cfg.n_q_heads * D * 2 + R * k * 4
    # f3: the paper's geometry -- (32,16) compressed-key grid (4 keys per block), max-pool to blocks, budget 96 = 1 + 32 + 63
    del kpools
    grids = [torch.randn((R, 4 * Nb, D), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16) for _ in range(2)]
    ids96 = torch.empty((R, 96), dtype=torch.int32, device="cuda")
    ctx96 = binding.Sparda(cfg.batch, cfg.n_q_heads, cfg.n_kv_heads, D, Nb, 96)
    t_grid = timed(lambda i, s: ctx96.forecast_select_grid(Fs[i], grids[i], Nb, 96, ids96, n_init=1, n_local=32, stream=s), 2)
    grid_bytes = R * (4 * Nb - 1) * D * 2 + R * D * 2 + R * 96 * 4
    ctx96.close()
    del grids
    out = []
    for name, t, b in (("forecast_select_kernel<128>", t_sel, sel_bytes), ("sparse_decode_kernel<128>", t_att, att_bytes),
                       ("forecast_select_kernel<128,grid>", t_grid, grid_bytes)):
        out.append({"kernel": name, "workload": "cfg4 shape, batch 32, one layer, cold HBM (rotating buffer sets > L2), launches replayed from a CUDA graph",
                    "bound": "hbm", "us_per_launch": t * 1e6, "algorithmic_bytes": b, "achieved": b / t / 1e9,
                    "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": b / t / 1e9 / peaks["hbm_gbs"],
                    "frac_of_nominal_8tbs": b / t / 1e9 / 8000.0, "peak_source": peaks["source"], "traffic": None})
    # DRAM read + write bytes per launch of the same shapes from the committed ncu --set full captures
    out[0]["traffic"], out[0]["traffic_source"] = 33612800, "profiles/r1c_ncu_summary.md (prof_b32_select_c: dram read 33.61 MB, write 0)"
    out[1]["traffic"], out[1]["traffic_source"] = 134544640 + 3627776, "profiles/r1c_ncu_summary.md (prof_b32_attn_c: dram read 134.54 MB, 3.6 MB of evictions)"
    out[1]["attn_splits"] = ctx.attn_splits(k)
    out[2]["workload"] = ("f3 (reading q19, unpinned by the paper): batch 32, 2048 blocks x 4 compressed keys, max-pool to blocks, "
                          "top-96 = 1 initial + 32 local + 63 ranked; cold HBM (two 128 MiB grids > L2), CUDA-graph replay")
    ctx.close()
    del pools
    torch.cuda.empty_cache()
    return out


def bench_prefill(torch, binding, peaks_all):
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
    st = torch.cuda.current_stream()

    def chunked(fn, src):
        for r0 in range(0, T, cfg.chunk):
            fn(src, kpool, T, Nb, r0, cfg.chunk, k, part)

    def timed(fn, reps):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for _ in range(reps):
            fn()
        e1.record(st)
        e1.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / reps

    n0 = ctx.launch_count
    t_one = timed(lambda: ctx.prefill_select(P["F"], kpool, T, Nb, 0, T, k, ids), 20)
    t_chunk = timed(lambda: chunked(ctx.prefill_select, P["F"]), 10)
    t_base = timed(lambda: chunked(ctx.prefill_select_baseline, P["Q"]), 3)
    launches = ctx.launch_count - n0
    # causal contraction: row i multiplies min(Nb, (i+1)//64) pooled keys of width D
    ncand = sum(min(Nb, (i + 1) // 64) for i in range(T))
    flops = 2.0 * Hkv * ncand * D
    bf16_peak = peaks_all.get("bf16_tflops_sustained") or peaks_all.get("bf16_tflops") or 1400.0
    ranked_rows = Hkv * sum(1 for i in range(T) if (i + 1) // 64 > k)
    out = {
        "workload": f"{cfg.name}: T={T}, {Hkv} groups, {Nb} pooled keys, top-{k}, {cfg.chunk}-row chunks",
        "forecast_select_us_per_pass_chunked": t_chunk * 1e6, "forecast_select_us_one_launch": t_one * 1e6,
        "baseline_selector_us_per_pass_chunked": t_base * 1e6, "selection_cost_ratio_baseline_over_forecast": t_base / t_chunk,
        "tokens_per_s_selection_only": T / t_chunk, "gpu_launches": launches,
        "ns_per_ranked_row": t_chunk * 1e9 / ranked_rows,
        "roofline": {"kernel": "prefill_select_kernel<128,false>", "bound": "tensor", "achieved": flops / t_chunk / 1e12,
                     "peak": bf16_peak, "unit": "TFLOP/s", "frac": flops / t_chunk / 1e12 / bf16_peak, "traffic": None,
                     "algorithmic_flops": flops,
                     "note": "the contraction is ~1% of the kernel; the fused per-row top-k (plain ALU, DESIGN.md 5.5) is the cost"},
        # the bound that matters: warp instructions executed by the one-launch kernel (ncu smsp__inst_executed.sum,
        # profiles/r1c_ncu_summary.md prof_prefill_c) over the live duration, against 148 SMs x 4 schedulers x 1 warp-instr/clk
        "roofline_alu": {"kernel": "prefill_select_kernel<128,false,false> (whole sequence, one launch)", "bound": "alu",
                         "achieved": 40551465 / t_one / 1e9, "peak": 148 * 4 * 1.965, "unit": "G warp-instr/s",
                         "frac": 40551465 / t_one / 1e9 / (148 * 4 * 1.965), "us_per_launch": t_one * 1e6,
                         "executed_warp_instructions": 40551465},
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
        out[f"us_per_append_{where}"] = e0.elapsed_time(e1) * 1e3 / (5 * 64)
        del graph, kv
    out["workload"] = f"append_kv_kernel<128>, R = {R} rows (batch 32), one token per launch, 64 launches per graph"
    out["bytes_per_launch"] = R * D * 2 * 2 + 2 * R * D * 4
    ctx.close()
    return out


def bench_reuse(torch, binding, ctx, cfg, dev_layers, F0, cs, ps, steps):
    """SURVEY 8(f) f1 / 8(d) "gather hidden": the same 32-layer decode step with the previous step's blocks kept per
    layer, so only newly selected blocks cross the host link.  The Forecast alternates between F_A and
    F_B = bf16(F_A + alpha * N(0,1)) from step to step; alpha sets how much the selection drifts, the fresh-fetch
    fraction rho is MEASURED (blocks fetched / blocks selected, from the plan kernel's counters).  alpha = 0 gives
    rho = 0: the compute-only floor of the step; exposed gather time = step(rho) - step(0)."""
    R, k, Nb, D, NL = cfg.rows, cfg.topk, cfg.n_blocks, cfg.head_dim, cfg.n_layers
    g = torch.Generator(device="cuda").manual_seed(777)
    layers = []
    for l, d in enumerate(dev_layers):
        e = dict(d)
        e["F"] = d["F"].clone()
        if l:
            e["pool"] = torch.zeros((R, k, 2, cfg.block_size, D), dtype=torch.bfloat16, device="cuda")
            e["slot_ids"] = torch.full((R, k), -1, dtype=torch.int32, device="cuda")
            e["fetch"] = torch.full((R, k), -1, dtype=torch.int32, device="cuda")
            e["n_fetch"] = torch.zeros((R,), dtype=torch.int32, device="cuda")
        layers.append(e)
    arr = ctx.make_cached_layers(layers)
    F0w = F0.clone()
    FA = [d["F"].clone() for d in dev_layers]
    noise = [torch.randn(d["F"].shape, generator=g, device="cuda") for d in dev_layers]
    noise0 = torch.randn(F0.shape, generator=g, device="cuda")

    def set_F(which, alpha):
        for l, e in enumerate(layers):
            e["F"].copy_(FA[l] if which == 0 else (FA[l].float() + alpha * noise[l]).to(torch.bfloat16))
        F0w.copy_(F0 if which == 0 else (F0.float() + alpha * noise0).to(torch.bfloat16))

    def one(which, alpha):
        with torch.cuda.stream(cs):                          # the Forecast of this step is produced on the compute stream
            set_F(which, alpha)
        ctx.decode_step_cached(arr, F0w, Nb, k, cs, ps, binding.STEP_OVERLAP)

    out = []
    for alpha in (0.0, 0.05, 0.1, 0.2, 0.4, 0.8, 1e9):
        for e in layers[1:]:
            e["slot_ids"].fill_(-1)
        for i in range(4):
            one(i & 1, alpha)
        torch.cuda.synchronize()
        fetched = 0
        for i in range(2):                                   # periodic state: count one A step and one B step
            one(i & 1, alpha)
            torch.cuda.synchronize()
            fetched += sum(int(e["n_fetch"].sum().item()) for e in layers[1:])
        rho = fetched / (2.0 * (NL - 1) * R * k)
        n = max(4, steps - steps % 2)
        torch.cuda.synchronize()
        # one A step and one B step captured into a CUDA graph (two streams, events and the F copies included): the
        # ~300 enqueue calls of a step would otherwise pace this compute-sized step from the host
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=cs):
            for i in range(2):
                set_F(i & 1, alpha)
                ctx.decode_step_cached(arr, F0w, Nb, k, cs, ps, binding.STEP_OVERLAP)
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
        out.append({"alpha": alpha if alpha < 1e8 else "independent", "fresh_fetch_fraction": rho, "ms_per_step": ms,
                    "tok_s": cfg.batch / (ms * 1e-3), "host_link_mib_per_step": rho * (NL - 1) * cfg.gather_bytes_per_layer / 2**20})
    floor = out[0]["ms_per_step"]
    for o in out:
        o["gather_exposed_us_per_layer"] = max(0.0, (o["ms_per_step"] - floor) * 1e3 / (NL - 1))
    del layers, arr
    torch.cuda.empty_cache()
    return {"workload": f"{cfg.name}, per-layer persistent pools ({(NL - 1) * cfg.gather_bytes_per_layer / 2**20:.0f} MiB of HBM), "
                        "Forecast alternating F_A / F_A + alpha*N(0,1) (F copied on the device each step, inside the timed region); steps replayed from a CUDA graph",
            "compute_floor_ms_per_step": floor, "sweep": out}


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
    if args.section == "kernels":
        print(json.dumps({"section": "kernels", "roofline_kernels": bench_kernels_b32(torch, binding, peaks, args),
                          "prefill_select": bench_prefill(torch, binding, peaks), "cache_maintenance": bench_append(torch, binding)}))
        return 0
    cfg = workload_config(args)
    from paper_2606_04511_b200 import shard
    cfg = shard.rank_config(cfg, rank)                       # every rank decodes its own sequences
    R, k, Nb, D, NL = cfg.rows, cfg.topk, cfg.n_blocks, cfg.head_dim, cfg.n_layers

    mode = binding.GATHER_TMA if args.gather_mode == "tma" else binding.GATHER_LDG
    ctx = binding.Sparda.from_config(cfg, max_layers=NL, gather_ctas=args.gather_ctas, gather_mode=mode)

    # ---- pinned host KV: as many distinct layers as the box can hold, layer l -> l mod resident otherwise
    import psutil
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
    cs, ps = torch.cuda.Stream(), torch.cuda.Stream()

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
    time.sleep(0.15)
    launches0 = ctx.launch_count
    ms_total = timed_region(step, args.steps)
    launches = ctx.launch_count - launches0
    # keep the sampler running through the e2e region too (same load)
    def step_host():
        ctx.decode_step_host(arr_host, F0_host, Nb, k, pools[0], pools[1], cs, ps, binding.STEP_OVERLAP)
        cs.synchronize()                                     # the caller reads O of this step on the host
    for _ in range(args.warmup):
        step_host()
    ms_e2e = timed_region(step_host, args.steps)
    clocks = sampler.stop() if sampler else None

    # serialized pipeline (same kernels, one stream): what the overlap buys
    for _ in range(2):
        step(binding.STEP_SERIAL)
    ms_serial = timed_region(lambda: step(binding.STEP_SERIAL), max(3, args.steps // 3)) / max(3, args.steps // 3)

    reuse = None
    if not args.no_kernels and rank == 0:
        reuse = bench_reuse(torch, binding, ctx, cfg, dev_layers, F0, cs, ps, args.steps)

    # ---- per-kernel device times inside the pipeline (second pass over the same K steps, timing events on)
    ctx.profile_enable(True)
    prof = {"select": [0.0, 0], "gather": [0.0, 0], "attn": [0.0, 0]}
    for _ in range(args.steps):
        step()
        torch.cuda.synchronize()
        for kind, (ms, n) in ctx.profile_read().items():
            prof[kind][0] += ms
            prof[kind][1] += n
    ctx.profile_enable(False)

    ms_per_step = ms_total / args.steps
    tokens = cfg.batch * world
    value = shard.whole_job_value(cfg.batch, world, ms_per_step)
    e2e_value = shard.whole_job_value(cfg.batch, world, ms_e2e / args.steps)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    def per(kind):
        ms, n = prof[kind]
        return ms / n * 1e-3 if n else float("nan")
    t_sel, t_gat, t_att = per("select"), per("gather"), per("attn")
    gather_bytes = cfg.gather_bytes_per_layer
    sel_bytes = cfg.kpool_bytes_per_layer + R * D * 2 + R * k * 4
    att_bytes = cfg.gather_bytes_per_layer + 2 * cfg.batch * cfg.n_q_heads * D * 2 + R * k * 4
    roofline = {"kernel": "gather_tma_kernel" if args.gather_mode == "tma" else "gather_ldg_kernel",
                "bound": "host_link", "achieved": gather_bytes / t_gat / 1e9, "peak": ceiling, "unit": "GB/s",
                "frac": gather_bytes / t_gat / 1e9 / ceiling,
                "traffic": 56064 if cfg.name == "cfg3_128k_pipeline" else None,
                "traffic_note": "DRAM bytes of one batch-4 launch (ncu, profiles/r1c_ncu_summary.md): the ids only; the payload crosses the "
                                "host link (sysmem read sectors x 32 B = the algorithmic 16 MiB, profiles/r1_ncu_summary.md) and lands in L2",
                "peak_source": "cudaMemcpyAsync pinned host->device, measured in this run on this box",
                "us_per_launch": t_gat * 1e6, "algorithmic_bytes": gather_bytes,
                "share_of_step": prof["gather"][0] / args.steps / ms_per_step,
                "note": "dominant kernel of the step; its roofline is the host link, not HBM (DESIGN.md 'Kernels')"}
    kernels = [
        {"kernel": "forecast_select_kernel<128>", "workload": f"{cfg.name} in-pipeline", "bound": "hbm",
         "us_per_launch": t_sel * 1e6, "algorithmic_bytes": sel_bytes, "achieved": sel_bytes / t_sel / 1e9,
         "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": sel_bytes / t_sel / 1e9 / peaks["hbm_gbs"], "traffic": None,
         "note": "launch-latency-sized at batch 4 (ideal 0.64 us); the event bracket of the profiling pass includes the gaps of the "
                 "eager enqueue -- device time per launch is 8.7 us (profiles/r1c_launches.csv)"},
        {"kernel": "sparse_decode_kernel<128>", "workload": f"{cfg.name} in-pipeline (pool just written by the gather: L2-warm)",
         "bound": "hbm", "us_per_launch": t_att * 1e6, "algorithmic_bytes": att_bytes, "achieved": att_bytes / t_att / 1e9,
         "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": att_bytes / t_att / 1e9 / peaks["hbm_gbs"], "traffic": None,
         "note": "launch-latency-sized at batch 4 (ideal 2.6 us); event bracket as above -- device time per launch is 10.1 us "
                 "(profiles/r1c_launches.csv)"},
    ]
    prefill = append = None
    if not args.no_kernels:
        del pools
        kernels += bench_kernels_b32(torch, binding, peaks, args)
        prefill = bench_prefill(torch, binding, peaks)
        append = bench_append(torch, binding)

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
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": cfg.name, "batch_per_gpu": cfg.batch, "global_batch": tokens, "context": cfg.context,
                   "layers": NL, "q_heads": cfg.n_q_heads, "kv_heads": cfg.n_kv_heads, "head_dim": D, "block": cfg.block_size,
                   "topk": k, "parallelism": f"batch shards x{world}, no collective",
                   "kv_residency": f"layers 1..{NL - 1} in pinned host memory ({resident} distinct resident layers"
                                   + ("" if resident >= NL - 1 else f", layer l -> (l-1) mod {resident}") + "), layer 0 in HBM",
                   "fresh_fetch_fraction": 1.0,
                   "l2": f"inputs larger than L2: {(cfg.kpool_bytes_per_layer * NL + gather_bytes * (NL - 1)) / 2**20:.0f} MiB touched per step",
                   "gather": {"mode": args.gather_mode, "ctas": ctx.gather_ctas}, "attn_splits": ctx.attn_splits(k)},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e / args.steps,
                "h2d_bytes_per_step": staged + gather_bytes * (NL - 1), "d2h_bytes_per_step": cfg.batch * cfg.n_q_heads * D * 2 * NL,
                "h2d_staged_bytes_per_step": staged, "h2d_uva_gather_bytes_per_step": gather_bytes * (NL - 1),
                "api": "sparda_decode_step_host (pinned host F/Q/O, copies enqueued just in time inside the call) + stream sync per step"},
        "gpu_launches": launches,
        "roofline": roofline,
        "roofline_kernels": kernels,
        "cpu_baseline": base,
        "prefill_select": prefill,
        "reuse_cache": reuse,
        "cache_maintenance": append,
        "pipeline": {"ms_per_step_overlap": ms_per_step, "ms_per_step_serial": ms_serial,
                     "us_per_layer_step": ms_per_step * 1e3 / NL,
                     "us_select": t_sel * 1e6, "us_gather": t_gat * 1e6, "us_attn": t_att * 1e6,
                     "gather_exposed_us_per_layer": max(0.0, (ms_per_step * 1e3 - (t_sel * NL + t_att * NL) * 1e6) / max(1, NL - 1)),
                     "host_link_ceiling_gbs": ceiling, "gather_gbs": gather_bytes / t_gat / 1e9,
                     "tok_s_ceiling_at_host_link": cfg.batch * world / (gather_bytes * (NL - 1) / (ceiling * 1e9))},
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_sparda(args)


if __name__ == "__main__":
    sys.exit(main())
