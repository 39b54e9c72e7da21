#!/usr/bin/env python
"""bench.py — MosaicKV decode hot path on B200: PackedAttention us/layer and % of the HBM roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload llama8b-128k-b8] [--layers n]
    python bench.py --impl reference ...        # the CPU oracle on a bounded sample (slow on purpose)

A step = one decode step over all layers of the workload: per layer mkv_select (score + top-k on
the packed block keys) and mkv_packed_attention (packed QK, softmax, PV, split-K combine), on a
cache that was compressed (mkv_segment_loss -> mkv_strategy_quantile -> mkv_compress_segment,
timed and reported under "compress") before the timed region.  Consecutive layers touch different
packed arenas (1.9 GB each at config 2), so inputs are far larger than L2 (126 MB).

Prints ONE JSON line (see DESIGN.md "Measurement" for every key).
"""
import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "PackedAttention us/layer (8B-shape, 128K ctx, batch 8)"
UNIT = "us/layer"
NOMINAL_HBM_GBS = 8000.0
FALLBACK_HBM_GBS = 6650.0
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the committed `ncu --set full` captures.  NOT measured by
# this run: "traffic" carries the number of the capture (null for a workload without one) and "traffic_from_capture"
# names the file it came from.
NCU_CAPTURE = {"llama8b-128k-b8": {"source": "profiles/r3/ncu_decode_config2.md (ncu --set full, first launch of each kernel)",
                                   "attention": 28732672, "score+topk": 125498880},
               "llama8b-1m-b1": {"source": "profiles/r2/ncu_decode_config3.md", "attention": None, "score+topk": None},
               "qwen7b-64k-b16": {"source": "profiles/r2/ncu_decode_config4.md", "attention": None, "score+topk": None}}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="llama8b-128k-b8")
    ap.add_argument("--layers", type=int, default=0, help="0 = all layers of the workload")
    ap.add_argument("--batch", type=int, default=0)
    ap.add_argument("--context", type=int, default=0)
    ap.add_argument("--impl", default="mkv", choices=["mkv", "reference"])
    ap.add_argument("--no-graph", action="store_true", help="launch eagerly instead of CUDA graphs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-units", type=int, default=8, help="units of one layer the oracle is timed on")
    ap.add_argument("--sweep", action="store_true",
                    help="BASELINE config 5: keep ratio x token budget on the config-2 shape, 6 layers per point")
    ap.add_argument("--sweep-layers", type=int, default=6, help="layers cycled per sweep point (6 x >= 20 MB > L2)")
    ap.add_argument("--verbose", action="store_true")
    return ap.parse_args()


def workload_config(w, n_layers, Bt, N, budget):
    """`config` of the JSON line: the workload, identical for the mkv arm and the reference arm (the driver compares them)"""
    return {"workload": w.name, "baseline_config": w.config_id, "n_layers": n_layers, "batch_per_gpu": Bt,
            "n_q_heads": w.n_q_heads, "n_kv_heads": w.n_kv_heads, "head_dim": 128, "context": N,
            "segment_len": w.segment_len, "token_block": 8, "keep_ratio": w.keep_ratio, "r_keep": w.r_keep,
            "dense_segments": f"{w.dense_num}/{w.dense_den}", "token_budget": budget,
            "l2": "inputs larger than L2: consecutive layers read different packed arenas"}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """SM clock + throttle reasons sampled through NVML DURING the timed region (same fields as the
    nvidia-smi line of B200_PROFILING.md, polled every ~2 ms from a thread so that a region of a few
    tens of milliseconds still gets samples)."""

    def __init__(self, torch_index):
        self.samples, self.reasons, self.max_mhz, self.h, self._stop, self.th = [], set(), None, None, False, None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            p = torch.cuda.get_device_properties(torch_index)
            bus = "%08x:%02x:%02x.0" % (p.pci_domain_id, p.pci_bus_id, p.pci_device_id)
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByPciBusId(bus.encode())
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.h = None

    def _run(self):
        nv = self.nv
        bits = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                "hw_power_brake_slowdown": 0x80}
        while not self._stop:
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for n, b in bits.items():
                    if r & b:
                        self.reasons.add(n)
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.h is None:
            return
        import threading
        self._stop = False
        self.th = threading.Thread(target=self._run, daemon=True)
        self.th.start()

    def stop(self):
        if self.th is not None:
            self._stop = True
            self.th.join()
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


# ------------------------------------------------------------------------------ timing helpers

def timed_loop(torch, fn, steps, warmup, dist_barrier, graph=True, stats=None):
    """W untimed + K timed calls of fn() on torch's current stream; returns ms per call (mean over the K calls).
    fn's launches are captured in one CUDA graph (launch-bound inner loop) unless graph=False.  If `stats` is a dict
    it receives the median and the minimum of the K per-call times (events between the calls)."""
    stream = torch.cuda.current_stream()
    runner = fn
    if graph:
        fn()  # warm (lazy module load) before capture
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=torch.cuda.Stream()):
            fn()
        runner = g.replay
    for _ in range(warmup):
        runner()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    dist_barrier()
    torch.cuda.synchronize()
    ev[0].record(stream)
    for i in range(steps):
        runner()
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    dist_barrier()
    if stats is not None:
        per = sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(steps))
        stats["median_ms"], stats["min_ms"] = per[len(per) // 2], per[0]
    return ev[0].elapsed_time(ev[steps]) / steps


def max_over_ranks(torch, dist, x, world):
    if world == 1:
        return x
    t = torch.tensor([x], dtype=torch.float64, device="cuda")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


# ------------------------------------------------------------------------------ the mkv arm

def run_mkv(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    barrier = (lambda: dist.barrier()) if world > 1 else (lambda: None)

    import __graft_entry__
    if rank == 0:
        __graft_entry__.build()
    barrier()
    from paper_2607_00760_b200 import binding as mkv
    from paper_2607_00760_b200 import shard, synth, workload

    w = synth.WORKLOADS[args.workload]
    n_layers = args.layers or w.n_layers
    Bt = args.batch or w.batch
    N = args.context or w.context
    # weak scaling: every rank holds its own batch of Bt requests (units are independent: no collective)
    w = shard.rank_workload(w, rank)
    t0 = time.time()
    built = workload.build(w, dev, n_layers=n_layers, batch=Bt, context=N, verbose=args.verbose and rank == 0)
    build_s = time.time() - t0
    cache = built.cache
    Hkv, Hq, G = w.n_kv_heads, w.n_q_heads, w.group
    budget = w.token_budget
    k_max = min(budget // 8 + 1, (N + 7) // 8)
    scale = 1.0 / math.sqrt(128)
    sel = [torch.full((Bt, Hkv, k_max), -1, dtype=torch.int32, device=dev) for _ in range(n_layers)]
    cnt = [torch.zeros((Bt, Hkv), dtype=torch.int32, device=dev) for _ in range(n_layers)]
    out = torch.zeros((n_layers, Bt, Hq, 128), dtype=torch.float32, device=dev)

    def step_select():
        for l in range(n_layers):
            cache.select(l, built.q[l], budget, sel[l], cnt[l])

    def step_attention():
        for l in range(n_layers):
            cache.packed_attention(l, built.q[l], sel[l], cnt[l], scale, out[l])

    def step_decode():
        for l in range(n_layers):
            cache.select(l, built.q[l], budget, sel[l], cnt[l])
            cache.packed_attention(l, built.q[l], sel[l], cnt[l], scale, out[l])

    step_decode()
    torch.cuda.synchronize()
    cache.status()
    launches = cache.last_launch_count()
    n_sel_total = [int(c.sum().item()) for c in cnt]
    attn_split = [workload.attention_bytes(built, l, sel[l], cnt[l], split=True) for l in range(n_layers)]
    attn_bytes = [x[0] for x in attn_split]
    v_parts = sum(x[2] for x in attn_split) / n_layers
    sel_bytes = [workload.select_bytes(built, l, n_sel_total[l]) for l in range(n_layers)]
    comp_bytes = workload.compress_bytes(built, 0)

    graph = not args.no_graph
    clocks = ClockSampler(local)
    clocks.start()
    st_step, st_attn, st_sel = {}, {}, {}
    ms_step = timed_loop(torch, step_decode, args.steps, args.warmup, barrier, graph, st_step)
    cache.attention_stats(reset=True)
    ms_attn = timed_loop(torch, step_attention, args.steps, args.warmup, barrier, graph, st_attn)
    stats = cache.attention_stats(reset=True)
    ms_sel = timed_loop(torch, step_select, args.steps, args.warmup, barrier, graph, st_sel)
    clk = clocks.stop()

    # the same selection attended with q = 0 (flat softmax: phase 2 may skip nothing, every V part is fetched)
    q_zero = [torch.zeros_like(x) for x in built.q]

    def step_attention_flat():
        for l in range(n_layers):
            cache.packed_attention(l, q_zero[l], sel[l], cnt[l], scale, out[l])

    ms_flat = timed_loop(torch, step_attention_flat, args.steps, args.warmup, barrier, graph)
    stats_flat = cache.attention_stats(reset=True)

    # calibration: (ii) the attention kernel's own staging of the same selected payloads (K parts, then V
    # parts, nothing skipped) with all arithmetic removed; (i) a plain streaming read of the same number of bytes
    def step_gather():
        for l in range(n_layers):
            cache.calibrate_gather(l, sel[l], cnt[l])

    ms_gather = timed_loop(torch, step_gather, args.steps, args.warmup, barrier, graph)
    a_bytes_int = int(sum(attn_bytes) / n_layers)

    def step_stream():
        for l in range(n_layers):
            cache.calibrate_stream(l, a_bytes_int)

    ms_stream = timed_loop(torch, step_stream, args.steps, args.warmup, barrier, graph)

    # calibration (iii): the QK expansion alone on groups of the real selection, resident in shared memory
    def walk_us(reps):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        cache.calibrate_walk(0, built.q[0], sel[0], cnt[0], reps)
        torch.cuda.synchronize()
        ev0.record()
        cache.calibrate_walk(0, built.q[0], sel[0], cnt[0], reps)
        ev1.record()
        torch.cuda.synchronize()
        return ev0.elapsed_time(ev1) * 1e3

    WALK_R1, WALK_R2, WALK_WARPS = 200, 1200, 16
    us_walk_group = (walk_us(WALK_R2) - walk_us(WALK_R1)) / (WALK_R2 - WALK_R1) / WALK_WARPS  # one SM, one group of 16 tokens
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    groups_attn = sum(n_sel_total) / n_layers / 2.0                 # K groups of one attention launch
    c_attn = max([c for c in (16, 8, 4, 2, 1) if Bt * Hkv * c <= sm_count] or [1])  # CTAs per unit (attention.cu: pick_cluster)
    sms_attn = min(sm_count, Bt * Hkv * c_attn)
    groups_score = Bt * Hkv * math.ceil(N / 8) / 16.0                # groups of 16 block keys of one score launch

    # end to end through the public host call: pinned q in, out back, every layer, every step
    q_host = [q.cpu().pin_memory() for q in built.q]
    out_host = [torch.zeros((Bt, Hq, 128), dtype=torch.float32).pin_memory() for _ in range(n_layers)]

    def step_e2e():  # every mkv_decode_host call enqueues H2D(q) -> select -> attention -> D2H(out) on the stream
        for l in range(n_layers):
            cache.decode_host(l, q_host[l], budget, scale, out_host[l])
        if not graph:
            torch.cuda.current_stream().synchronize()

    # the host call is CUDA-graph capturable (pinned buffers, no allocation, no synchronisation): one graph per step
    ms_e2e = timed_loop(torch, step_e2e, max(3, args.steps // 2), 3, barrier, graph)
    cache.status()

    ms_step = max_over_ranks(torch, dist, ms_step, world)
    ms_attn = max_over_ranks(torch, dist, ms_attn, world)
    ms_sel = max_over_ranks(torch, dist, ms_sel, world)
    ms_e2e = max_over_ranks(torch, dist, ms_e2e, world)

    peak, peak_src = measured_peak()
    us_attn = ms_attn * 1e3 / n_layers
    us_sel = ms_sel * 1e3 / n_layers
    a_bytes = sum(attn_bytes) / n_layers
    s_bytes = sum(sel_bytes) / n_layers
    attn_gbs = a_bytes / (us_attn * 1e-6) / 1e9
    sel_gbs = s_bytes / (us_sel * 1e-6) / 1e9
    comp_ms = np.array(built.compress_ms[1:] or built.compress_ms).mean(axis=0)
    comp_gbs = (comp_bytes["read"] + comp_bytes["write"]) / (comp_ms[2] * 1e-3) / 1e9

    full_size = Bt == w.batch and N == w.context
    cap = NCU_CAPTURE.get(w.name, {}) if full_size else {}
    # bytes the kernel actually fetched per launch: everything but the V parts phase 2 skipped (the kernel counts the
    # blocks it walked and the bytes of their V copies; ratios are independent of how many launches fed the counters)
    v_frac = stats["v_blocks"] / max(1, stats["blocks"])
    sel_blocks = sum(n_sel_total) / n_layers
    bytes_fetched = int(a_bytes - v_parts + stats["v_bytes"] / max(1, stats["blocks"]) * sel_blocks)
    us_attn_in_step = (ms_step - ms_sel) * 1e3 / n_layers
    metric = METRIC if w.name == "llama8b-128k-b8" and full_size else f"PackedAttention us/layer ({w.name}, batch {Bt}, context {N})"
    line = {
        "metric": metric, "value": round(us_attn, 3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": round(ms_step, 4), "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16 storage, fp32 accumulate", "data": "synthetic",
        "config": workload_config(w, n_layers, Bt, N, budget),
        "launch": "cuda-graph of one decode step" if graph else "eager",
        # the headline above is on BASELINE's generator, whose softmax is so peaked that phase 2 skips most V parts
        # (v_blocks_fetched_fraction); the same launch with a flat softmax (q = 0: nothing can be skipped, as with any
        # logit spread below 27 nats) is the data-independent figure, printed right beside it
        "value_nothing_skipped_q0": round(ms_flat * 1e3 / n_layers, 3),
        "v_blocks_fetched_fraction": round(v_frac, 4),
        "decode_tokens_per_s_attention_only": round(world * Bt / (ms_step * 1e-3), 1),
        "select_us_per_layer": round(us_sel, 3),
        "attention_us_per_layer": {"mean": round(us_attn, 3), "median": round(st_attn["median_ms"] * 1e3 / n_layers, 3),
                                   "min": round(st_attn["min_ms"] * 1e3 / n_layers, 3),
                                   "inside_decode_step": round(us_attn_in_step, 3),
                                   "flat_softmax_q0": round(ms_flat * 1e3 / n_layers, 3)},
        "roofline": {"kernel": "mkv_packed_attention", "bound": "hbm", "achieved": round(attn_gbs, 1), "peak": peak,
                     "unit": "GB/s", "frac": round(attn_gbs / peak, 4),
                     "frac_flat": round(a_bytes / (ms_flat * 1e-3 / n_layers) / 1e9 / peak, 4),
                     "frac_on_bytes_fetched": round((bytes_fetched or 0) / (us_attn * 1e-6) / 1e9 / peak, 4),
                     "traffic": cap.get("attention"),
                     "traffic_from_capture": {"bytes": cap.get("attention"), "source": cap.get("source")},
                     "peak_source": peak_src,
                     "frac_of_nominal_8TBs": round(attn_gbs / NOMINAL_HBM_GBS, 4),
                     "algorithmic_bytes_per_launch": int(a_bytes),
                     "what": "frac = algorithmic bytes (every selected K and V payload, SURVEY 8(d)) / time / peak, on BASELINE's "
                             "generator.  The kernel fetches every K part but only the V parts of blocks with a probability >= "
                             "2^-40 of the unit's largest (bytes_fetched_per_launch, from the kernel's counters), and this "
                             "generator's softmax is peaked enough to skip most of them: frac is NOT the DRAM rate.  "
                             "frac_on_bytes_fetched is the rate on the bytes that did move; frac_flat is the same launch with "
                             "q = 0 (flat softmax, every V part fetched, algorithmic bytes = bytes fetched): the figure to "
                             "expect when the logits of the selected tokens spread over less than 27 nats",
                     "v_blocks_fetched_fraction": round(v_frac, 4),
                     "bytes_fetched_per_launch": bytes_fetched,
                     "flat_softmax_q0": {"us_per_layer": round(ms_flat * 1e3 / n_layers, 3),
                                         "v_blocks_fetched_fraction": round(stats_flat["v_blocks"] / max(1, stats_flat["blocks"]), 4),
                                         "frac": round(a_bytes / (ms_flat * 1e-3 / n_layers) / 1e9 / peak, 4)}},
        "roofline_select": {"kernel": "mkv_select", "bound": "hbm", "achieved": round(sel_gbs, 1), "peak": peak,
                            "unit": "GB/s", "frac": round(sel_gbs / peak, 4), "traffic": cap.get("score+topk"),
                            "traffic_from_capture": {"bytes": cap.get("score+topk"), "source": cap.get("source")},
                            "algorithmic_bytes_per_launch": int(s_bytes)},
        "compress": {"loss_ms_per_layer": round(float(comp_ms[0]), 3), "strategy_ms_per_layer": round(float(comp_ms[1]), 3),
                     "compress_ms_per_layer": round(float(comp_ms[2]), 3), "achieved": round(comp_gbs, 1), "unit": "GB/s",
                     "frac": round(comp_gbs / peak, 4), "bytes_read": comp_bytes["read"], "bytes_written": comp_bytes["write"],
                     "build_all_layers_s": round(build_s, 2)},
        "e2e": {"value": round(ms_e2e * 1e3 / n_layers, 3), "unit": UNIT,
                "what": "select + attention through mkv_decode_host: pinned host q in, host out back, both transfers inside the timed region (kernels of the chain read q_host and write out_host over PCIe)",
                "launch": "cuda-graph of one decode step of mkv_decode_host calls" if graph else "eager, synchronised per step",
                "h2d_bytes_per_step": n_layers * Bt * Hq * 128 * 2, "d2h_bytes_per_step": n_layers * Bt * Hq * 128 * 4,
                "ms_per_step": round(ms_e2e, 4)},
        "calibration": {"stream_read_us_per_layer": round(ms_stream * 1e3 / n_layers, 3),
                        "stream_read_gbs": round(a_bytes / (ms_stream * 1e-3 / n_layers) / 1e9, 1),
                        "gather_only_us_per_layer": round(ms_gather * 1e3 / n_layers, 3),
                        "gather_only_gbs": round(a_bytes / (ms_gather * 1e-3 / n_layers) / 1e9, 1),
                        "walk_only_ns_per_group_per_sm": round(us_walk_group * 1e3, 2),
                        "walk_only_attention_qk_us_per_layer": round(us_walk_group * groups_attn / sms_attn, 3),
                        "walk_only_score_us_per_layer": round(us_walk_group * groups_score / sm_count, 3),
                        "what_walk": "mkv_calibrate_walk: every warp (16 per SM) runs the QK expansion of one group (two selected "
                                     "token blocks, already in shared memory) over and over; ns per group per SM from the "
                                     "difference of two repeat counts.  x groups per launch / SMs in use = the time the "
                                     "shared-memory pipe alone needs for phase 1 of PackedAttention and for the score kernel",
                        "what": "stream_read: mkv_calibrate_stream, a plain 16-byte-load read of algorithmic_bytes_per_launch bytes of "
                                "the layer's arena in the attention kernel's launch shape (148 x 512).  gather_only: "
                                "mkv_calibrate_gather, the attention kernel's own staging of every selected K part then every V "
                                "part (bulk copies into the warps' rings, nothing skipped), no walk, no MMA, no output"},
        "gpu_launches": args.steps * n_layers * (launches["select"] + launches["attention"]),
        "kernels_per_layer": launches,
        "clocks": clk,
    }
    if rank == 0:
        line["update_buffer"] = measure_update_buffer(torch, mkv, synth, w, dev, Bt, cache, built, step_attention,
                                                      n_layers, graph, args)
    if rank == 0 and world == 1:
        line["element_groups_g2"] = measure_element_groups(torch, workload, w, dev, Bt, N, args, graph, us_attn, us_sel)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args, w, built, dev, n_units=args.cpu_units, repeats=1)
    built.free()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


def measure_update_buffer(torch, mkv, synth, w, dev, Bt, cache, built, step_attention, n_layers, graph, args):
    """KV update buffer: (i) flush = compress a full buffer of every unit of one layer through
    step 1 (the paper's only absolute kernel time: 40.6 us on an H800 for its 32-token buffer), measured for a
    32-token and a 64-token buffer (buffer = one segment); (ii) PackedAttention with 32 tokens buffered per unit."""
    Hkv, Hq = w.n_kv_heads, w.n_q_heads
    res = {"paper_h800_flush_us_32_tokens": 40.6, "units_per_layer": Bt * Hkv}
    for L in (32, 64):
        c = mkv.Cache(1, Bt, Hkv, Hq, 128, 4 * L, L, device=dev.index or 0)
        try:
            k = torch.randn((Bt, Hkv, L, 128), device=dev).to(torch.bfloat16)
            v = torch.randn((Bt, Hkv, L, 128), device=dev).to(torch.bfloat16)
            st = torch.tensor([w.r_keep, w.r_keep, 1, 8], dtype=torch.uint8, device=dev).repeat(Bt, Hkv, 1, 1)
            ts = []
            for it in range(8):
                c.reset()
                c.update_append(0, k, v)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                c.update_flush(0, st)
                e1.record()
                torch.cuda.synchronize()
                if it >= 3:
                    ts.append(e0.elapsed_time(e1) * 1e3)
            c.status()
            res[f"flush_us_{L}_tokens"] = round(sorted(ts)[len(ts) // 2], 2)
        finally:
            c.free()
    kn = torch.randn((Bt, Hkv, 32, 128), device=dev).to(torch.bfloat16)
    vn = torch.randn((Bt, Hkv, 32, 128), device=dev).to(torch.bfloat16)
    for l in range(n_layers):
        cache.update_append(l, kn, vn)
    ms = timed_loop(torch, step_attention, args.steps, args.warmup, lambda: None, graph)
    cache.status()
    res["attention_us_per_layer_with_32_buffered_tokens"] = round(ms * 1e3 / n_layers, 3)
    return res


def measure_element_groups(torch, workload, w, dev, Bt, N, args, graph, us_attn_g1, us_sel_g1):
    """The same workload compressed with element groups g = 2 (one of the paper's candidate group
    sizes), six layers cycled (touched set > L2): K values and block keys are stored pair-major and the QK walk loads one
    aligned 32-bit pair per kept group.  Printed BESIDE the g = 1 headline; the north-star config is g = 1."""
    NL = 6
    scale = 1.0 / math.sqrt(128)
    built = workload.build(w, dev, n_layers=NL, batch=Bt, context=N, g=2)
    try:
        cache, Hkv, Hq, budget = built.cache, w.n_kv_heads, w.n_q_heads, w.token_budget
        k_max = min(budget // 8 + 1, (N + 7) // 8)
        sel = [torch.full((Bt, Hkv, k_max), -1, dtype=torch.int32, device=dev) for _ in range(NL)]
        cnt = [torch.zeros((Bt, Hkv), dtype=torch.int32, device=dev) for _ in range(NL)]
        out = torch.zeros((NL, Bt, Hq, 128), dtype=torch.float32, device=dev)

        def step_select():
            for l in range(NL):
                cache.select(l, built.q[l], budget, sel[l], cnt[l])

        def step_attention():
            for l in range(NL):
                cache.packed_attention(l, built.q[l], sel[l], cnt[l], scale, out[l])

        step_select()
        torch.cuda.synchronize()
        ms_a = timed_loop(torch, step_attention, args.steps, args.warmup, lambda: None, graph)
        ms_s = timed_loop(torch, step_select, args.steps, args.warmup, lambda: None, graph)
        cache.status()
        comp = [sum(x[i] for x in built.compress_ms[1:]) / max(1, len(built.compress_ms) - 1) for i in range(3)]
        return {"g": 2, "n_layers": NL, "attention_us_per_layer": round(ms_a * 1e3 / NL, 3),
                "select_us_per_layer": round(ms_s * 1e3 / NL, 3),
                "attention_vs_g1": round(ms_a * 1e3 / NL / us_attn_g1, 3), "select_vs_g1": round(ms_s * 1e3 / NL / us_sel_g1, 3),
                "loss_ms_per_layer": round(comp[0], 3), "compress_ms_per_layer": round(comp[2], 3)}
    finally:
        built.free()


# ------------------------------------------------------------------------------ the oracle legs

def oracle_sample(w, units, N, verbose=False):
    """units: list of (K u16 [N][D], V u16 [N][D], q u16 [G][D]).  Runs the oracle as it stands:
    prep (loss -> strategy -> compress, one python thread per unit) then timed decode legs."""
    import numpy as np
    from concurrent.futures import ThreadPoolExecutor

    import oracle as orc

    r, L = w.r_keep, w.segment_len
    S = N // L

    def prep(u):
        K, V, _ = u
        if w.dense_num > 0:
            lk, lv = orc.segment_loss(K, V, L, r, r)
            st = orc.strategy_quantile(lk, lv, w.dense_num, w.dense_den, 128, r, r)
        else:
            st = orc.uniform_strategy(S, r, r)
        return orc.compress_unit(K, V, L, st)

    t0 = time.time()
    with ThreadPoolExecutor(max(1, min(len(units), os.cpu_count() or 1))) as ex:
        blobs = list(ex.map(prep, units))
    prep_s = time.time() - t0
    q = np.stack([u[2] for u in units])
    scale = 1.0 / math.sqrt(128)

    def one_step():
        t0 = time.time()
        sel, cnt, _, _ = orc.decode_units(blobs, q, w.token_budget, scale, 0, k_max=w.token_budget // 8 + 1)
        t_decode = time.time() - t0
        t0 = time.time()
        orc.attention_units(blobs, q, sel, cnt, scale)
        return t_decode, time.time() - t0

    return one_step, prep_s, orc.num_threads()


def sample_units(w, dev, n_units, Bt, N):
    """raw K/V/q of n_units units of layer 0, from the same seeded generator the GPU path consumes"""
    import numpy as np
    import torch
    from paper_2607_00760_b200 import synth
    G, Hkv = w.group, w.n_kv_heads
    units = []
    if torch.cuda.is_available():
        K, V, q = synth.make_layer_torch(w, 0, dev, batch=Bt, context=N)
        u16 = lambda t: t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
        for i in range(n_units):
            u = (i * (Bt * Hkv - 1)) // max(1, n_units - 1) if n_units > 1 else 0  # spread, first and last included
            b, h = divmod(u, Hkv)
            units.append((u16(K[b, h]), u16(V[b, h]), u16(q[b, h * G:(h + 1) * G])))
        del K, V
        src = "torch CUDA generator (the bytes the GPU path consumed)"
    else:
        nb = -(-n_units // Hkv)
        K, V, q = synth.make_inputs_np(nb, Hkv, w.n_q_heads, N, 128, w.segment_len, seed=1000 * w.config_id)
        for u in range(n_units):
            b, h = divmod(u, Hkv)
            units.append((K[b, h], V[b, h], q[b, h * G:(h + 1) * G]))
        src = "numpy generator (no GPU present)"
    return units, src


def cpu_baseline(args, w, built, dev, n_units, repeats):
    Bt = built.batch if built is not None else (args.batch or w.batch)
    N = built.context if built is not None else (args.context or w.context)
    n_units = min(n_units, Bt * w.n_kv_heads)
    units, src = sample_units(w, dev, n_units, Bt, N)
    one_step, prep_s, threads = oracle_sample(w, units, N)
    t = [one_step() for _ in range(repeats)]
    t_dec, t_att = min(x[0] for x in t), min(x[1] for x in t)
    scale_up = Bt * w.n_kv_heads / n_units
    return {"value": round(t_att * scale_up * 1e6, 1), "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"{n_units} of {Bt * w.n_kv_heads} units of layer 0 ({src}); oracle attention (O8) on the oracle's own "
                      f"selection, OpenMP over units, time scaled by {scale_up:g} to one layer; prep (loss, strategy, "
                      f"compress) {prep_s:.1f} s untimed",
            "select_plus_attention_us_per_layer": round(t_dec * scale_up * 1e6, 1)}


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    if rank != 0:
        return
    import torch
    from oracle import build as orc_build
    orc_build.build()
    from paper_2607_00760_b200 import synth
    w = synth.WORKLOADS[args.workload]
    n_layers = args.layers or w.n_layers
    Bt, N = args.batch or w.batch, args.context or w.context
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", 0))) if torch.cuda.is_available() else None
    n_units = min(args.cpu_units, Bt * w.n_kv_heads)
    units, src = sample_units(w, dev, n_units, Bt, N)
    one_step, prep_s, threads = oracle_sample(w, units, N)
    for _ in range(args.warmup):
        one_step()
    steps = max(1, args.steps)
    t0 = time.time()
    ts = [one_step() for _ in range(steps)]
    wall = time.time() - t0
    scale_up = Bt * w.n_kv_heads / n_units
    t_att = sum(x[1] for x in ts) / steps
    t_dec = sum(x[0] for x in ts) / steps
    value = t_att * scale_up * 1e6
    sample = (f"{n_units} of {Bt * w.n_kv_heads} units of one layer ({src}); each step = oracle select + attention then "
              f"attention alone on the sample; us/layer = attention time x {scale_up:g}; prep {prep_s:.1f} s untimed")
    line = {"impl": "reference", "metric": METRIC, "value": round(value, 1), "unit": UNIT, "n_gpus": world,
            "steps": steps, "warmup": args.warmup, "ms_per_step": round(wall / steps * 1e3, 3),
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, n_layers, Bt, N, w.token_budget),
            "launch": "CPU oracle (OpenMP over units), bounded sample",
            "cpu_baseline": {"value": round(value, 1), "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                             "select_plus_attention_us_per_layer": round(t_dec * scale_up * 1e6, 1)},
            "e2e": {"value": round(t_dec * scale_up * 1e6, 1), "unit": UNIT, "what": "oracle select + attention on the sample, scaled to one layer",
                    "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_sweep(args):
    """BASELINE config 5 on one GPU: keep ratio in {1.0, 0.7, 0.5, 0.3} x token budget in {1024, 4096, 16384} (the 10 %
    dense mix held fixed) plus the dense-full point (r = 128, budget = context).  Six layers are cycled per point so
    that the set touched between two visits of a layer exceeds the 126 MB L2 at every point.  Prints one JSON line."""
    import dataclasses
    import torch
    import __graft_entry__
    __graft_entry__.build()
    from paper_2607_00760_b200 import synth, workload
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    base = synth.WORKLOADS[args.workload]
    Bt, N = args.batch or base.batch, args.context or base.context
    peak, peak_src = measured_peak()
    scale = 1.0 / math.sqrt(128)
    NL = max(2, args.sweep_layers)  # layers cycled per point: >= 6 x the touched set exceeds the 126 MB L2 at every point
    points = []
    for keep in (1.0, 0.7, 0.5, 0.3):
        w = dataclasses.replace(base, keep_ratio=keep)
        built = workload.build(w, dev, n_layers=NL, batch=Bt, context=N)
        cache, Hkv, Hq = built.cache, w.n_kv_heads, w.n_q_heads
        budgets = [1024, 4096, 16384] + ([N] if keep == 1.0 else [])
        for budget in budgets:
            k_max = min(budget // 8 + 1, (N + 7) // 8)
            sel = [torch.full((Bt, Hkv, k_max), -1, dtype=torch.int32, device=dev) for _ in range(NL)]
            cnt = [torch.zeros((Bt, Hkv), dtype=torch.int32, device=dev) for _ in range(NL)]
            out = torch.zeros((NL, Bt, Hq, 128), dtype=torch.float32, device=dev)
            for l in range(NL):
                cache.select(l, built.q[l], budget, sel[l], cnt[l])
            torch.cuda.synchronize()

            def step_attention():
                for l in range(NL):
                    cache.packed_attention(l, built.q[l], sel[l], cnt[l], scale, out[l])

            def step_select():
                for l in range(NL):
                    cache.select(l, built.q[l], budget, sel[l], cnt[l])

            cache.attention_stats(reset=True)
            ms_a = timed_loop(torch, step_attention, args.steps, max(3, args.warmup), lambda: None, True)
            stats = cache.attention_stats(reset=True)
            ms_s = timed_loop(torch, step_select, args.steps, max(3, args.warmup), lambda: None, True)
            cache.status()
            split = [workload.attention_bytes(built, l, sel[l], cnt[l], split=True) for l in range(NL)]
            ab = sum(x[0] for x in split) / NL
            v_parts = sum(x[2] for x in split) / NL
            n_blocks = sum(int(c.sum().item()) for c in cnt) / NL
            # bytes the kernel fetched: everything but the V parts phase 2 skipped (kernel counters).  `frac`
            # is on those bytes (a DRAM rate, never above 1); `frac_algorithmic` counts every selected payload
            # whether fetched or not
            fetched = ab - v_parts + stats["v_bytes"] / max(1, stats["blocks"]) * n_blocks
            us = ms_a * 1e3 / NL
            gbs = ab / (us * 1e-6) / 1e9
            points.append({"keep_ratio": keep, "r_keep": w.r_keep, "token_budget": budget,
                           "attention_us_per_layer": round(us, 2), "select_us_per_layer": round(ms_s * 1e3 / NL, 2),
                           "bytes_fetched_per_launch": int(fetched),
                           "achieved_gbs": round(fetched / (us * 1e-6) / 1e9, 1),
                           "frac": round(fetched / (us * 1e-6) / 1e9 / peak, 4),
                           "frac_of_nominal_8TBs": round(fetched / (us * 1e-6) / 1e9 / NOMINAL_HBM_GBS, 4),
                           "v_blocks_fetched_fraction": round(stats["v_blocks"] / max(1, stats["blocks"]), 4),
                           "algorithmic_bytes_per_launch": int(ab), "frac_algorithmic": round(gbs / peak, 4)})
            del sel, cnt, out
        built.free()
        del built
        torch.cuda.empty_cache()
    print(json.dumps({"metric": "PackedAttention us/layer, compression sweep (BASELINE config 5)", "unit": UNIT,
                      "n_gpus": 1, "steps": args.steps, "warmup": max(3, args.warmup), "data": "synthetic",
                      "config": {"workload": base.name + "-sweep", "batch_per_gpu": Bt, "context": N, "n_layers": NL,
                                 "dense_segments": f"{base.dense_num}/{base.dense_den} (all dense at keep 1.0)"},
                      "peak": peak, "peak_source": peak_src, "sweep": points}), flush=True)


if __name__ == "__main__":
    a = parse()
    if a.sweep:
        run_sweep(a)
    elif a.impl == "reference":
        run_reference(a)
    else:
        run_mkv(a)
