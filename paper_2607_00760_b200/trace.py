"""Where the time of one PackedAttention launch goes: %globaltimer stamps at the kernel's phase boundaries.

    python -m paper_2607_00760_b200.trace [--workload llama8b-128k-b8] [--layers 4] [--flat] > trace.md

Builds libmkv_trace.so (the tracked sources with -DMKV_TRACE: lane 0 of every warp stores the timer at twelve points of
mkv_packed_attention_kernel; libmkv.so itself has no such code), builds the workload's cache exactly as bench.py does,
runs select + attention over the layers a few times so that the last launch is a steady-state one (eager launches with
programmatic dependent launch, previous layer's arena long evicted), reads the stamps of that last launch and prints a
markdown table: per stamp the earliest / median / latest warp, in microseconds after the launch's first stamp.
--flat: attend with q = 0 (nothing skipped in phase 2).  Measurement aid only; no arithmetic of the method lives here.
"""
import argparse
import ctypes as C
import math
import os
import sys

STAMPS = ["CTA scheduled, mbarriers initialised", "griddepcontrol.wait returned", "counts known (sel_count, update buffer)",
          "first <= 24 blocks described", "first K part landed", "phase 1 done (QK, logits, maxima)",
          "first cluster barrier passed (maxima exchanged)", "phase 2 done (sums, lists, V parts fetched and walked)",
          "warps' partials stored, CTA barrier passed", "CTA partial summed (rank 1: pushed to rank 0)",
          "second cluster barrier passed", "output stored / CTA leaves", "(between 8 and 9) the CTA's partial O summed"]
ORDER = [0, 1, 2, 3, 4, 5, 6, 7, 8, 12, 9, 10, 11]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="llama8b-128k-b8")
    ap.add_argument("--layers", type=int, default=4)
    ap.add_argument("--flat", action="store_true")
    args = ap.parse_args()

    from . import build as mkv_build
    lib_path = mkv_build.build(trace=True)
    os.environ["MKV_LIBRARY"] = lib_path
    import numpy as np
    import torch
    from . import binding as mkv, synth, workload
    assert mkv.LIB_PATH == lib_path
    lib = C.CDLL(lib_path)
    lib.mkv_trace_read.argtypes = [C.c_void_p, C.c_uint64, C.c_int]
    lib.mkv_trace_read.restype = C.c_int

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    w = synth.WORKLOADS[args.workload]
    NL = args.layers
    built = workload.build(w, dev, n_layers=NL)
    cache, Bt, Hkv, Hq, N, budget = built.cache, w.batch, w.n_kv_heads, w.n_q_heads, w.context, w.token_budget
    k_max = min(budget // 8 + 1, (N + 7) // 8)
    scale = 1.0 / math.sqrt(128)
    sel = [torch.full((Bt, Hkv, k_max), -1, dtype=torch.int32, device=dev) for _ in range(NL)]
    cnt = [torch.zeros((Bt, Hkv), dtype=torch.int32, device=dev) for _ in range(NL)]
    out = torch.zeros((Bt, Hq, 128), dtype=torch.float32, device=dev)
    q = [torch.zeros_like(x) for x in built.q] if args.flat else built.q
    for l in range(NL):
        cache.select(l, built.q[l], budget, sel[l], cnt[l])
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for rep in range(6):
        if rep == 5:
            ev0.record()
        for l in range(NL):
            cache.packed_attention(l, q[l], sel[l], cnt[l], scale, out)
    ev1.record()
    torch.cuda.synchronize()
    cache.status()
    us_launch = ev0.elapsed_time(ev1) * 1e3 / NL
    buf = np.zeros((160, 16, 16), np.uint64)
    rc = lib.mkv_trace_read(buf.ctypes.data, buf.nbytes, 0)
    assert rc == 0, rc
    n_units = Bt * Hkv
    ctas = int((buf[:, 0, 0] != 0).sum())
    t = buf[:ctas].astype(np.int64)
    t0 = t[:, :, 1].min()  # the launch proper starts when griddepcontrol.wait returns (CTAs are scheduled during the previous launch's tail)
    rel = (t - t0) / 1e3
    c = ctas // n_units
    print(f"# PackedAttention, one launch traced ({w.name}, {'q = 0: flat softmax' if args.flat else 'generator q'})\n")
    print(f"Command: `python -m paper_2607_00760_b200.trace --workload {args.workload} --layers {NL}{' --flat' if args.flat else ''}`"
          f" (libmkv_trace.so = the tracked sources with -DMKV_TRACE).  Last of {6 * NL} eager launches over {NL} layers; "
          f"{ctas} CTAs = {n_units} units x clusters of {c}, 16 warps each; mean time per launch of the last round (CUDA "
          f"events, stamps included): {us_launch:.1f} us.  Microseconds after the earliest `griddepcontrol.wait returned` (CTAs are scheduled earlier, during the previous launch's tail); a warp that skips a "
          f"step keeps the stamp of an earlier launch and is left out of that row.\n")
    print("| # | stamp | earliest warp | median | latest warp | median step |")
    print("|---|---|---|---|---|---|")
    prev = None
    for i in ORDER:
        name = STAMPS[i]
        v = rel[:, :, i].ravel()
        v = v[(v > -1e3) & (v < 1e4)]
        if v.size == 0:
            continue
        med = float(np.median(v))
        step = "" if prev is None else f"{med - prev:+.2f}"
        print(f"| {i} | {name} | {v.min():.2f} | {med:.2f} | {v.max():.2f} | {step} |")
        prev = med
    # per-CTA view of the two ranks of a cluster (phase ends), for the imbalance between the ranks
    if c >= 2:
        print("\nBy cluster rank (median over CTAs of the rank; latest warp of the CTA):\n")
        print("| rank | 5 phase 1 done | 7 phase 2 done | 8 | 12 | 9 | 10 | 11 leaves |")
        print("|---|---|---|---|---|---|---|---|")
        for r in range(min(c, 4)):
            rr = rel[r::c]
            f = lambda i: float(np.median(np.where((rr[:, :, i] > -1e3) & (rr[:, :, i] < 1e4), rr[:, :, i], -1e3).max(axis=1)))
            print(f"| {r} | {f(5):.2f} | {f(7):.2f} | {f(8):.2f} | {f(12):.2f} | {f(9):.2f} | {f(10):.2f} | {f(11):.2f} |")
    built.free()


if __name__ == "__main__":
    sys.exit(main())
