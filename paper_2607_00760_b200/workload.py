"""Build a packed cache for one of the BASELINE.json workloads through the C ABI, layer by layer
(raw K/V of one layer at a time: config 2 holds 4.3 GB raw per layer, 62 GB packed in total),
and count the algorithmic bytes each kernel must move.

Used by bench.py and the full-size parity test so both run the same launch configuration.
Holds none of the method's arithmetic: every step runs in libmkv's kernels.
"""
import math
from dataclasses import dataclass, field

from . import binding as mkv
from . import synth

D = 128


def vec_bytes(r: int) -> int:
    return 2 * r + (16 if r < D else 0)


def unit_payload_bytes(w: synth.Workload, context=None) -> int:
    """exact packed bytes (token payloads + block keys) of one unit under the quantile policy"""
    N = context or w.context
    S = N // w.segment_len
    n_dense = -(-S * w.dense_num // w.dense_den)
    r = w.r_keep
    blk = w.segment_len // 8
    per_seg = lambda rr: blk * 8 * 2 * vec_bytes(rr) + (blk * vec_bytes(rr) + 15) // 16 * 16
    return n_dense * per_seg(D) + (S - n_dense) * per_seg(r)


@dataclass
class BuiltCache:
    w: synth.Workload
    cache: "mkv.Cache"
    n_layers: int
    batch: int
    context: int
    q: list = field(default_factory=list)        # per layer: bf16 [Bt][Hq][D] on the device
    strat: list = field(default_factory=list)    # per layer: uint8 [Bt][Hkv][S][4] on the device
    compress_ms: list = field(default_factory=list)  # per layer: (loss_ms, strategy_ms, compress_ms)
    raw_units: dict = field(default_factory=dict)    # (layer, b, h) -> (K u16 [N][D], V u16 [N][D]) on the host
    loss: dict = field(default_factory=dict)         # layer -> (loss_k, loss_v) device tensors (kept if asked)

    def free(self):
        self.cache.free()


def build(w: synth.Workload, dev, n_layers=None, batch=None, context=None, keep_units=(), keep_loss=False,
          verbose=False, g=1) -> BuiltCache:
    """Generate (seeded, on the device), choose strategies (quantile rule) and compress every layer.

    keep_units: iterable of (layer, b, h) whose raw K/V bytes are copied to the host for the oracle.
    g: element-group size of the sparse strategy (r_keep must be a multiple of it).
    """
    import numpy as np
    import torch

    n_layers = n_layers or w.n_layers
    Bt = batch or w.batch
    N = context or w.context
    L, Hkv, Hq = w.segment_len, w.n_kv_heads, w.n_q_heads
    S = N // L
    r = w.r_keep
    per_layer = Bt * Hkv * unit_payload_bytes(w, N) + (1 << 20)
    cache = mkv.Cache(n_layers, Bt, Hkv, Hq, D, N, L, device=dev.index or 0, arena_bytes=per_layer * n_layers)
    built = BuiltCache(w, cache, n_layers, Bt, N)
    keep_units = set(keep_units)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    for layer in range(n_layers):
        K, V, q = synth.make_layer_torch(w, layer, dev, batch=Bt, context=N)
        loss_k = torch.empty((Bt, Hkv, S), dtype=torch.float64, device=dev)
        loss_v = torch.empty_like(loss_k)
        strat = torch.empty((Bt, Hkv, S, 4), dtype=torch.uint8, device=dev)
        ev[0].record()
        if w.dense_num > 0:
            cache.segment_loss(K, V, (r, r, g, 8), loss_k, loss_v)
        ev[1].record()
        if w.dense_num > 0:
            cache.strategy_quantile(loss_k, loss_v, S, w.dense_num, w.dense_den, (r, r, g, 8), strat)
        else:
            strat[:] = torch.tensor([r, r, g, 8], dtype=torch.uint8, device=dev)
        ev[2].record()
        cache.compress_segment(layer, K, V, strat)
        ev[3].record()
        torch.cuda.synchronize()
        built.compress_ms.append(tuple(ev[i].elapsed_time(ev[i + 1]) for i in range(3)))
        built.q.append(q)
        built.strat.append(strat)
        if keep_loss:
            built.loss[layer] = (loss_k, loss_v)
        for (l, b, h) in keep_units:
            if l == layer:
                built.raw_units[(l, b, h)] = (K[b, h].view(torch.int16).cpu().numpy().view(np.uint16),
                                              V[b, h].view(torch.int16).cpu().numpy().view(np.uint16))
        del K, V
        if verbose:
            print(f"  layer {layer}: loss {built.compress_ms[-1][0]:.2f} ms, strategy {built.compress_ms[-1][1]:.2f} ms, "
                  f"compress {built.compress_ms[-1][2]:.2f} ms", flush=True)
    cache.status()
    return built


# ---- algorithmic bytes ----------------------

def compress_bytes(built: BuiltCache, layer: int) -> dict:
    by = built.cache.bytes(layer)
    w = built.w
    raw = 2 * built.batch * w.n_kv_heads * built.context * D * 2
    return dict(read=raw, write=by["packed"] + by["block_keys"] + by["tables"])


def select_bytes(built: BuiltCache, layer: int, n_selected: int) -> int:
    """per block key vec_bytes(r_k); per segment 8 B strategy + 4 B offset; q; 4 B per selected block out"""
    import torch
    w = built.w
    st = built.strat[layer]
    rk = st[..., 0].to(torch.int64)
    vb = 2 * rk + torch.where(rk < D, 16, 0)
    blk = w.segment_len // 8
    keys = int(((vb * blk + 15) // 16 * 16).sum().item())
    n_seg = st.shape[0] * st.shape[1] * st.shape[2]
    q_bytes = built.batch * w.n_q_heads * D * 2
    return keys + 12 * n_seg + q_bytes + 4 * n_selected


def attention_bytes(built: BuiltCache, layer: int, sel, cnt, split=False):
    """per selected block its token-block payload; + 4 B per selected block (sel) + 16 B per touched
    segment (strategy record + offsets) + per unit q (G*D*2) and out (G*D*4).
    split=True: (total, bytes of the K parts alone, bytes of the V parts alone)."""
    import torch
    w = built.w
    st = built.strat[layer].view(-1, built.strat[layer].shape[2], 4)  # [units][S][4]
    U, k_max = sel.shape[0] * sel.shape[1], sel.shape[2]
    sel2 = sel.view(U, k_max).to(torch.int64)
    valid = torch.arange(k_max, device=sel.device).view(1, -1) < cnt.view(U, 1)
    seg = torch.where(valid, sel2 // w.segment_len, 0)
    rk = torch.gather(st[..., 0].to(torch.int64), 1, seg)
    rv = torch.gather(st[..., 1].to(torch.int64), 1, seg)
    vb = lambda r: 2 * r + torch.where(r < D, 16, 0)
    payload = ((8 * (vb(rk) + vb(rv)) + 15) // 16 * 16) * valid
    key = torch.where(valid, seg + torch.arange(U, device=sel.device).view(-1, 1) * st.shape[1], -1)
    touched = int(torch.unique(key).numel()) - (1 if (~valid).any() else 0)
    G = w.group
    total = int(payload.sum().item()) + 4 * int(valid.sum().item()) + 16 * touched + U * G * D * 6
    if not split:
        return total
    return total, int((8 * vb(rk) * valid).sum().item()), int((8 * vb(rv) * valid).sum().item())
