"""CPU oracle for the MosaicKV decode hot path — TEST INFRASTRUCTURE ONLY.

Plain C (oracle/mkv_oracle.c, fp64) behind a ctypes/numpy wrapper.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It imports nothing from paper_2607_00760_b200 and shares no code with the CUDA path.

All arrays are numpy; bf16 tensors are uint16 bit patterns.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_LIB = None


def lib():
    global _LIB
    if _LIB is None:
        path = _build.build()
        _LIB = C.CDLL(path)
        _declare(_LIB)
    return _LIB


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def _declare(L):
    u8p, u16p, i32p, f64p = (C.POINTER(C.c_uint8), C.POINTER(C.c_uint16), C.POINTER(C.c_int32),
                             C.POINTER(C.c_double))
    L.orc_topr.argtypes = [u16p, C.c_int, C.c_int, C.c_int, u8p]
    L.orc_topr.restype = None
    L.orc_block_key.argtypes = [u16p, C.c_int, C.c_int, u16p]
    L.orc_block_key.restype = None
    L.orc_segment_loss.argtypes = [u16p, u16p] + [C.c_int] * 6 + [f64p, f64p]
    L.orc_strategy_quantile.argtypes = [f64p, f64p] + [C.c_int] * 8 + [u8p]
    L.orc_strategy_threshold.argtypes = [f64p, f64p, C.c_int, C.c_int, u8p, C.c_double, C.c_int, u8p]
    L.orc_blob_size.argtypes = [C.c_int, C.c_int, C.c_int, u8p]
    L.orc_blob_size.restype = C.c_uint64
    L.orc_compress_unit.argtypes = [u16p, u16p, C.c_int, C.c_int, C.c_int, u8p, u8p, C.c_uint64]
    L.orc_unpack_unit.argtypes = [u8p, u16p, u8p, u16p, u8p, u16p, u8p]
    L.orc_blob_blocks.argtypes = [u8p, i32p, i32p]
    L.orc_scores.argtypes = [u8p, u16p, C.c_int, C.c_int, f64p]
    L.orc_topk.argtypes = [f64p, i32p, i32p, C.c_int, C.c_int, i32p]
    L.orc_attention.argtypes = [u8p, u16p, C.c_int, i32p, C.c_int, C.c_double, f64p, f64p]
    L.orc_attention_weights.argtypes = [u8p, u16p, C.c_int, i32p, C.c_int, C.c_double, f64p, f64p,
                                        f64p, i32p, C.c_int]
    L.orc_merge.argtypes = [C.c_int, C.c_int, f64p, f64p, f64p, f64p, f64p, f64p]
    L.orc_merge.restype = None
    L.orc_compress_units.argtypes = [u16p, u16p, C.c_int, C.c_int, C.c_int, C.c_int, u8p,
                                     C.POINTER(u8p), C.POINTER(C.c_uint64)]
    L.orc_decode_units.argtypes = [C.POINTER(u8p), C.c_int, u16p, C.c_int, C.c_int, C.c_int,
                                   C.c_double, i32p, i32p, C.c_int, f64p, f64p]
    L.orc_attention_units.argtypes = [C.POINTER(u8p), C.c_int, u16p, C.c_int, i32p, i32p, C.c_int,
                                      C.c_double, f64p, f64p]
    L.orc_num_threads.restype = C.c_int
    L.orc_rotate_query.argtypes = [u16p, C.c_int, C.c_int, C.POINTER(C.c_float), u16p]
    L.orc_rotate_query.restype = None
    L.orc_rotate_output.argtypes = [f64p, C.c_int, C.c_int, C.POINTER(C.c_float)]
    L.orc_rotate_output.restype = None


def _u16(a):
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, a.dtype
    return a


def num_threads() -> int:
    return int(lib().orc_num_threads())


def topr(x, g: int, r: int):
    """O1: 0/1 keep flag per element group of one bf16 vector."""
    x = _u16(x)
    D = x.shape[-1]
    keep = np.zeros(D // g, np.uint8)
    lib().orc_topr(_p(x, C.c_uint16), D, g, r, _p(keep, C.c_uint8))
    return keep


def block_key(k):
    """O2: bf16 mean of the nb uncompressed keys k[nb][D]."""
    k = _u16(k)
    nb, D = k.shape
    out = np.zeros(D, np.uint16)
    lib().orc_block_key(_p(k, C.c_uint16), nb, D, _p(out, C.c_uint16))
    return out


def segment_loss(k, v, L: int, r_k: int, r_v: int, g: int = 1):
    """O3: per-segment relative squared loss of one candidate, one unit."""
    k, v = _u16(k), _u16(v)
    N, D = k.shape
    S = (N + L - 1) // L
    lk, lv = np.zeros(S), np.zeros(S)
    rc = lib().orc_segment_loss(_p(k, C.c_uint16), _p(v, C.c_uint16), N, D, L, r_k, r_v, g,
                                _p(lk, C.c_double), _p(lv, C.c_double))
    if rc < 0:
        raise ValueError("orc_segment_loss: bad strategy")
    return lk, lv


def strategy_quantile(lk, lv, num: int, den: int, D: int, r_k: int, r_v: int, g: int = 1, B: int = 8):
    """O4a: the ceil(S*num/den) highest-importance segments stay dense. Returns strat4[S][4]."""
    lk = np.ascontiguousarray(lk, np.float64)
    lv = np.ascontiguousarray(lv, np.float64)
    S = lk.shape[0]
    out = np.zeros((S, 4), np.uint8)
    rc = lib().orc_strategy_quantile(_p(lk, C.c_double), _p(lv, C.c_double), S, num, den, D, r_k,
                                     r_v, g, B, _p(out, C.c_uint8))
    if rc < 0:
        raise ValueError("orc_strategy_quantile")
    return out


def strategy_threshold(lk, lv, cands, tau: float, D: int):
    """O4b: first candidate with I <= tau, else dense. lk, lv: [ncand][S]."""
    lk = np.ascontiguousarray(lk, np.float64)
    lv = np.ascontiguousarray(lv, np.float64)
    cands = np.ascontiguousarray(cands, np.uint8)
    ncand, S = lk.shape
    out = np.zeros((S, 4), np.uint8)
    lib().orc_strategy_threshold(_p(lk, C.c_double), _p(lv, C.c_double), ncand, S,
                                 _p(cands, C.c_uint8), float(tau), D, _p(out, C.c_uint8))
    return out


def uniform_strategy(S: int, r_k: int, r_v: int, g: int = 1, B: int = 8):
    out = np.zeros((S, 4), np.uint8)
    out[:] = (r_k, r_v, g, B)
    return out


def blob_size(N: int, D: int, L: int, strat4) -> int:
    """bytes of the canonical export blob (0 if the strategy is invalid)."""
    strat4 = np.ascontiguousarray(strat4, np.uint8)
    return int(lib().orc_blob_size(N, D, L, _p(strat4, C.c_uint8)))


def compress_unit(k, v, L: int, strat4):
    """O5: canonical export blob (uint8 array) of one unit."""
    k, v = _u16(k), _u16(v)
    N, D = k.shape
    strat4 = np.ascontiguousarray(strat4, np.uint8)
    assert strat4.shape == ((N + L - 1) // L, 4)
    size = int(lib().orc_blob_size(N, D, L, _p(strat4, C.c_uint8)))
    if size == 0:
        raise ValueError("orc_blob_size: bad strategy")
    blob = np.zeros(size, np.uint8)
    rc = lib().orc_compress_unit(_p(k, C.c_uint16), _p(v, C.c_uint16), N, D, L,
                                 _p(strat4, C.c_uint8), _p(blob, C.c_uint8), size)
    if rc:
        raise ValueError(f"orc_compress_unit rc={rc}")
    return blob


def blob_header(blob):
    h = np.frombuffer(blob[:48].tobytes(), np.uint32)
    q = np.frombuffer(blob[24:40].tobytes(), np.uint64)
    return dict(magic=int(h[0]), D=int(h[1]), N=int(h[2]), L=int(h[3]), S=int(h[4]),
                tok_bytes=int(q[0]), bk_bytes=int(q[1]))


def blob_blocks(blob):
    n = lib().orc_blob_blocks(_p(blob, C.c_uint8), None, None)
    ft, nt = np.zeros(n, np.int32), np.zeros(n, np.int32)
    lib().orc_blob_blocks(_p(blob, C.c_uint8), _p(ft, C.c_int32), _p(nt, C.c_int32))
    return ft, nt


def unpack_unit(blob):
    """inverse of O5: dense bf16 K, V, block keys (zeros where dropped) + 0/1 masks."""
    h = blob_header(blob)
    N, D = h["N"], h["D"]
    nblk = lib().orc_blob_blocks(_p(blob, C.c_uint8), None, None)
    k, v = np.zeros((N, D), np.uint16), np.zeros((N, D), np.uint16)
    km, vm = np.zeros((N, D), np.uint8), np.zeros((N, D), np.uint8)
    bk, bm = np.zeros((nblk, D), np.uint16), np.zeros((nblk, D), np.uint8)
    lib().orc_unpack_unit(_p(blob, C.c_uint8), _p(k, C.c_uint16), _p(km, C.c_uint8),
                          _p(v, C.c_uint16), _p(vm, C.c_uint8), _p(bk, C.c_uint16),
                          _p(bm, C.c_uint8))
    return dict(k=k, k_mask=km, v=v, v_mask=vm, bk=bk, bk_mask=bm)


def scores(blob, q, mode: int = 0):
    """O6: fp64 block scores for q[G][D] (bf16 bits)."""
    q = _u16(q)
    G, _ = q.shape
    nblk = lib().orc_blob_blocks(_p(blob, C.c_uint8), None, None)
    s = np.zeros(nblk)
    lib().orc_scores(_p(blob, C.c_uint8), _p(q, C.c_uint16), G, mode, _p(s, C.c_double))
    return s


def topk(s, first_tok, n_tok, budget: int):
    """O7: selected blocks' first-token indices, ascending."""
    s = np.ascontiguousarray(s, np.float64)
    ft = np.ascontiguousarray(first_tok, np.int32)
    nt = np.ascontiguousarray(n_tok, np.int32)
    sel = np.zeros(max(1, s.shape[0]), np.int32)
    n = lib().orc_topk(_p(s, C.c_double), _p(ft, C.c_int32), _p(nt, C.c_int32), s.shape[0], budget,
                       _p(sel, C.c_int32))
    return sel[:n].copy()


def attention(blob, q, sel, scale: float, with_weights: bool = False):
    """O8: fp64 out[G][D], lse[G] over the selected blocks."""
    q = _u16(q)
    G, D = q.shape
    sel = np.ascontiguousarray(sel, np.int32)
    out, lse = np.zeros((G, D)), np.zeros(G)
    if not with_weights:
        rc = lib().orc_attention(_p(blob, C.c_uint8), _p(q, C.c_uint16), G, _p(sel, C.c_int32),
                                 sel.shape[0], float(scale), _p(out, C.c_double), _p(lse, C.c_double))
        if rc < 0:
            raise ValueError(f"orc_attention rc={rc}")
        return out, lse
    cap = sel.shape[0] * 64 + 1
    p = np.zeros((G, cap))
    toks = np.zeros(cap, np.int32)
    # first call to learn ntok
    n = lib().orc_attention_weights(_p(blob, C.c_uint8), _p(q, C.c_uint16), G, _p(sel, C.c_int32),
                                    sel.shape[0], float(scale), _p(out, C.c_double),
                                    _p(lse, C.c_double), None, _p(toks, C.c_int32), cap)
    if n < 0:
        raise ValueError(f"orc_attention_weights rc={n}")
    p = np.zeros((G, max(n, 1)))
    lib().orc_attention_weights(_p(blob, C.c_uint8), _p(q, C.c_uint16), G, _p(sel, C.c_int32),
                                sel.shape[0], float(scale), _p(out, C.c_double),
                                _p(lse, C.c_double), _p(p, C.c_double), _p(toks, C.c_int32), cap)
    return out, lse, p[:, :n], toks[:n].copy()


def merge(o1, lse1, o2, lse2):
    """split-K merge rule (step 3d)."""
    o1, o2 = np.ascontiguousarray(o1, np.float64), np.ascontiguousarray(o2, np.float64)
    l1, l2 = np.ascontiguousarray(lse1, np.float64), np.ascontiguousarray(lse2, np.float64)
    G, D = o1.shape
    out, lse = np.zeros((G, D)), np.zeros(G)
    lib().orc_merge(G, D, _p(o1, C.c_double), _p(l1, C.c_double), _p(o2, C.c_double),
                    _p(l2, C.c_double), _p(out, C.c_double), _p(lse, C.c_double))
    return out, lse


def attention_with_update_buffer(blob, q, sel, scale: float, k_buf, v_buf):
    """O8 + KV update buffer: the newest tokens are held uncompressed and attended
    densely next to the selected packed blocks.  fp64: O8 over the packed part, plain softmax
    attention over the buffer rows k_buf, v_buf [n][D] (bf16 bits), merged with the split-K rule
    (pinned: equals O8 on a blob that holds the buffer as a dense, fully selected segment)."""
    out, lse = attention(blob, q, sel, scale)
    k_buf, v_buf = _u16(k_buf), _u16(v_buf)
    if k_buf.shape[0] == 0:
        return out, lse
    f = lambda a: (a.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)
    logits = float(scale) * (f(_u16(q)) @ f(k_buf).T)  # [G][n]
    m = logits.max(axis=1)
    p = np.exp(logits - m[:, None])
    l = p.sum(axis=1)
    o_buf, lse_buf = (p @ f(v_buf)) / l[:, None], m + np.log(l)
    return merge(out, lse, o_buf, lse_buf)


def compress_units(k, v, L: int, strat4):
    """Batched O5 over units (OpenMP). k, v: [U][N][D]; strat4: [U][S][4]. Returns list of blobs."""
    k, v = _u16(k), _u16(v)
    U, N, D = k.shape
    strat4 = np.ascontiguousarray(strat4, np.uint8)
    S = (N + L - 1) // L
    assert strat4.shape == (U, S, 4)
    sizes = [int(lib().orc_blob_size(N, D, L, _p(strat4[u], C.c_uint8))) for u in range(U)]
    if min(sizes) == 0:
        raise ValueError("bad strategy")
    blobs = [np.zeros(s, np.uint8) for s in sizes]
    ptrs = (C.POINTER(C.c_uint8) * U)(*[_p(b, C.c_uint8) for b in blobs])
    caps = (C.c_uint64 * U)(*sizes)
    rc = lib().orc_compress_units(_p(k, C.c_uint16), _p(v, C.c_uint16), U, N, D, L,
                                  _p(strat4, C.c_uint8), ptrs, caps)
    if rc:
        raise ValueError(f"orc_compress_units rc={rc}")
    return blobs


def decode_units(blobs, q, budget: int, scale: float, mode: int = 0, k_max: int = None):
    """One decode step for every unit (O6 -> O7 -> O8), OpenMP over units.
    q: [U][G][D] bf16 bits. Returns sel [U][k_max], sel_count [U], out [U][G][D], lse [U][G]."""
    q = _u16(q)
    U, G, D = q.shape
    if k_max is None:
        k_max = max(1, max(int(lib().orc_blob_blocks(_p(b, C.c_uint8), None, None)) for b in blobs))
    ptrs = (C.POINTER(C.c_uint8) * U)(*[_p(b, C.c_uint8) for b in blobs])
    sel = np.full((U, k_max), -1, np.int32)
    cnt = np.zeros(U, np.int32)
    out, lse = np.zeros((U, G, D)), np.zeros((U, G))
    rc = lib().orc_decode_units(ptrs, U, _p(q, C.c_uint16), G, mode, budget, float(scale),
                                _p(sel, C.c_int32), _p(cnt, C.c_int32), k_max, _p(out, C.c_double),
                                _p(lse, C.c_double))
    if rc:
        raise ValueError(f"orc_decode_units rc={rc}")
    return sel, cnt, out, lse


def attention_units(blobs, q, sel, sel_count, scale: float):
    """O8 for every unit with a given selection (OpenMP over units).
    q: [U][G][D] bf16 bits; sel: [U][k_max] int32; sel_count: [U]. Returns out [U][G][D], lse [U][G]."""
    q = _u16(q)
    U, G, D = q.shape
    sel = np.ascontiguousarray(sel, np.int32)
    cnt = np.ascontiguousarray(sel_count, np.int32)
    ptrs = (C.POINTER(C.c_uint8) * U)(*[_p(b, C.c_uint8) for b in blobs])
    out, lse = np.zeros((U, G, D)), np.zeros((U, G))
    rc = lib().orc_attention_units(ptrs, U, _p(q, C.c_uint16), G, _p(sel, C.c_int32), _p(cnt, C.c_int32),
                                   sel.shape[1], float(scale), _p(out, C.c_double), _p(lse, C.c_double))
    if rc:
        raise ValueError(f"orc_attention_units rc={rc}")
    return out, lse


def rotate_query(q, R):
    """Rotation fold: q' = q R_k^T, fp32 FMA chain in ascending j, RNE to bf16.
    q: [n][D] bf16 bits, R: [D][D] float32.  Returns [n][D] bf16 bits."""
    q = _u16(q)
    n, D = q.shape
    R = np.ascontiguousarray(R, np.float32)
    assert R.shape == (D, D)
    out = np.zeros((n, D), np.uint16)
    lib().orc_rotate_query(_p(q, C.c_uint16), n, D, _p(R, C.c_float), _p(out, C.c_uint16))
    return out


def rotate_output(o, R):
    """out = o' R_v (the rotated cache 'must be transformed back'), fp64.  o: [n][D] float64."""
    o = np.array(o, np.float64, copy=True, order="C")
    n, D = o.shape
    R = np.ascontiguousarray(R, np.float32)
    assert R.shape == (D, D)
    lib().orc_rotate_output(_p(o, C.c_double), n, D, _p(R, C.c_float))
    return o
