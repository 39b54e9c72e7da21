"""Thin ctypes binding of libmkv.so (include/mkv.h).  Argument marshalling only — every step
of the hot path runs in the library's CUDA kernels.  PyTorch supplies device memory and streams.

Importing this module loads the shared library and raises ImportError if it is missing: there
is no CPU fallback.  Build it with `python -m paper_2607_00760_b200.build`.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# MKV_LIBRARY: another build of the same sources (the -DMKV_TRACE library of trace.py); never set by tests or bench.py
LIB_PATH = os.environ.get("MKV_LIBRARY") or os.path.join(_HERE, "libmkv.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} not found: run `python -m paper_2607_00760_b200.build` "
                      "(the CUDA extension is required; there is no fallback)")
_lib = C.CDLL(LIB_PATH)

MKV_OK, MKV_E_ARG, MKV_E_UNSUPPORTED, MKV_E_NOMEM, MKV_E_CUDA, MKV_E_STATE, MKV_E_DEVICE = 0, -1, -2, -3, -4, -5, -6
MKV_DEV_ARENA_OVERFLOW, MKV_DEV_BAD_STRATEGY = 1, 2

# every symbol include/mkv.h declares (checked by tests/test_abi.py against the header text)
SYMBOLS = ["mkv_cache_create", "mkv_cache_free", "mkv_cache_reset", "mkv_segment_loss",
           "mkv_strategy_quantile", "mkv_strategy_threshold", "mkv_compress_segment", "mkv_select",
           "mkv_packed_attention", "mkv_update_append", "mkv_update_flush", "mkv_update_count", "mkv_calibrate_gather", "mkv_calibrate_stream", "mkv_calibrate_walk",
           "mkv_attention_stats", "mkv_rotation_set", "mkv_rotate_query", "mkv_rotate_output", "mkv_decode_step", "mkv_decode_host", "mkv_cache_export", "mkv_cache_bytes",
           "mkv_cache_status", "mkv_last_launch_count", "mkv_last_error", "mkv_version", "mkv_topk_static"]


class mkv_cache_desc(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("batch", C.c_int32), ("n_kv_heads", C.c_int32),
                ("n_q_heads", C.c_int32), ("head_dim", C.c_int32), ("max_tokens", C.c_int32),
                ("segment_len", C.c_int32), ("device", C.c_int32), ("arena_bytes", C.c_uint64),
                ("token_block", C.c_int32), ("reserved", C.c_int32)]


class mkv_strategy(C.Structure):
    _fields_ = [("r_k", C.c_uint8), ("r_v", C.c_uint8), ("g", C.c_uint8), ("B", C.c_uint8)]


_vp, _i32, _i64, _u64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64
_lib.mkv_cache_create.argtypes = [C.POINTER(mkv_cache_desc), C.POINTER(_vp)]
_lib.mkv_cache_free.argtypes = [_vp]
_lib.mkv_cache_reset.argtypes = [_vp, _i32, _vp]
_lib.mkv_segment_loss.argtypes = [_vp, _vp, _vp, _i64, _i64, _i64, _i32, _i32, _i32, _i32, _i32,
                                  mkv_strategy, _vp, _vp, _vp]
_lib.mkv_strategy_quantile.argtypes = [_vp, _vp, _vp, _i32, _i32, _i32, _i32, mkv_strategy, _vp, _vp]
_lib.mkv_strategy_threshold.argtypes = [_vp, _vp, _vp, _i32, _i32, _i32, C.POINTER(mkv_strategy),
                                        C.c_double, _vp, _vp]
_lib.mkv_compress_segment.argtypes = [_vp, _i32, _vp, _vp, _i64, _i64, _i64, _i32, _i32, _i32, _i32,
                                      _i32, _vp, _vp]
_lib.mkv_select.argtypes = [_vp, _i32, _vp, _i32, _i32, _vp, _vp, _i32, _vp, _vp]
_lib.mkv_packed_attention.argtypes = [_vp, _i32, _vp, _vp, _vp, _i32, C.c_float, _vp, _vp, _vp]
_lib.mkv_update_append.argtypes = [_vp, _i32, _vp, _vp, _i64, _i64, _i64, _i32, _vp]
_lib.mkv_update_flush.argtypes = [_vp, _i32, _vp, _vp]
_lib.mkv_update_count.argtypes = [_vp, _i32, C.POINTER(_i32)]
_lib.mkv_calibrate_gather.argtypes = [_vp, _i32, _vp, _vp, _i32, _vp]
_lib.mkv_calibrate_stream.argtypes = [_vp, _i32, _u64, _vp]
_lib.mkv_calibrate_walk.argtypes = [_vp, _i32, _vp, _vp, _vp, _i32, _i32, _vp]
_lib.mkv_attention_stats.argtypes = [_vp, C.POINTER(_u64), C.POINTER(_u64), C.POINTER(_u64), _i32]
_lib.mkv_rotation_set.argtypes = [_vp, _i32, _vp, _vp, _vp]
_lib.mkv_rotate_query.argtypes = [_vp, _i32, _vp, _vp, _vp]
_lib.mkv_rotate_output.argtypes = [_vp, _i32, _vp, _vp]
_lib.mkv_decode_step.argtypes = [_vp, _i32, _vp, _i32, _i32, C.c_float, _vp, _vp, _vp, _vp, _i32, _vp]
_lib.mkv_decode_host.argtypes = [_vp, _i32, _vp, _i32, _i32, C.c_float, _vp, _vp, _vp, _vp]
_lib.mkv_cache_export.argtypes = [_vp, _i32, _i32, _i32, _vp, _u64, C.POINTER(_u64)]
_lib.mkv_cache_bytes.argtypes = [_vp, _i32, C.POINTER(_u64), C.POINTER(_u64), C.POINTER(_u64)]
_lib.mkv_cache_status.argtypes = [_vp, C.POINTER(C.c_uint32)]
_lib.mkv_last_launch_count.argtypes = [_vp, C.POINTER(_i32), C.POINTER(_i32), C.POINTER(_i32)]
_lib.mkv_topk_static.argtypes = [_i32, _vp, _vp, _i32, _i32, _i32, _i32, _vp, _vp, _i32, _vp]
_lib.mkv_last_error.restype = C.c_char_p
for _n in SYMBOLS:
    if _n != "mkv_last_error":
        getattr(_lib, _n).restype = C.c_int


class MkvError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mkv error {code}: {msg}")
        self.code = code


def mkv_last_error() -> str:
    return _lib.mkv_last_error().decode()


def mkv_version() -> int:
    return _lib.mkv_version()


def _check(rc):
    if rc != MKV_OK:
        raise MkvError(rc, mkv_last_error())


def _ptr(t):
    """device/host pointer of a torch tensor, numpy array, int or None"""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream if isinstance(stream, int) else stream.cuda_stream


def _strategy(s):
    if isinstance(s, mkv_strategy):
        return s
    r_k, r_v, g, B = s
    return mkv_strategy(r_k, r_v, g, B)


def _kv_strides(k, v):
    assert k.dim() == 4 and k.shape == v.shape and k.stride() == v.stride() and k.stride(3) == 1
    assert k.element_size() == 2 and v.element_size() == 2
    return k.stride(0), k.stride(1), k.stride(2)


# ---- functions named as in include/mkv.h ---------------------------------------------------

def mkv_cache_create(n_layers, batch, n_kv_heads, n_q_heads, head_dim, max_tokens, segment_len,
                     device=0, arena_bytes=0, token_block=0):
    desc = mkv_cache_desc(n_layers, batch, n_kv_heads, n_q_heads, head_dim, max_tokens, segment_len,
                          device, arena_bytes, token_block, 0)
    h = _vp()
    _check(_lib.mkv_cache_create(C.byref(desc), C.byref(h)))
    return h


def mkv_cache_free(cache):
    _check(_lib.mkv_cache_free(cache))


def mkv_cache_reset(cache, layer=-1, stream=None):
    _check(_lib.mkv_cache_reset(cache, layer, _stream(stream)))


def mkv_segment_loss(cache, k, v, b0, seg0, cand, loss_k, loss_v, stream=None):
    """k, v: torch bf16 [nb][Hkv][n_tok][D] (any batch/head/token strides)."""
    sb, sh, st = _kv_strides(k, v)
    nb, _, n_tok, _ = k.shape
    L = cache_segment_len(cache)
    nseg = (n_tok + L - 1) // L
    _check(_lib.mkv_segment_loss(cache, _ptr(k), _ptr(v), sb, sh, st, b0, nb, seg0, nseg, n_tok,
                                 _strategy(cand), _ptr(loss_k), _ptr(loss_v), _stream(stream)))


def mkv_strategy_quantile(cache, loss_k, loss_v, n_units, nseg, dense_num, dense_den, sparse,
                          strat_out, stream=None):
    _check(_lib.mkv_strategy_quantile(cache, _ptr(loss_k), _ptr(loss_v), n_units, nseg, dense_num,
                                      dense_den, _strategy(sparse), _ptr(strat_out), _stream(stream)))


def mkv_strategy_threshold(cache, loss_k, loss_v, n_units, nseg, cands, tau, strat_out, stream=None):
    arr = (mkv_strategy * len(cands))(*[_strategy(c) for c in cands])
    _check(_lib.mkv_strategy_threshold(cache, _ptr(loss_k), _ptr(loss_v), len(cands), n_units, nseg,
                                       arr, float(tau), _ptr(strat_out), _stream(stream)))


def mkv_compress_segment(cache, layer, k, v, b0, seg0, strat, stream=None):
    """strat: torch uint8 [nb][Hkv][nseg][4] on the device."""
    sb, sh, st = _kv_strides(k, v)
    nb, _, n_tok, _ = k.shape
    L = cache_segment_len(cache)
    nseg = (n_tok + L - 1) // L
    _check(_lib.mkv_compress_segment(cache, layer, _ptr(k), _ptr(v), sb, sh, st, b0, nb, seg0, nseg,
                                     n_tok, _ptr(strat), _stream(stream)))


def mkv_select(cache, layer, q, token_budget, sel, sel_count, reduce=0, scores=None, stream=None):
    _check(_lib.mkv_select(cache, layer, _ptr(q), token_budget, reduce, _ptr(sel), _ptr(sel_count),
                           sel.shape[-1], _ptr(scores), _stream(stream)))


MKV_TOPK_STATIC_MAX_CANDIDATES = 1 << 19


def mkv_topk_static(device, scores, n_tokens, token_block, token_budget, sel, sel_count, stream=None):
    """Budgeted top-k on caller-owned scores [n_units][score_stride] with the library's static scratch: no
    cache, no device allocation (include/mkv.h).  n_tokens, sel [n_units][k_max], sel_count: int32 on the device."""
    n_units, score_stride = int(scores.shape[0]), int(scores.shape[-1])
    _check(_lib.mkv_topk_static(device, _ptr(scores), _ptr(n_tokens), n_units, score_stride, token_block,
                                token_budget, _ptr(sel), _ptr(sel_count), sel.shape[-1], _stream(stream)))


def mkv_packed_attention(cache, layer, q, sel, sel_count, softmax_scale, out, lse=None, stream=None):
    _check(_lib.mkv_packed_attention(cache, layer, _ptr(q), _ptr(sel), _ptr(sel_count), sel.shape[-1],
                                     float(softmax_scale), _ptr(out), _ptr(lse), _stream(stream)))


def mkv_update_append(cache, layer, k_new, v_new, stream=None):
    """k_new, v_new: torch bf16 [batch][Hkv][n_new][D] (any batch/head/token strides)."""
    sb, sh, st = _kv_strides(k_new, v_new)
    _check(_lib.mkv_update_append(cache, layer, _ptr(k_new), _ptr(v_new), sb, sh, st, k_new.shape[2], _stream(stream)))


def mkv_update_flush(cache, layer, strat, stream=None):
    """strat: torch uint8 [batch][Hkv][1][4] on the device."""
    _check(_lib.mkv_update_flush(cache, layer, _ptr(strat), _stream(stream)))


def mkv_update_count(cache, layer) -> int:
    n = _i32(0)
    _check(_lib.mkv_update_count(cache, layer, C.byref(n)))
    return n.value


def mkv_calibrate_gather(cache, layer, sel, sel_count, stream=None):
    _check(_lib.mkv_calibrate_gather(cache, layer, _ptr(sel), _ptr(sel_count), sel.shape[-1], _stream(stream)))


def mkv_calibrate_stream(cache, layer, nbytes, stream=None):
    _check(_lib.mkv_calibrate_stream(cache, layer, int(nbytes), _stream(stream)))


def mkv_calibrate_walk(cache, layer, q, sel, sel_count, reps, stream=None):
    _check(_lib.mkv_calibrate_walk(cache, layer, _ptr(q), _ptr(sel), _ptr(sel_count), sel.shape[-1], int(reps), _stream(stream)))


def mkv_attention_stats(cache, reset=False):
    a, b, c = _u64(0), _u64(0), _u64(0)
    _check(_lib.mkv_attention_stats(cache, C.byref(a), C.byref(b), C.byref(c), 1 if reset else 0))
    return dict(blocks=a.value, v_blocks=b.value, v_bytes=c.value)


def mkv_rotation_set(cache, layer, r_k, r_v, stream=None):
    """r_k, r_v: torch float32 [Hkv][D][D] on the device, or both None to remove the layer's rotation."""
    _check(_lib.mkv_rotation_set(cache, layer, _ptr(r_k), _ptr(r_v), _stream(stream)))


def mkv_rotate_query(cache, layer, q, q_out, stream=None):
    _check(_lib.mkv_rotate_query(cache, layer, _ptr(q), _ptr(q_out), _stream(stream)))


def mkv_rotate_output(cache, layer, out, stream=None):
    _check(_lib.mkv_rotate_output(cache, layer, _ptr(out), _stream(stream)))


def mkv_decode_step(cache, layer, q, token_budget, softmax_scale, out, reduce=0, lse=None, sel=None, sel_count=None,
                    stream=None):
    k_max = int(sel.shape[-1]) if sel is not None else 0
    _check(_lib.mkv_decode_step(cache, layer, _ptr(q), token_budget, reduce, float(softmax_scale), _ptr(out),
                                _ptr(lse), _ptr(sel), _ptr(sel_count), k_max, _stream(stream)))


def mkv_decode_host(cache, layer, q_host, token_budget, softmax_scale, out_host, reduce=0,
                    sel_host=None, sel_count_host=None, stream=None):
    _check(_lib.mkv_decode_host(cache, layer, _ptr(q_host), token_budget, reduce, float(softmax_scale),
                                _ptr(out_host), _ptr(sel_host), _ptr(sel_count_host), _stream(stream)))


def mkv_cache_export(cache, layer, b, h) -> np.ndarray:
    need = _u64(0)
    _check(_lib.mkv_cache_export(cache, layer, b, h, None, 0, C.byref(need)))
    buf = np.zeros(need.value, np.uint8)
    _check(_lib.mkv_cache_export(cache, layer, b, h, buf.ctypes.data, need.value, C.byref(need)))
    return buf


def mkv_cache_bytes(cache, layer):
    a, b, c = _u64(0), _u64(0), _u64(0)
    _check(_lib.mkv_cache_bytes(cache, layer, C.byref(a), C.byref(b), C.byref(c)))
    return dict(packed=a.value, block_keys=b.value, tables=c.value)


def mkv_cache_status(cache, raise_on_flag=True) -> int:
    f = C.c_uint32(0)
    rc = _lib.mkv_cache_status(cache, C.byref(f))
    if rc != MKV_OK and (raise_on_flag or rc != MKV_E_DEVICE):
        raise MkvError(rc, mkv_last_error())
    return f.value


def mkv_last_launch_count(cache):
    a, b, c = _i32(0), _i32(0), _i32(0)
    _check(_lib.mkv_last_launch_count(cache, C.byref(a), C.byref(b), C.byref(c)))
    return dict(select=a.value, attention=b.value, compress=c.value)


# ---- convenience wrapper ---------------------------------------------------------------------

_SEGLEN = {}


def cache_segment_len(cache):
    return _SEGLEN[cache.value]


class Cache:
    """Owns one mkv_cache; methods forward to the functions above (same names minus `mkv_`)."""

    def __init__(self, n_layers, batch, n_kv_heads, n_q_heads, head_dim=128, max_tokens=0,
                 segment_len=64, device=0, arena_bytes=0, token_block=8):
        self.h = mkv_cache_create(n_layers, batch, n_kv_heads, n_q_heads, head_dim, max_tokens,
                                  segment_len, device, arena_bytes, token_block)
        _SEGLEN[self.h.value] = segment_len
        self.n_layers, self.batch, self.n_kv_heads, self.n_q_heads = n_layers, batch, n_kv_heads, n_q_heads
        self.head_dim, self.max_tokens, self.segment_len = head_dim, max_tokens, segment_len
        self.n_units = batch * n_kv_heads
        self.token_block = token_block
        self.score_stride = (max_tokens + token_block - 1) // token_block

    def free(self):
        if self.h is not None:
            _SEGLEN.pop(self.h.value, None)
            mkv_cache_free(self.h)
            self.h = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass

    def reset(self, layer=-1, stream=None):
        mkv_cache_reset(self.h, layer, stream)

    def segment_loss(self, k, v, cand, loss_k, loss_v, b0=0, seg0=0, stream=None):
        mkv_segment_loss(self.h, k, v, b0, seg0, cand, loss_k, loss_v, stream)

    def strategy_quantile(self, loss_k, loss_v, nseg, dense_num, dense_den, sparse, strat_out,
                          n_units=None, stream=None):
        mkv_strategy_quantile(self.h, loss_k, loss_v, n_units or self.n_units, nseg, dense_num,
                              dense_den, sparse, strat_out, stream)

    def strategy_threshold(self, loss_k, loss_v, nseg, cands, tau, strat_out, n_units=None, stream=None):
        mkv_strategy_threshold(self.h, loss_k, loss_v, n_units or self.n_units, nseg, cands, tau,
                               strat_out, stream)

    def compress_segment(self, layer, k, v, strat, b0=0, seg0=0, stream=None):
        mkv_compress_segment(self.h, layer, k, v, b0, seg0, strat, stream)

    def select(self, layer, q, token_budget, sel, sel_count, reduce=0, scores=None, stream=None):
        mkv_select(self.h, layer, q, token_budget, sel, sel_count, reduce, scores, stream)

    def packed_attention(self, layer, q, sel, sel_count, softmax_scale, out, lse=None, stream=None):
        mkv_packed_attention(self.h, layer, q, sel, sel_count, softmax_scale, out, lse, stream)

    def update_append(self, layer, k_new, v_new, stream=None):
        mkv_update_append(self.h, layer, k_new, v_new, stream)

    def update_flush(self, layer, strat, stream=None):
        mkv_update_flush(self.h, layer, strat, stream)

    def update_count(self, layer):
        return mkv_update_count(self.h, layer)

    def calibrate_gather(self, layer, sel, sel_count, stream=None):
        mkv_calibrate_gather(self.h, layer, sel, sel_count, stream)

    def calibrate_stream(self, layer, nbytes, stream=None):
        mkv_calibrate_stream(self.h, layer, nbytes, stream)

    def calibrate_walk(self, layer, q, sel, sel_count, reps, stream=None):
        mkv_calibrate_walk(self.h, layer, q, sel, sel_count, reps, stream)

    def attention_stats(self, reset=False):
        return mkv_attention_stats(self.h, reset)

    def rotation_set(self, layer, r_k, r_v, stream=None):
        mkv_rotation_set(self.h, layer, r_k, r_v, stream)

    def rotate_query(self, layer, q, q_out, stream=None):
        mkv_rotate_query(self.h, layer, q, q_out, stream)

    def rotate_output(self, layer, out, stream=None):
        mkv_rotate_output(self.h, layer, out, stream)

    def decode_step(self, layer, q, token_budget, softmax_scale, out, reduce=0, lse=None, sel=None, sel_count=None,
                    stream=None):
        mkv_decode_step(self.h, layer, q, token_budget, softmax_scale, out, reduce, lse, sel, sel_count, stream)

    def decode_host(self, layer, q_host, token_budget, softmax_scale, out_host, reduce=0,
                    sel_host=None, sel_count_host=None, stream=None):
        mkv_decode_host(self.h, layer, q_host, token_budget, softmax_scale, out_host, reduce,
                        sel_host, sel_count_host, stream)

    def export(self, layer, b, h):
        return mkv_cache_export(self.h, layer, b, h)

    def bytes(self, layer):
        return mkv_cache_bytes(self.h, layer)

    def status(self, raise_on_flag=True):
        return mkv_cache_status(self.h, raise_on_flag)

    def last_launch_count(self):
        return mkv_last_launch_count(self.h)
