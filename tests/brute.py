"""numpy brute-force references used to PIN the oracle (tests only).

Independent of oracle/: textbook definitions written with numpy (dense softmax attention,
stable argsort top-r / top-k, exhaustive mask enumeration).  Nothing here is used by the
CUDA path.
"""
import itertools

import numpy as np


def bf16_to_f64(bits):
    b = np.ascontiguousarray(bits, np.uint16).astype(np.uint32) << np.uint32(16)
    return b.view(np.float32).astype(np.float64)


def f32_to_bf16(x):
    u = np.ascontiguousarray(x, np.float32).view(np.uint32)
    lsb = (u >> np.uint32(16)) & np.uint32(1)
    return ((u + np.uint32(0x7FFF) + lsb) >> np.uint32(16)).astype(np.uint16)


def dense_attention(q, K, V, scale):
    """textbook softmax attention, fp64. q [G][D], K/V [T][D] (float64). Returns out [G][D], lse [G]."""
    z = scale * (q @ K.T)
    m = z.max(axis=1, keepdims=True)
    e = np.exp(z - m)
    s = e.sum(axis=1, keepdims=True)
    return (e / s) @ V, (m + np.log(s))[:, 0]


def masked_dense_attention(q, K, V, Mk, Mv, tok_mask, scale):
    """softmax(q (K*Mk)^T * scale + (-inf where token not selected)) (V*Mv)."""
    z = scale * (q @ (K * Mk).T)
    z = np.where(tok_mask[None, :], z, -np.inf)
    m = z.max(axis=1, keepdims=True)
    e = np.exp(z - m)
    s = e.sum(axis=1, keepdims=True)
    return (e / s) @ (V * Mv), (m + np.log(s))[:, 0]


def topr_mask(x_bits, r):
    """g = 1: keep the r largest |x| (15-bit magnitude), ties -> lower index; stable argsort."""
    mag = (np.asarray(x_bits, np.uint16) & 0x7FFF).astype(np.int64)
    order = np.argsort(-mag, kind="stable")
    keep = np.zeros(mag.shape[0], np.uint8)
    keep[order[:r]] = 1
    return keep


def topr_mask_groups(x_bits, g, r):
    x = bf16_to_f64(x_bits).astype(np.float32)
    D = x.shape[0]
    e = np.zeros(D // g, np.float32)
    for i in range(g):  # left-to-right fp32 energy
        e = (e + x[i::g] * x[i::g]).astype(np.float32)
    order = np.argsort(-e.astype(np.float64), kind="stable")
    keep = np.zeros(D // g, np.uint8)
    keep[order[: r // g]] = 1
    return keep


def best_mask_by_enumeration(x_bits, r):
    """all C(D, r) masks; returns the minimal dropped energy (Frobenius-optimal value)."""
    x = bf16_to_f64(x_bits)
    D = x.shape[0]
    best = None
    for comb in itertools.combinations(range(D), r):
        m = np.zeros(D, bool)
        m[list(comb)] = True
        loss = float((x[~m] ** 2).sum())
        if best is None or loss < best:
            best = loss
    return best


def topk_blocks(s, budget, B):
    """uniform block size: the floor(budget/B) best by (score desc, index asc), ascending index."""
    k = min(len(s), budget // B)
    order = np.argsort(-np.asarray(s, np.float64), kind="stable")
    return np.sort(order[:k])
