"""Pins for the CPU oracle (P1..P12): closed forms, invariants, special cases that
reduce to textbook routines, brute force on tiny inputs.  CPU only (-m "not gpu").

Each pin is chosen so that a plausible mistake in the oracle (dropped term, wrong sign or
index, transposed operand, wrong tie-break, wrong byte order) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest

import brute
import oracle as orc
from paper_2607_00760_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def rand_bf16(rng, shape, scale=1.0):
    return synth.f32_to_bf16_bits((rng.standard_normal(shape) * scale).astype(np.float32))


def small_unit(seed=1, N=200, D=128, G=4):
    """one unit with the generator's structure, ragged tail (N not a multiple of 8 or 64)."""
    K, V, q = synth.make_inputs_np(1, 1, G, N, D, 64, seed=seed)
    return K[0, 0], V[0, 0], q[0]


# ----------------------------------------------------------------------------- P6: top-r (O1)

@pytest.mark.parametrize("D,r", [(128, 38), (128, 1), (128, 127), (128, 128), (64, 16), (8, 3)])
def test_P6_topr_matches_stable_argsort(D, r):
    rng = np.random.default_rng(10 + D + r)
    for trial in range(40):
        x = rand_bf16(rng, D, scale=3.0)
        if trial % 4 == 0:  # force ties: coarse values and +-0
            x = synth.f32_to_bf16_bits(rng.integers(-2, 3, D).astype(np.float32))
            x[rng.integers(0, D)] = 0x8000  # -0.0
        keep = orc.topr(x, 1, r)
        np.testing.assert_array_equal(keep, brute.topr_mask(x, r))
        assert keep.sum() == r


def test_P6_topr_tie_goes_to_lower_index():
    x = synth.f32_to_bf16_bits(np.array([1, -1, 1, -1, 1, -1, 1, -1], np.float32))
    np.testing.assert_array_equal(orc.topr(x, 1, 3), [1, 1, 1, 0, 0, 0, 0, 0])
    x = synth.f32_to_bf16_bits(np.array([0.5, 2, -2, 0.5, 2, 0.25, -2, 0.5], np.float32))
    np.testing.assert_array_equal(orc.topr(x, 1, 3), [0, 1, 1, 0, 1, 0, 0, 0])
    np.testing.assert_array_equal(orc.topr(x, 1, 5), [1, 1, 1, 0, 1, 0, 1, 0])


def test_P6_topr_is_frobenius_optimal_by_enumeration():
    rng = np.random.default_rng(3)
    for _ in range(20):
        x = rand_bf16(rng, 8, 2.0)
        keep = orc.topr(x, 1, 3).astype(bool)
        dropped = float((brute.bf16_to_f64(x)[~keep] ** 2).sum())
        assert dropped == pytest.approx(brute.best_mask_by_enumeration(x, 3), rel=0, abs=0)


@pytest.mark.parametrize("g,r", [(2, 32), (4, 32), (2, 2), (4, 124)])
def test_P6_topr_groups(g, r):
    rng = np.random.default_rng(g * 100 + r)
    for _ in range(20):
        x = rand_bf16(rng, 128, 2.0)
        keep = orc.topr(x, g, r)
        np.testing.assert_array_equal(keep, brute.topr_mask_groups(x, g, r))
        assert keep.sum() == r // g


def test_P6_group_mask_is_frobenius_optimal_by_enumeration():
    """Independent pin of the g > 1 rank key ("selects groups of adjacent elements together";
    DESIGN.md R4): the kept groups must minimise the dropped energy over ALL C(D/g, r/g) group masks.  The
    enumeration below knows nothing of the oracle's key (it sums squares in fp64 over explicit masks); a wrong
    group stride, a key that ranks by max |x| or by the first element only, or keeping the smallest groups
    fails it.  Inputs are small integers, so energies are exact and ties are real: among equal-energy groups the
    lower group index must be kept (north_star tie rule)."""
    import itertools
    rng = np.random.default_rng(17)
    for D, g, r in [(8, 2, 4), (8, 2, 2), (8, 2, 6), (16, 4, 8), (16, 4, 4), (12, 2, 6)]:
        ng, nk = D // g, r // g
        for trial in range(30):
            if trial % 3 == 0:   # integers -> exact ties between groups
                x = synth.f32_to_bf16_bits(rng.integers(-3, 4, D).astype(np.float32))
            else:
                x = rand_bf16(rng, D, 2.0)
            xf = brute.bf16_to_f64(x)
            e = (xf.reshape(ng, g) ** 2).sum(axis=1)          # exact in fp64 (bf16 squares, <= 4 terms)
            keep = orc.topr(x, g, r).astype(bool)
            assert keep.sum() == nk
            best, best_masks = None, []
            for comb in itertools.combinations(range(ng), nk):
                m = np.zeros(ng, bool)
                m[list(comb)] = True
                loss = float(e[~m].sum())
                if best is None or loss < best - 1e-300:
                    best, best_masks = loss, [m]
                elif loss == best:
                    best_masks.append(m)
            assert float(e[~keep].sum()) == best, (D, g, r, trial)
            # among the optimal masks the oracle's is the one that prefers lower group indices:
            # lexicographically largest keep-vector read from group 0 upwards
            lex = max(best_masks, key=lambda m: tuple(m.astype(int)))
            if trial % 3 == 0:
                np.testing.assert_array_equal(keep, lex)


# ----------------------------------------------------------------------------- P9: block key (O2)

def test_P9_block_key_constant_block_and_B1():
    rng = np.random.default_rng(5)
    x = rand_bf16(rng, 128, 2.0)
    # exact for power-of-two blocks: sum of nb equal bf16 values /nb is that value
    for nb in (1, 2, 4, 8, 16):
        np.testing.assert_array_equal(orc.block_key(np.tile(x, (nb, 1))), x)


def test_P9_block_key_is_fp32_sequential_mean_rounded_rne():
    rng = np.random.default_rng(6)
    k = rand_bf16(rng, (8, 128), 3.0)
    kf = brute.bf16_to_f64(k).astype(np.float32)
    s = np.zeros(128, np.float32)
    for t in range(8):
        s = (s + kf[t]).astype(np.float32)
    np.testing.assert_array_equal(orc.block_key(k), brute.f32_to_bf16((s / np.float32(8)).astype(np.float32)))
    # close to the exact mean: |bk - mean| <= 2^-8 |mean| + fp32 noise
    exact = brute.bf16_to_f64(k).mean(axis=0)
    got = brute.bf16_to_f64(orc.block_key(k))
    assert np.all(np.abs(got - exact) <= 2.0 ** -8 * np.abs(exact) + 1e-6)
    # ragged block: nb = 3 uses IEEE division
    s3 = ((kf[0] + kf[1]).astype(np.float32) + kf[2]).astype(np.float32)
    np.testing.assert_array_equal(orc.block_key(k[:3]), brute.f32_to_bf16((s3 / np.float32(3)).astype(np.float32)))


# ----------------------------------------------------------------------------- P2: pack / unpack (O5)

@pytest.mark.parametrize("r,g,B", [(38, 1, 8), (128, 1, 8), (64, 2, 8), (32, 4, 16), (90, 1, 4)])
def test_P2_roundtrip(r, g, B):
    K, V, _ = small_unit(seed=r + g, N=200)
    S = 4
    blob = orc.compress_unit(K, V, 64, orc.uniform_strategy(S, r, r, g, B))
    u = orc.unpack_unit(blob)
    for X, name in ((K, "k"), (V, "v")):
        mask = u[name + "_mask"]
        assert np.all(mask.sum(axis=1) == r)
        np.testing.assert_array_equal(u[name], np.where(mask == 1, X, 0).astype(np.uint16))
        if g == 1:
            for t in (0, 63, 64, 199):
                np.testing.assert_array_equal(mask[t], brute.topr_mask(X[t], r))
    if r == 128:
        np.testing.assert_array_equal(u["k"], K)
        np.testing.assert_array_equal(u["v"], V)
    # idempotent: packing the unpacked K/V again gives the same token arena
    blob2 = orc.compress_unit(u["k"], u["v"], 64, orc.uniform_strategy(S, r, r, g, B))
    h = orc.blob_header(blob)
    t0 = len(blob) - h["tok_bytes"] - h["bk_bytes"]
    np.testing.assert_array_equal(blob[t0:t0 + h["tok_bytes"]], blob2[t0:t0 + h["tok_bytes"]])


def test_P2_block_keys_in_blob_are_means_with_same_topr():
    K, V, _ = small_unit(seed=9, N=200)
    blob = orc.compress_unit(K, V, 64, orc.uniform_strategy(4, 38, 38))
    u = orc.unpack_unit(blob)
    ft, nt = orc.blob_blocks(blob)
    assert len(ft) == 25 and nt[-1] == 8 and ft[-1] == 192
    for b in (0, 7, 8, 24):
        bk = orc.block_key(K[ft[b]:ft[b] + nt[b]])
        m = brute.topr_mask(bk, 38)
        np.testing.assert_array_equal(u["bk_mask"][b], m)
        np.testing.assert_array_equal(u["bk"][b], np.where(m == 1, bk, 0))


def test_P2_hand_worked_layout_D8():
    """bytes of one tiny unit worked out by hand from the format text (tests/golden/layout_d8.txt)."""
    vals_k = np.array([[1.0, -3.0, 0.5, 2.0, 0.0, -0.25, 4.0, 1.5], [2.0, 2.0, -2.0, 1.0, 8.0, 0.0, 0.0, -1.0]], np.float32)
    vals_v = np.array([[0.5, 0.25, -8.0, 0.0, 1.0, -1.0, 2.0, 3.0], [1.0, 1.0, 1.0, 1.0, -1.0, -1.0, -1.0, -1.0]], np.float32)
    K, V = synth.f32_to_bf16_bits(vals_k), synth.f32_to_bf16_bits(vals_v)
    blob = orc.compress_unit(K, V, 4, np.array([[3, 2, 1, 2]], np.uint8))
    lines = [l.split("#")[0].strip() for l in open(os.path.join(GOLDEN, "layout_d8.txt")) if l.split("#")[0].strip()]
    expect = np.array([int(x, 16) for l in lines for x in l.split()], np.uint8)
    np.testing.assert_array_equal(blob, expect)


# ----------------------------------------------------------------------------- P3: byte accounting

def test_P3_paper_memory_figures():
    """PAPER.md:293 (3x vs Full, 3.18x vs Quest at 25 % retention), :196 (bitmap = 12.5 %), :317 (1.44M tokens)."""
    fig = {}
    for line in open(os.path.join(GOLDEN, "paper_memory_figures.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            fig[k.strip()] = float(v)
    N, D, L = 4096, 128, 64
    S = N // L
    size = orc.blob_size(N, D, L, orc.uniform_strategy(S, 32, 32))
    payload = size - (48 + 16 * S)  # minus header + tables
    per_token = payload / N
    assert per_token == fig["bytes_per_token_r32_B8"]  # 2*(16+64) + (16+64)/8
    full = 2 * D * 2
    assert full / per_token == pytest.approx(fig["ratio_vs_full"], abs=0.02)          # paper: 3x
    quest = full * (1 + fig["quest_overhead"])
    assert quest / per_token == pytest.approx(fig["ratio_vs_quest"], abs=0.03)        # paper: 3.18x
    # bitmap bytes = 12.5 % of a vector of D 8-bit elements
    assert (D // 8) / (D * 1.0) == fig["bitmap_fraction_of_8bit_vector"]
    # 1.44M tokens of LLaMA-3.1-8B (32 layers x 8 KV heads) + ~16 GB of weights fit 80 GB; Full at 512K does not
    ours = fig["max_tokens"] * per_token * 8 * 32
    assert ours + 16e9 < 80e9 * 1.0 and ours + 16e9 > 0.95 * 80e9
    assert 512 * 1024 * full * 8 * 32 + 16e9 > 80e9


def test_P3_sizes_of_measured_strategies():
    D = 128
    def blk(r, nb=8):
        return orc.blob_size(nb, D, 64, orc.uniform_strategy(1, r, r)) - 64
    # token block payload + that block's share of the block-key payload (padded to 16)
    assert blk(38) == 1472 + 96 and blk(128) == 4096 + 256 and blk(90) == 3136 + 208 and blk(64) == 2304 + 144


# ----------------------------------------------------------------------------- P1: dense equivalence (O6-O8)

def test_P1_no_compression_equals_dense_softmax_attention():
    K, V, q = small_unit(seed=2, N=200)
    blob = orc.compress_unit(K, V, 64, orc.uniform_strategy(4, 128, 128))
    ft, nt = orc.blob_blocks(blob)
    s = orc.scores(blob, q)
    sel = orc.topk(s, ft, nt, 10 ** 6)
    np.testing.assert_array_equal(sel, ft)
    scale = 1 / math.sqrt(128)
    out, lse = orc.attention(blob, q, sel, scale)
    ref_o, ref_l = brute.dense_attention(brute.bf16_to_f64(q), brute.bf16_to_f64(K), brute.bf16_to_f64(V), scale)
    np.testing.assert_allclose(out, ref_o, rtol=0, atol=1e-12)
    np.testing.assert_allclose(lse, ref_l, rtol=0, atol=1e-12)


# ----------------------------------------------------------------------------- P5: brute-force masked attention

@pytest.mark.parametrize("D,r,N,G", [(128, 38, 200, 4), (8, 3, 50, 2), (128, 90, 96, 7)])
def test_P5_bruteforce_masked_dense_attention(D, r, N, G):
    rng = np.random.default_rng(D + r)
    if D == 128:
        K, V, q = small_unit(seed=D + r, N=N, D=D, G=G)
    else:
        K, V, q = rand_bf16(rng, (N, D), 2.0), rand_bf16(rng, (N, D)), rand_bf16(rng, (G, D))
    L, B = 64 if D == 128 else 16, 8 if D == 128 else 4
    S = (N + L - 1) // L
    blob = orc.compress_unit(K, V, L, orc.uniform_strategy(S, r, r, 1, B))
    ft, nt = orc.blob_blocks(blob)
    Kf, Vf, qf = brute.bf16_to_f64(K), brute.bf16_to_f64(V), brute.bf16_to_f64(q)
    Mk = np.stack([brute.topr_mask(K[t], r) for t in range(N)]).astype(np.float64)
    Mv = np.stack([brute.topr_mask(V[t], r) for t in range(N)]).astype(np.float64)
    # scores: q . topr(mean key)
    s = orc.scores(blob, q, mode=0)
    s_sum = orc.scores(blob, q, mode=1)
    for b in range(len(ft)):
        kf32 = Kf[ft[b]:ft[b] + nt[b]].astype(np.float32)
        acc = np.zeros(D, np.float32)
        for t in range(nt[b]):
            acc = (acc + kf32[t]).astype(np.float32)
        bk = brute.f32_to_bf16((acc / np.float32(nt[b])).astype(np.float32))
        bkf = brute.bf16_to_f64(bk) * brute.topr_mask(bk, r)
        per_head = qf @ bkf
        assert s[b] == pytest.approx(per_head.max(), rel=1e-13, abs=1e-13)
        assert s_sum[b] == pytest.approx(per_head.sum(), rel=1e-12, abs=1e-12)
    budget = 5 * B
    sel = orc.topk(s, ft, nt, budget)
    tok_mask = np.zeros(N, bool)
    for t0 in sel:
        tok_mask[t0:t0 + B] = True
    scale = 1 / math.sqrt(D)
    out, lse = orc.attention(blob, q, sel, scale)
    ref_o, ref_l = brute.masked_dense_attention(qf, Kf, Vf, Mk, Mv, tok_mask, scale)
    np.testing.assert_allclose(out, ref_o, rtol=0, atol=1e-12)
    np.testing.assert_allclose(lse, ref_l, rtol=0, atol=1e-12)


# ----------------------------------------------------------------------------- P4: softmax invariants

def test_P4_weights_sum_to_one_and_output_in_hull():
    K, V, q = small_unit(seed=4, N=200)
    blob = orc.compress_unit(K, V, 64, orc.uniform_strategy(4, 38, 38))
    ft, nt = orc.blob_blocks(blob)
    sel = orc.topk(orc.scores(blob, q), ft, nt, 64)
    out, lse, p, toks = orc.attention(blob, q, sel, 1 / math.sqrt(128), with_weights=True)
    np.testing.assert_allclose(p.sum(axis=1), 1.0, rtol=0, atol=1e-12)
    assert len(toks) == 64 and np.all(p >= 0)
    u = orc.unpack_unit(blob)
    Vm = brute.bf16_to_f64(u["v"])[toks]  # masked V rows (zeros where dropped)
    assert np.all(out <= Vm.max(axis=0) + 1e-12) and np.all(out >= Vm.min(axis=0) - 1e-12)


# ----------------------------------------------------------------------------- P7: top-k (O7)

def test_P7_topk_bruteforce_ties_budget_order():
    rng = np.random.default_rng(7)
    for trial in range(30):
        nblk = int(rng.integers(1, 80))
        s = rng.integers(-3, 4, nblk).astype(np.float64) if trial % 2 else rng.standard_normal(nblk)
        if trial % 5 == 0:
            s[rng.integers(0, nblk)] = -0.0
        B = 8
        ft = np.arange(nblk, dtype=np.int32) * B
        nt = np.full(nblk, B, np.int32)
        budget = int(rng.integers(0, nblk * B + 20))
        sel = orc.topk(s, ft, nt, budget)
        np.testing.assert_array_equal(sel // B, brute.topk_blocks(s, budget, B))
        assert len(sel) * B <= budget or len(sel) == nblk
        assert np.all(np.diff(sel) > 0)


def test_P7_topk_ragged_last_block_walk():
    # 5 blocks, the last has 3 tokens. budget 19 = 2 full blocks + 3
    ft = np.array([0, 8, 16, 24, 32], np.int32)
    nt = np.array([8, 8, 8, 8, 3], np.int32)
    # ragged block ranks 3rd: fits in the remainder -> taken, then the walk stops
    np.testing.assert_array_equal(orc.topk(np.array([5., 1., 4., 0., 3.]), ft, nt, 19), [0, 16, 32])
    # ragged block ranks 1st: 3 + 8 + 8 = 19 fits -> three blocks
    np.testing.assert_array_equal(orc.topk(np.array([5., 1., 4., 0., 9.]), ft, nt, 19), [0, 16, 32])
    # ragged block ranks last: two full blocks, third full block does not fit -> stop
    np.testing.assert_array_equal(orc.topk(np.array([5., 1., 4., 2., 0.]), ft, nt, 19), [0, 16])
    # budget 18: remainder 2 < 3 -> ragged block never fits as the third
    np.testing.assert_array_equal(orc.topk(np.array([5., 1., 4., 0., 3.]), ft, nt, 18), [0, 16])
    # everything fits
    np.testing.assert_array_equal(orc.topk(np.array([5., 1., 4., 0., 3.]), ft, nt, 35), ft)
    assert len(orc.topk(np.array([5., 1., 4., 0., 3.]), ft, nt, 7)) == 0


def test_P7_attention_invariant_under_permutation_of_selection():
    K, V, q = small_unit(seed=8, N=200)
    blob = orc.compress_unit(K, V, 64, orc.uniform_strategy(4, 38, 38))
    sel = np.array([0, 40, 64, 128, 192], np.int32)
    o1, l1 = orc.attention(blob, q, sel, 0.1)
    o2, l2 = orc.attention(blob, q, sel[::-1].copy(), 0.1)
    np.testing.assert_allclose(o1, o2, rtol=0, atol=1e-13)
    np.testing.assert_allclose(l1, l2, rtol=0, atol=1e-13)


# ----------------------------------------------------------------------------- P8: loss (O3)

def test_P8_loss_properties_and_gaussian_closed_form():
    rng = np.random.default_rng(8)
    N, D = 64 * 64, 128
    V = synth.f32_to_bf16_bits(rng.standard_normal((N, D)).astype(np.float32))
    K = synth.f32_to_bf16_bits((rng.standard_normal((N, D)) * np.exp(rng.standard_normal(D))).astype(np.float32))
    prev = None
    for r in (128, 90, 64, 38, 8):
        lk, lv = orc.segment_loss(K[:256], V[:256], 64, r, r)
        assert np.all(lk >= 0) and np.all(lk <= 1) and np.all(lv >= 0) and np.all(lv <= 1)
        if r == 128:
            assert np.all(lk == 0) and np.all(lv == 0)
        if prev is not None:
            assert np.all(lk >= prev[0]) and np.all(lv >= prev[1])  # non-increasing in r
        prev = (lk, lv)
    # brute force for one segment
    lk, lv = orc.segment_loss(K[:64], V[:64], 64, 38, 38)
    Vf = brute.bf16_to_f64(V[:64])
    M = np.stack([brute.topr_mask(V[t], 38) for t in range(64)]).astype(bool)
    assert lv[0] == pytest.approx((Vf[~M] ** 2).sum() / (Vf ** 2).sum(), rel=1e-13)
    # iid N(0,1): keeping the fraction f = r/D largest |x| leaves
    #   L = 1 - 2 [ z phi(z) + 1 - Phi(z) ],  z = Phi^-1(1 - f/2)     (truncated second moment)
    from scipy.stats import norm
    _, lv = orc.segment_loss(K, V, 64, 38, 38)
    f = 38 / 128
    z = norm.ppf(1 - f / 2)
    closed = 1 - 2 * (z * norm.pdf(z) + 1 - norm.cdf(z))
    assert closed == pytest.approx(0.220, abs=2e-3)
    assert lv.mean() == pytest.approx(closed, abs=1e-2)
    # scale invariance per segment: K scaled by a power of two has the same loss
    Ks = synth.f32_to_bf16_bits(brute.bf16_to_f64(K[:128]).astype(np.float32) * np.float32(4.0))
    np.testing.assert_allclose(orc.segment_loss(Ks, V[:128], 64, 38, 38)[0], orc.segment_loss(K[:128], V[:128], 64, 38, 38)[0], rtol=1e-14)


# ----------------------------------------------------------------------------- P9 / P11: score special cases

def test_P9_B1_score_equals_logit_over_scale_and_P11_G1_modes_coincide():
    K, V, q = small_unit(seed=11, N=96, G=1)
    blob = orc.compress_unit(K, V, 64, orc.uniform_strategy(2, 38, 38, 1, 1))  # block size 1
    ft, nt = orc.blob_blocks(blob)
    assert len(ft) == 96 and np.all(nt == 1)
    s0, s1 = orc.scores(blob, q, 0), orc.scores(blob, q, 1)
    np.testing.assert_array_equal(s0, s1)  # P11: G = 1 -> max == sum
    # B = 1: block key == key, so the score is the attention logit / scale of that token
    u = orc.unpack_unit(blob)
    logits = brute.bf16_to_f64(q)[0] @ brute.bf16_to_f64(u["k"]).T
    np.testing.assert_allclose(s0, logits, rtol=0, atol=1e-12)
    # and per-query selection == top-k over logits
    sel = orc.topk(s0, ft, nt, 10)
    np.testing.assert_array_equal(sel, np.sort(np.argsort(-logits, kind="stable")[:10]))


# ----------------------------------------------------------------------------- P10: split-K merge

def test_P10_merge_of_halves_equals_single_pass():
    K, V, q = small_unit(seed=12, N=200)
    blob = orc.compress_unit(K, V, 64, orc.uniform_strategy(4, 38, 38))
    sel = np.array([0, 8, 64, 72, 128, 184, 192], np.int32)
    o, l = orc.attention(blob, q, sel, 0.09)
    o1, l1 = orc.attention(blob, q, sel[:3], 0.09)
    o2, l2 = orc.attention(blob, q, sel[3:], 0.09)
    om, lm = orc.merge(o1, l1, o2, l2)
    np.testing.assert_allclose(om, o, rtol=0, atol=1e-12)
    np.testing.assert_allclose(lm, l, rtol=0, atol=1e-12)
    # empty partial is the identity
    oe, le = orc.attention(blob, q, sel[:0], 0.09)
    assert np.all(oe == 0) and np.all(np.isneginf(le))
    om, lm = orc.merge(o, l, oe, le)
    np.testing.assert_allclose(om, o, rtol=0, atol=1e-15)


# ----------------------------------------------------------------------------- P13: KV update buffer

@pytest.mark.parametrize("n_buf", [1, 7, 8, 13, 32, 64])
def test_P13_update_buffer_equals_dense_selected_segment(n_buf):
    """the buffered (uncompressed) tokens are attended next to the selected packed blocks.
    Pin: the result equals O8 on a blob that holds the buffer as one more, dense and fully selected
    segment, and the brute-force masked dense attention of tests/brute.py."""
    N = 192
    K, V, q = small_unit(seed=21, N=N + n_buf)
    blob = orc.compress_unit(K[:N], V[:N], 64, orc.uniform_strategy(3, 38, 38))
    sel = np.array([0, 16, 64, 120, 184], np.int32)
    o, l = orc.attention_with_update_buffer(blob, q, sel, 0.11, K[N:], V[N:])
    strat = orc.uniform_strategy(4, 38, 38)
    strat[3, 0:2] = 128
    blob2 = orc.compress_unit(K, V, 64, strat)
    sel2 = np.concatenate([sel, N + 8 * np.arange((n_buf + 7) // 8)]).astype(np.int32)
    o2, l2 = orc.attention(blob2, q, sel2, 0.11)
    np.testing.assert_allclose(o, o2, rtol=0, atol=1e-12)
    np.testing.assert_allclose(l, l2, rtol=0, atol=1e-12)
    un = orc.unpack_unit(blob2)
    Kd, Vd, Mk, Mv = un["k"], un["v"], un["k_mask"], un["v_mask"]
    tok = np.zeros(N + n_buf, bool)
    for t0 in sel2:
        tok[t0:t0 + 8] = True
    ob, lb = brute.masked_dense_attention(brute.bf16_to_f64(q), brute.bf16_to_f64(Kd), brute.bf16_to_f64(Vd),
                                          Mk.astype(np.float64), Mv.astype(np.float64), tok, 0.11)
    np.testing.assert_allclose(o, ob, rtol=0, atol=1e-12)
    np.testing.assert_allclose(l, lb, rtol=0, atol=1e-12)
    # an empty selection leaves plain dense attention over the buffer
    oe, le = orc.attention_with_update_buffer(blob, q, sel[:0], 0.11, K[N:], V[N:])
    od, ld = brute.dense_attention(brute.bf16_to_f64(q), brute.bf16_to_f64(K[N:]), brute.bf16_to_f64(V[N:]), 0.11)
    np.testing.assert_allclose(oe, od, rtol=0, atol=1e-12)
    np.testing.assert_allclose(le, ld, rtol=0, atol=1e-12)


# ----------------------------------------------------------------------------- P12: strategies (O4)

def test_P12_quantile_and_threshold():
    rng = np.random.default_rng(13)
    for S in (1, 10, 11, 64, 2048):
        lk, lv = rng.random(S), rng.random(S)
        st = orc.strategy_quantile(lk, lv, 1, 10, 128, 38, 38)
        dense = (st[:, 0] == 128)
        assert dense.sum() == math.ceil(S / 10) and np.all(st[dense, 1] == 128)
        assert np.all(st[~dense, 0] == 38) and np.all(st[:, 2] == 1) and np.all(st[:, 3] == 8)
        I = 0.5 * (lk + lv)
        order = np.argsort(-I, kind="stable")[: dense.sum()]
        assert set(np.nonzero(dense)[0]) == set(order)
    # ties -> lower segment index
    st = orc.strategy_quantile(np.ones(20), np.ones(20), 1, 10, 128, 38, 38)
    np.testing.assert_array_equal(np.nonzero(st[:, 0] == 128)[0], [0, 1])
    assert (orc.strategy_quantile(np.ones(20), np.ones(20), 0, 1, 128, 38, 38)[:, 0] == 38).all()
    # threshold rule
    cands = np.array([[16, 16, 4, 8], [32, 32, 2, 8], [48, 48, 1, 8]], np.uint8)
    lk = np.array([[0.5, 0.3, 0.1], [0.4, 0.2, 0.05], [0.3, 0.1, 0.01]])
    st = orc.strategy_threshold(lk, lk, cands, float("inf"), 128)
    assert (st == cands[0]).all()
    st = orc.strategy_threshold(lk, lk, cands, -1.0, 128)
    assert (st[:, 0] == 128).all() and (st[:, 1] == 128).all() and (st[:, 2] == 1).all()
    st = orc.strategy_threshold(lk, lk, cands, 0.25, 128)
    np.testing.assert_array_equal(st, [[128, 128, 1, 8], [32, 32, 2, 8], [16, 16, 4, 8]])


# ----------------------------------------------------------------------------- batched drivers

def test_batched_drivers_equal_per_unit_calls():
    """orc_compress_units / orc_decode_units / orc_attention_units (the OpenMP drivers that bench.py's cpu_baseline
    times) against the per-unit functions pinned above, on 3 units with different K, V, q and strategies: a wrong
    per-unit offset (q + u*G*D, sel + u*k_max, blob pointer) changes a unit's result and fails here."""
    G, N, L, D = 4, 1000, 64, 128
    K, V, q = synth.make_inputs_np(3, 1, G, N, D, L, seed=21)
    K, V, q = K[:, 0], V[:, 0], q  # [3][N][D], [3][G][D]
    S = (N + L - 1) // L
    strat = np.stack([orc.uniform_strategy(S, 38, 38), orc.uniform_strategy(S, 64, 90), orc.uniform_strategy(S, 128, 38)])
    strat[1, ::3, 0:2] = 128
    blobs = orc.compress_units(K, V, L, strat)
    for u in range(3):
        np.testing.assert_array_equal(blobs[u], orc.compress_unit(K[u], V[u], L, strat[u]))
    scale, budget = 1.0 / math.sqrt(D), 256
    for mode in (0, 1):
        sel, cnt, out, lse = orc.decode_units(blobs, q, budget, scale, mode, k_max=budget // 8 + 1)
        for u in range(3):
            ft, nt = orc.blob_blocks(blobs[u])
            s = orc.scores(blobs[u], q[u], mode)
            ref = orc.topk(s, ft, nt, budget)
            assert cnt[u] == len(ref)
            np.testing.assert_array_equal(sel[u, :cnt[u]], ref)
            o, l = orc.attention(blobs[u], q[u], ref, scale)
            np.testing.assert_array_equal(out[u], o)
            np.testing.assert_array_equal(lse[u], l)
    # attention_units on a selection that differs per unit (different counts, shifted blocks)
    k_max = 40
    sel = np.full((3, k_max), -1, np.int32)
    cnt = np.array([40, 7, 0], np.int32)
    sel[0, :40] = np.arange(40) * 16
    sel[1, :7] = np.array([8, 64, 72, 200, 504, 512, 992])
    out, lse = orc.attention_units(blobs, q, sel, cnt, scale)
    for u in range(3):
        o, l = orc.attention(blobs[u], q[u], sel[u, :cnt[u]], scale)
        np.testing.assert_array_equal(out[u], o)
        np.testing.assert_array_equal(lse[u], l)
    assert np.all(out[2] == 0) and np.all(np.isneginf(lse[2]))


# ----------------------------------------------------------------------------- P14: rotation fold (NEXT-3)

def test_P14_rotation_fold_is_mathematically_equivalent():
    """folding the rotation into the query (and the inverse into the output) "is mathematically
    equivalent" to attention in the original space.  Pinned three ways, none of which repeats the oracle's loops:
    (i) with a SIGNED PERMUTATION R (orthogonal, and K R^T, q R^T are exact in bf16) and no compression, attention on the
    rotated cache with the folded query, rotated back, equals numpy dense attention on the ORIGINAL K, V, q to 1e-12;
    (ii) rotate_query equals the numpy matmul q R^T to bf16 rounding, and exactly for the permutation; a transposed R
    fails both; (iii) rotate_output equals numpy o @ R."""
    rng = np.random.default_rng(31)
    D, N, G = 128, 96, 4
    K, V, q = small_unit(seed=9, N=N, D=D, G=G)
    perm_k, perm_v = rng.permutation(D), rng.permutation(D)
    sgn_k, sgn_v = rng.choice([-1.0, 1.0], D), rng.choice([-1.0, 1.0], D)
    Rk = np.zeros((D, D), np.float32); Rk[np.arange(D), perm_k] = sgn_k   # K'[:, i] = sgn_k[i] * K[:, perm_k[i]]
    Rv = np.zeros((D, D), np.float32); Rv[np.arange(D), perm_v] = sgn_v
    f = brute.bf16_to_f64
    Kp = synth.f32_to_bf16_bits((f(K) @ Rk.T.astype(np.float64)).astype(np.float32))  # exact: one nonzero per column
    Vp = synth.f32_to_bf16_bits((f(V) @ Rv.T.astype(np.float64)).astype(np.float32))
    assert np.array_equal(f(Kp), f(K) @ Rk.T) and np.array_equal(f(Vp), f(V) @ Rv.T)
    qp = orc.rotate_query(q, Rk)
    np.testing.assert_array_equal(f(qp), f(q) @ Rk.T.astype(np.float64))                 # (ii) exact for a permutation
    assert not np.array_equal(f(orc.rotate_query(q, Rk.T.copy())), f(q) @ Rk.T)          # a transposed operand is caught
    S = (N + 63) // 64
    blob = orc.compress_unit(Kp, Vp, 64, orc.uniform_strategy(S, D, D))
    ft, nt = orc.blob_blocks(blob)
    scale = 1.0 / math.sqrt(D)
    o_rot, lse_rot = orc.attention(blob, qp, ft, scale)
    o_back = orc.rotate_output(o_rot, Rv)
    o_ref, lse_ref = brute.dense_attention(f(q), f(K), f(V), scale)
    np.testing.assert_allclose(o_back, o_ref, rtol=0, atol=1e-12)                        # (i)
    np.testing.assert_allclose(lse_rot, lse_ref, rtol=0, atol=1e-12)
    # a general orthogonal matrix: bf16 rounding of q' only; rotate_output against numpy
    Q, _ = np.linalg.qr(rng.standard_normal((D, D)))
    Q = Q.astype(np.float32)
    qr = f(orc.rotate_query(q, Q))
    exact = f(q) @ Q.T.astype(np.float64)
    assert np.abs(qr - exact).max() <= 2.0 ** -8 * np.abs(exact).max() + 1e-6           # one bf16 rounding + fp32 sums
    o = rng.standard_normal((G, D))
    np.testing.assert_allclose(orc.rotate_output(o, Q), o @ Q.astype(np.float64), rtol=0, atol=1e-13)
