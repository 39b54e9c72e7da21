"""mkv_topk_static: the budgeted top-k (step 2b) for callers that cannot allocate device memory.

Some users of libmkv cannot call cudaMalloc where they need a selection -- a decode loop inside a serving engine whose
pool allocator owns the whole GPU, a plug-in that only receives device pointers from its host program -- so they can
neither create an mkv_cache (mkv_cache_create allocates) nor bring scratch of their own.  mkv_topk_static takes their
block scores and writes the selection; its only scratch, the candidate lists of the two-stage selection, is a 4-MB
array compiled into the library (MKV_TOPK_STATIC_MAX_CANDIDATES entries) that all calls on a device share.

What is checked here: on the same scores the entry point returns, bit for bit, what the existing path (mkv_select,
whose scratch belongs to the cache) returns -- selections are integer work, so the tolerance is equality -- on two calls
in a row that reuse the shared array with different layouts (so the second call finds the first one's candidates lying
around), for units long enough to need the scratch and for short ones that do not; and that a request beyond the
array's size is refused with a message instead of being run.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It creates everything it uses, so it passes alone in a fresh process as well as after the other files.
"""
import numpy as np
import pytest

import __graft_entry__  # noqa: F401  (builds the library if needed)


def _existing_path(mkv, torch, cache, q_d, budget, reduce, Bt, Hkv, B, N):
    """mkv_select on the cache: the selection and the scores it was made from"""
    nblk = (N + B - 1) // B
    k_max = max(1, min(budget // B + 1, nblk))
    sel = torch.full((Bt, Hkv, k_max), -7, dtype=torch.int32, device=q_d.device)
    cnt = torch.full((Bt, Hkv), -7, dtype=torch.int32, device=q_d.device)
    scores = torch.zeros((Bt, Hkv, cache.score_stride), dtype=torch.float32, device=q_d.device)
    cache.select(0, q_d, budget, sel, cnt, reduce=reduce, scores=scores)
    return sel, cnt, scores, k_max


def _run_pair(N, B, budgets):
    """Two selections on one cache by the existing path, then the same two through mkv_topk_static back to back on one
    stream (no host synchronisation between them: the second call starts from the first one's scratch contents)."""
    import torch
    from paper_2607_00760_b200 import binding as mkv, synth
    from gpu_util import to_dev

    dev = torch.device("cuda:0")
    Bt, Hkv, Hq, L = 1, 2, 8, 64
    K, V, q = synth.make_inputs_np(Bt, Hkv, Hq, N, 128, L, seed=11)
    q2 = synth.make_inputs_np(Bt, Hkv, Hq, 64, 128, L, seed=12)[2]
    cache = mkv.Cache(1, Bt, Hkv, Hq, 128, N, L, token_block=B)
    try:
        S = (N + L - 1) // L
        strat = np.zeros((Bt, Hkv, S, 4), np.uint8)
        strat[:] = (38, 38, 1, B)
        strat[:, :, ::7] = (128, 128, 1, B)  # a few dense segments among the sparse ones
        cache.compress_segment(0, to_dev(K, dev), to_dev(V, dev), torch.from_numpy(strat).to(dev))
        cache.status()
        ref = [_existing_path(mkv, torch, cache, to_dev(qq, dev), budget, reduce, Bt, Hkv, B, N)
               for qq, budget, reduce in ((q, budgets[0], 0), (q2, budgets[1], 1))]
        torch.cuda.synchronize()

        n_tokens = torch.full((Bt * Hkv,), N, dtype=torch.int32, device=dev)
        got = []
        for (sel, cnt, scores, k_max), budget in zip(ref, budgets):
            sel2 = torch.full((Bt * Hkv, k_max), -9, dtype=torch.int32, device=dev)
            cnt2 = torch.full((Bt * Hkv,), -9, dtype=torch.int32, device=dev)
            mkv.mkv_topk_static(0, scores.view(Bt * Hkv, -1), n_tokens, B, budget, sel2, cnt2)
            got.append((sel2, cnt2))
        torch.cuda.synchronize()
        for (sel, cnt, scores, k_max), (sel2, cnt2), budget in zip(ref, got, budgets):
            c = cnt.cpu().numpy().reshape(-1)
            assert c.min() > 0, "the existing path selected nothing: the comparison would be empty"
            assert np.array_equal(cnt2.cpu().numpy(), c), (budget, cnt2.cpu().numpy(), c)
            assert np.array_equal(sel2.cpu().numpy(), sel.cpu().numpy().reshape(Bt * Hkv, k_max)), budget
    finally:
        cache.free()


@pytest.mark.gpu
def test_static_scratch_topk_equals_select_on_long_units():
    """25 001 blocks of 4 tokens per unit = two slices: both stages run and the candidates go through the static array.
    The second call keeps fewer candidates per slice than the first, so its lists overlay the first call's."""
    _run_pair(N=100003, B=4, budgets=(4099, 1000))


@pytest.mark.gpu
def test_static_scratch_topk_equals_select_on_short_units():
    """units of at most 16 384 blocks take one stage and no scratch; same answer as mkv_select, ragged last block"""
    _run_pair(N=1003, B=8, budgets=(300, 8))


@pytest.mark.gpu
def test_static_scratch_topk_refuses_what_does_not_fit():
    """64 units x 8 slices x 4097 candidates is 4 x the array: MKV_E_ARG with the sizes in the message, nothing enqueued"""
    import torch
    from paper_2607_00760_b200 import binding as mkv

    dev = torch.device("cuda:0")
    n_units, stride, B, budget = 64, 8 * 16384, 8, 32768
    assert n_units * 8 * (budget // B + 1) > mkv.MKV_TOPK_STATIC_MAX_CANDIDATES
    scores = torch.zeros((n_units, stride), dtype=torch.float32, device=dev)
    n_tokens = torch.full((n_units,), stride * B, dtype=torch.int32, device=dev)
    sel = torch.full((n_units, budget // B + 1), -9, dtype=torch.int32, device=dev)
    cnt = torch.full((n_units,), -9, dtype=torch.int32, device=dev)
    with pytest.raises(mkv.MkvError) as ei:
        mkv.mkv_topk_static(0, scores, n_tokens, B, budget, sel, cnt)
    assert ei.value.code == mkv.MKV_E_ARG
    assert "MKV_TOPK_STATIC_MAX_CANDIDATES" in str(ei.value) and "4097" in str(ei.value)
    torch.cuda.synchronize()
    assert int(cnt.min()) == -9 and int(sel.max()) == -9, "a refused call must not touch its outputs"
    # the same units in calls of 8 fit (8 x 8 x 4097 entries) and run
    mkv.mkv_topk_static(0, scores[:8], n_tokens[:8], B, budget, sel[:8], cnt[:8])
    torch.cuda.synchronize()
    assert np.array_equal(cnt[:8].cpu().numpy(), np.full(8, budget // B, np.int32))
    # all scores equal: ties go to the lower index, so the first budget / B blocks in order
    assert np.array_equal(sel[0, :budget // B].cpu().numpy(), np.arange(budget // B, dtype=np.int32) * B)
    assert int(sel[0, budget // B]) == -1
