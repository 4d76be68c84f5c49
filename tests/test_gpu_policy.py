"""-m gpu: the base-policy kernels (block scores + importance-first top-k list, R10) through the
C ABI against the fp64 oracle.  Floating point decides an ordering here: positions are compared exactly wherever
the oracle's scores are separated by more than the fp32 tolerance, and bit-exactly on constructed ties."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from workloads import generators as gen
from helpers import np64, run_oracle
from oracle import art_oracle as ao
from parity import compare, OUT_TOL

pytestmark = pytest.mark.gpu


def art():
    import paper_2606_00024_b200 as a
    return a


def gpu_lists(w, top_k):
    a = art()
    wc = w.to("cuda")
    maxb = int(w.block_table.shape[1])
    scores = torch.full((w.batch, w.num_kv_heads, maxb), float("nan"), dtype=torch.float32, device="cuda")
    lists = torch.full((w.batch, w.num_kv_heads, max(top_k, 1)), -7, dtype=torch.int32, device="cuda")
    counts = torch.full((w.batch, w.num_kv_heads), -7, dtype=torch.int32, device="cuda")
    desc = a.make_desc(wc)
    desc.max_eligible = max(top_k, 1)
    a.art_topk_blocks(desc, wc.q, wc.k_cache, wc.block_table, wc.seq_lens, top_k, scores, lists, counts)
    torch.cuda.synchronize()
    return scores.cpu().numpy(), lists.cpu().numpy(), counts.cpu().numpy()


def check_policy(w, top_k):
    s_ref = ao.block_scores_oracle(np64(w.q), np64(w.k_cache), w.block_table.numpy(), w.seq_lens.numpy(),
                                   num_kv_heads=w.num_kv_heads, layout=w.layout)
    l_ref, c_ref = ao.topk_blocks_oracle(s_ref, w.seq_lens.numpy(), top_k)
    s, l, c = gpu_lists(w, top_k)
    assert np.array_equal(c, c_ref)
    fin = np.isfinite(s_ref)
    assert np.array_equal(np.isneginf(s), ~fin)                       # -inf exactly on the non-candidates
    tol = 2e-5 * max(1.0, float(np.abs(s_ref[fin]).max())) if fin.any() else 0.0
    assert np.abs(s[fin] - s_ref[fin]).max(initial=0.0) <= tol        # fp32 accumulation of 64 x d x G products
    for b in range(w.batch):
        for g in range(w.num_kv_heads):
            k = int(c[b, g]); got = l[b, g, :k]; ref = l_ref[b, g, :k]
            assert len(set(got.tolist())) == k and (got >= 0).all() and (got < -(-int(w.seq_lens[b]) // 64)).all()
            sorted_ref = s_ref[b, g, ref]
            assert np.abs(s_ref[b, g, got] - sorted_ref).max(initial=0.0) <= 2 * tol   # right scores at every rank
            # ranks whose oracle score is separated from both neighbours (and from the first one left out): exact
            allsorted = np.sort(s_ref[b, g][np.isfinite(s_ref[b, g])])[::-1]
            for i in range(k):
                lo = allsorted[i] - allsorted[i + 1] if i + 1 < len(allsorted) else np.inf
                hi = allsorted[i - 1] - allsorted[i] if i > 0 else np.inf
                if lo > 4 * tol and hi > 4 * tol:
                    assert got[i] == ref[i]
    return s, l, c


@pytest.mark.parametrize("G", [1, 2, 3, 4, 6, 8])
@pytest.mark.parametrize("dtype,layout", [(torch.bfloat16, gen.LAYOUT_HND), (torch.bfloat16, gen.LAYOUT_NHD),
                                          (torch.float32, gen.LAYOUT_HND)])
def test_scores_and_lists_match_oracle(G, dtype, layout):
    d = 64 if dtype == torch.float32 else 128
    w = gen.make_workload("pol", seed=31 + G, batch=5, num_q_heads=2 * G, num_kv_heads=2, head_dim=d,
                          seq_lens=[0, 1, 700, 64, 2049], dtype=dtype, layout=layout, planted_frac=0.01)
    check_policy(w, 7)
    check_policy(w, 0)
    check_policy(w, 40)                                               # more than some sequences have blocks


def test_ties_go_to_the_lower_block_index_bit_exactly():
    w = gen.make_workload("tie", seed=5, batch=1, num_q_heads=4, num_kv_heads=1, head_dim=128, seq_lens=[64 * 12])
    pages = w.block_table[0].long()
    for blk in (3, 7, 9):                                             # identical tiles => identical fp32 sums
        w.k_cache[pages[blk]] = w.k_cache[pages[1]]
    s_ref = ao.block_scores_oracle(np64(w.q), np64(w.k_cache), w.block_table.numpy(), w.seq_lens.numpy(), num_kv_heads=1)
    l_ref, _ = ao.topk_blocks_oracle(s_ref, w.seq_lens.numpy(), 12)
    s, l, c = gpu_lists(w, 12)
    assert s[0, 0, 1] == s[0, 0, 3] == s[0, 0, 7] == s[0, 0, 9]
    pos = {int(blk): i for i, blk in enumerate(l[0, 0])}
    assert pos[1] + 1 == pos[3] and pos[3] + 1 == pos[7] and pos[7] + 1 == pos[9]
    assert sorted(l[0, 0].tolist()) == list(range(12)) and int(c[0, 0]) == 12


def test_device_built_list_feeds_the_attention_kernel():
    """A1's input built on the device: GPU list -> art_decode_attention (policy LIST) == oracle on that same list."""
    a = art()
    w = gen.config(2, scale=1 / 8, batch=2, recency_decay=(0.2, 1.0))
    k = int(w.eligible_blocks.shape[2])
    _, l, c = gpu_lists(w, k)
    w2 = replace(w, eligible_blocks=torch.tensor(l, dtype=torch.int32), eligible_counts=torch.tensor(c, dtype=torch.int32))
    out, stop, _ = a.run_workload(w2.to("cuda"), tau=1e-3)
    rep = compare(w2, out, stop, art=True, oracle_over={"tau": float(np.float32(1e-3))})
    assert rep.ok(OUT_TOL[w.dtype]), rep.summary()


def test_full_size_config2_scores_sampled():
    a = art()
    w = gen.config(2, device="cuda")
    maxb = int(w.block_table.shape[1]); k = int(w.eligible_blocks.shape[2])
    scores = torch.empty((w.batch, w.num_kv_heads, maxb), dtype=torch.float32, device="cuda")
    lists = torch.empty((w.batch, w.num_kv_heads, k), dtype=torch.int32, device="cuda")
    counts = torch.empty((w.batch, w.num_kv_heads), dtype=torch.int32, device="cuda")
    a.art_topk_blocks(a.make_desc(w), w.q, w.k_cache, w.block_table, w.seq_lens, k, scores, lists, counts)
    torch.cuda.synchronize()
    assert (counts == k).all()
    # the generator's own list (torch, fp32) must agree wherever scores are not within rounding of each other
    agree = (lists == w.eligible_blocks).float().mean().item()
    assert agree > 0.98, agree
    from helpers import extract_groups
    for (b, g) in [(0, 0), (7, 3), (15, 7)]:
        mini = extract_groups(w, [(b, g)])
        s_ref = ao.block_scores_oracle(np64(mini.q), np64(mini.k_cache), mini.block_table.numpy(), mini.seq_lens.numpy(), num_kv_heads=1)
        got = scores[b, g].cpu().numpy()
        assert np.abs(got - s_ref[0, 0]).max() <= 2e-5 * max(1.0, np.abs(s_ref).max())
    del w
    torch.cuda.empty_cache()


@pytest.mark.parametrize("m,G", [(2, 4), (4, 2), (8, 1), (3, 2)])
def test_multi_token_queries_are_scored_by_their_last_token(m, G):
    """Reading R15: with q_len = m the policy's eligible set and order are the group's, computed as for the LAST query
    token.  art_topk_blocks on q [B, m, Hq, d] == the oracle on q[:, m - 1] == art_topk_blocks on that token alone
    (bit for bit), and the device-built list feeds the multi-token attention call."""
    a = art()
    base = gen.make_workload("pm", seed=77 + m, batch=2, num_q_heads=G * 2, num_kv_heads=2, head_dim=128,
                             seq_lens=[1500, 777], planted_frac=0.01, sink_plant=4, recency_decay=(0.2, 1.0))
    w = gen.with_query_tokens(base, m, seed=300 + m)
    last = replace(w, q=w.q[:, m - 1].contiguous())
    top_k = 9
    s_ref = ao.block_scores_oracle(np64(last.q), np64(w.k_cache), w.block_table.numpy(), w.seq_lens.numpy(),
                                   num_kv_heads=w.num_kv_heads, layout=w.layout)
    l_ref, c_ref = ao.topk_blocks_oracle(s_ref, w.seq_lens.numpy(), top_k)
    s_m, l_m, c_m = gpu_lists(w, top_k)
    s_1, l_1, c_1 = gpu_lists(last, top_k)
    assert np.array_equal(s_m, s_1) and np.array_equal(c_m, c_1)
    for b in range(w.batch):
        for g in range(w.num_kv_heads):
            assert np.array_equal(l_m[b, g, :c_m[b, g]], l_1[b, g, :c_1[b, g]])
    fin = np.isfinite(s_ref)
    assert np.array_equal(c_m, c_ref) and np.abs(s_m[fin] - s_ref[fin]).max() <= 2e-5 * max(1.0, float(np.abs(s_ref[fin]).max()))
    # the device-built list through the multi-token attention kernel, against the oracle on the same list
    wl = replace(w, policy=gen.POLICY_LIST, eligible_blocks=torch.from_numpy(l_m.astype(np.int32)),
                 eligible_counts=torch.from_numpy(c_m.astype(np.int32)))
    wc = wl.to("cuda")
    for art_on in (True, False):
        out, stop, _ = a.run_workload(wc, art=art_on, **({"tau": 1e-3} if art_on else {}))
        torch.cuda.synchronize()
        over = {"tau": float(np.float32(1e-3))} if art_on else {}
        rep = compare(wl, out, stop, art=art_on, oracle_over=over)
        assert rep.ok(OUT_TOL[wl.dtype]), rep.summary()


def test_error_codes():
    a = art()
    w = gen.make_workload("e", seed=1, batch=1, num_q_heads=4, num_kv_heads=1, head_dim=128, seq_lens=[300]).to("cuda")
    desc = a.make_desc(w); desc.max_eligible = 2
    sc = torch.empty((1, 1, 5), device="cuda"); li = torch.empty((1, 1, 2), dtype=torch.int32, device="cuda")
    co = torch.empty((1, 1), dtype=torch.int32, device="cuda")
    with pytest.raises(a.ArtError) as e:
        a.art_topk_blocks(desc, w.q, w.k_cache, w.block_table, w.seq_lens, 3, sc, li, co)      # top_k > row stride
    assert e.value.status == -2
    with pytest.raises(a.ArtError) as e:
        a.art_topk_blocks(desc, w.q, w.k_cache, w.block_table, w.seq_lens, 2, None, li, co)
    assert e.value.status == -1
