"""CPU pins of the base-policy oracle (block scores + importance-first top-k list, R10)."""
import numpy as np
import torch

from oracle import art_oracle as ao

N = ao.BLOCK_TOKENS


def _problem(seed, B=2, Hkv=2, G=2, d=16, lens=(300, 130), layout=ao.LAYOUT_HND):
    rng = np.random.default_rng(seed)
    nbs = [-(-L // N) for L in lens]
    pages = sum(nbs)
    perm = rng.permutation(pages)
    maxb = max(nbs)
    table = np.zeros((B, maxb), dtype=np.int32)
    o = 0
    for b, nb in enumerate(nbs):
        table[b, :nb] = perm[o:o + nb]; o += nb
    shape = (pages, Hkv, N, d) if layout == ao.LAYOUT_HND else (pages, N, Hkv, d)
    k = rng.standard_normal(shape)
    q = rng.standard_normal((B, Hkv * G, d))
    return q, k, table, np.array(lens)


def test_scores_match_a_library_contraction_both_layouts():
    for layout in (ao.LAYOUT_HND, ao.LAYOUT_NHD):
        q, k, table, lens = _problem(1, layout=layout)
        s = ao.block_scores_oracle(q, k, table, lens, num_kv_heads=2, layout=layout)
        B, Hq, d = q.shape
        for b in range(B):
            L = int(lens[b]); nb = -(-L // N)
            for g in range(2):
                kk = k[table[b, :nb], g] if layout == ao.LAYOUT_HND else k[table[b, :nb], :, g]   # [nb, 64, d]
                valid = (np.arange(nb * N).reshape(nb, N) < L)
                qg = torch.tensor(q[b, 2 * g:2 * g + 2]).sum(0)                                  # library third opinion
                ref = (torch.einsum("d,bnd->bn", qg, torch.tensor(kk)) * torch.tensor(valid)).sum(-1) / (2 * torch.tensor(valid).sum(-1))
                np.testing.assert_allclose(s[b, g, :nb], ref.numpy(), rtol=1e-12, atol=1e-12)
                assert np.isneginf(s[b, g, nb:]).all()


def test_scores_closed_form_constant_keys():
    """Every key of block j equals c_j * e_0  =>  score_j = c_j * mean_h q_h[0], whatever the partial tail."""
    B, Hkv, G, d = 1, 1, 4, 8
    L = 3 * N + 5
    nb = 4
    c = np.array([0.5, -2.0, 3.0, 7.0])
    k = np.zeros((nb, Hkv, N, d)); k[:, 0, :, 0] = c[:, None]
    q = np.random.default_rng(0).standard_normal((B, Hkv * G, d))
    s = ao.block_scores_oracle(q, k, np.arange(nb, dtype=np.int32)[None], [L], num_kv_heads=Hkv)
    np.testing.assert_allclose(s[0, 0], c * q[0, :, 0].mean(), rtol=1e-13)


def test_topk_order_ties_and_counts():
    scores = np.full((1, 2, 6), -np.inf)
    scores[0, 0, :5] = [1.0, 3.0, 3.0, -1.0, 2.0]          # tie between blocks 1 and 2 -> lower index first
    scores[0, 1, :5] = [0.0, 0.0, 0.0, 0.0, 0.0]           # all equal -> ascending index
    lists, counts = ao.topk_blocks_oracle(scores, [5 * N - 3], 3)
    assert lists[0, 0].tolist() == [1, 2, 4] and lists[0, 1].tolist() == [0, 1, 2] and counts.tolist() == [[3, 3]]
    lists, counts = ao.topk_blocks_oracle(scores, [5 * N - 3], 9)   # k larger than the number of blocks
    assert counts.tolist() == [[5, 5]] and lists[0, 0, :5].tolist() == [1, 2, 4, 0, 3] and (lists[0, 0, 5:] == -1).all()
    lists, counts = ao.topk_blocks_oracle(scores, [0], 3)           # empty sequence
    assert counts.tolist() == [[0, 0]] and (lists == -1).all()


def test_topk_agrees_with_library_topk_without_ties():
    rng = np.random.default_rng(3)
    scores = rng.standard_normal((2, 3, 40))
    lists, counts = ao.topk_blocks_oracle(scores, [40 * N, 40 * N], 7)
    ref = torch.topk(torch.tensor(scores), 7, dim=-1).indices.numpy()
    assert np.array_equal(lists, ref) and (counts == 7).all()
