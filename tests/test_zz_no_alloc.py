"""GPU: art_decode_attention_off_static, the entry point that allocates nothing (its scratch is a file-scope device
array inside the library, include/art_decode.h).  Collected last on purpose (file name): the suite runs with
pytest -x, and a failure here must not hide the tests before it.

The new entry point against the existing ones (art_decode_attention_off on static clusters and on persistent clusters
with a caller workspace) within the tolerance the other tests use for two schedules of the same computation (1e-5 of
the largest output, test_gpu_parity.py::test_dynamic_scheduler_stop_blocks_equal_cluster_kernel) and against the
oracle (OUT_TOL), on two calls in a row, with a different problem in between so that the shared array holds another
call's contents when the second call starts."""
import pytest
import torch

from workloads import generators as gen
from parity import compare, OUT_TOL

pytestmark = pytest.mark.gpu


def art():
    import paper_2606_00024_b200 as a
    return a


def run_static(a, w):
    out = torch.empty(tuple(w.q.shape), dtype=torch.float32, device=w.q.device)
    stop = torch.empty((w.batch, w.num_kv_heads), dtype=torch.int32, device=w.q.device)
    a.art_decode_attention_off_static(a.make_desc(w), w.q, w.k_cache, w.v_cache, w.block_table, w.eligible_blocks,
                                      w.seq_lens, out, stop)
    torch.cuda.synchronize()
    return out, stop


def close(x, ref):
    return float((x - ref).abs().max()) <= 1e-5 * float(ref.abs().max())


@pytest.mark.parametrize("index,kw", [(1, dict(scale=1 / 8, batch=4)), (2, dict(scale=1 / 8, batch=4)),
                                      (3, dict(scale=1 / 2, batch=24)), (4, dict(scale=1 / 32, batch=2))])
def test_two_calls_in_a_row_equal_the_existing_paths(index, kw):
    a = art()
    w = gen.config(index, **kw)
    wc = w.to("cuda")
    other = gen.make_workload("other", seed=77, batch=5, num_q_heads=16, num_kv_heads=2, head_dim=128,
                              seq_lens=[700, 64, 1, 2000, 333], dtype=torch.bfloat16).to("cuda")
    assert 0 < a.art_static_scratch_needed(a.make_desc(wc)) <= a.art_static_scratch_bytes()
    ref_o, ref_s, _ = a.run_workload(wc, art=False)                                  # static clusters (library default)
    pc_o, pc_s, _ = a.run_workload(wc, art=False, split=a.ART_SPLIT_DYNAMIC)        # persistent, caller workspace
    torch.cuda.synchronize()
    o1, s1 = run_static(a, wc)
    oo, so = run_static(a, other)                                                    # leaves its partial states in the array
    o2, s2 = run_static(a, wc)
    for o, s in ((o1, s1), (o2, s2)):
        assert torch.equal(s, ref_s) and torch.equal(s, pc_s)
        assert close(o, ref_o) and close(o, pc_o)
        rep = compare(w, o, s, art=False)
        assert rep.ok(OUT_TOL[w.dtype]), rep.summary()
    ref_oo, ref_so, _ = a.run_workload(other, art=False)
    assert torch.equal(so, ref_so) and close(oo, ref_oo)


def test_multi_token_and_empty_sequences():
    a = art()
    w = gen.make_workload("e", seed=3, batch=6, num_q_heads=4, num_kv_heads=2, head_dim=128,
                          seq_lens=[0, 1, 63, 64, 65, 1300], dtype=torch.bfloat16)
    for wl in (w, gen.with_query_tokens(w, 3, seed=3)):
        wc = wl.to("cuda")
        ref_o, ref_s, _ = a.run_workload(wc, art=False)
        for _ in range(2):
            o, s = run_static(a, wc)
            assert torch.equal(s, ref_s) and close(o, ref_o)
            assert (o[0] == 0).all() and int(s[0].abs().sum()) == 0


def test_limit_and_argument_errors():
    a = art()
    big = gen.config(3, scale=1 / 16).to("cuda")                                     # 1024 groups of 4 rows: 34 MB of partial states
    d = a.make_desc(big)
    assert a.art_static_scratch_needed(d) > a.art_static_scratch_bytes()
    out = torch.full(tuple(big.q.shape), 7.0, dtype=torch.float32, device="cuda")
    stop = torch.full((big.batch, big.num_kv_heads), -5, dtype=torch.int32, device="cuda")
    with pytest.raises(a.ArtError) as e:
        a.art_decode_attention_off_static(d, big.q, big.k_cache, big.v_cache, big.block_table, big.eligible_blocks,
                                          big.seq_lens, out, stop)
    assert e.value.status == -8 and "scratch" in str(e.value)
    torch.cuda.synchronize()
    assert (out == 7.0).all() and (stop == -5).all()                                 # rejected before anything was launched
    a.run_workload(big, art=False)                                                   # the existing path takes it (caller workspace)
    w = gen.config(1, scale=1 / 8, batch=2).to("cuda")
    o = torch.empty(tuple(w.q.shape), dtype=torch.float32, device="cuda")
    s = torch.empty((w.batch, w.num_kv_heads), dtype=torch.int32, device="cuda")
    with pytest.raises(a.ArtError) as e:                                             # a static cluster size: no scratch involved
        a.art_decode_attention_off_static(a.make_desc(w, split=2), w.q, w.k_cache, w.v_cache, w.block_table,
                                          w.eligible_blocks, w.seq_lens, o, s)
    assert e.value.status == -2
    f = gen.config(0).to("cuda")                                                     # fp32: the CUDA-core kernel has no scratch
    o = torch.empty(tuple(f.q.shape), dtype=torch.float32, device="cuda")
    s = torch.empty((f.batch, f.num_kv_heads), dtype=torch.int32, device="cuda")
    with pytest.raises(a.ArtError) as e:
        a.art_decode_attention_off_static(a.make_desc(f), f.q, f.k_cache, f.v_cache, f.block_table, f.eligible_blocks,
                                          f.seq_lens, o, s)
    assert e.value.status == -3


def test_the_library_does_not_allocate():
    """Device memory in use does not move across calls of the new entry point (cudaMemGetInfo; outputs allocated before)."""
    a = art()
    w = gen.config(1, scale=1 / 8, batch=4).to("cuda")
    out = torch.empty(tuple(w.q.shape), dtype=torch.float32, device="cuda")
    stop = torch.empty((w.batch, w.num_kv_heads), dtype=torch.int32, device="cuda")
    d = a.make_desc(w)
    args = (d, w.q, w.k_cache, w.v_cache, w.block_table, w.eligible_blocks, w.seq_lens, out, stop)
    a.art_decode_attention_off_static(*args)                                         # first call: module load, symbol address
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        a.art_decode_attention_off_static(*args)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
