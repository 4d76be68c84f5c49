"""CPU: the C-ABI library loads, exports every symbol include/art_decode.h declares, and validates
its arguments before touching CUDA (no compute calls without a GPU)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def art():
    import runpy                      # by path: the package refuses to import until the library exists
    runpy.run_path(os.path.join(ROOT, "paper_2606_00024_b200", "build.py"))["build"]()
    import paper_2606_00024_b200 as a
    return a


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "art_decode.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(art_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(art):
    lib = art.load_library()
    syms = declared_symbols()
    assert {"art_decode_attention", "art_decode_attention_off", "art_decode_attention_host", "art_topk_blocks",
            "art_workspace_bytes", "art_query_split", "art_query_clusters", "art_status_string", "art_version",
            "art_hbm_read_probe", "art_decode_attention_off_static", "art_static_scratch_bytes",
            "art_static_scratch_needed"} <= set(syms)
    for s in syms:
        assert hasattr(lib, s), s
    assert art.art_version() == 122
    assert "NULL" in art.art_status_string(-1) and art.art_status_string(0) == "ok"


def test_struct_layout_matches_header(art):
    assert C.sizeof(art.ArtDesc) == 80 and art.ArtDesc.q_len.offset == 56 and art.ArtDesc.eligible_counts.offset == 64
    assert C.sizeof(art.ArtThresholds) == 16


def _call_off(art, desc, q=16, k=32, v=48, bt=64, el=None, sl=80, out=96, stop=112):
    lib = art.load_library()
    vp = lambda x: None if x is None else C.c_void_p(x)
    return lib.art_decode_attention_off(C.byref(desc), vp(q), vp(k), vp(v), vp(bt), vp(el), vp(sl), vp(out), vp(stop),
                                        None, 0, None)


def good_desc(art, **kw):
    d = dict(batch=2, num_q_heads=8, num_kv_heads=2, head_dim=128, block_tokens=64, dtype=art.ART_DTYPE_BF16,
             kv_layout=0, policy=0, max_blocks_per_seq=4)
    d.update(kw)
    return art.ArtDesc(**d)


def test_argument_validation_happens_before_cuda(art):
    """Fake (never dereferenced) pointers: every error below is decided on the host."""
    assert _call_off(art, good_desc(art), q=None) == -1                      # ART_ERR_NULL
    assert _call_off(art, good_desc(art, num_q_heads=7)) == -2               # Hq % Hkv
    assert _call_off(art, good_desc(art, num_q_heads=32, num_kv_heads=2)) == -2   # G = 16 unsupported (1..8 are)
    assert _call_off(art, good_desc(art, block_tokens=32)) == -2
    assert _call_off(art, good_desc(art, head_dim=96)) == -2
    assert _call_off(art, good_desc(art, head_dim=64)) == -3                 # bf16 d=64 not built
    assert _call_off(art, good_desc(art, dtype=5)) == -3
    assert _call_off(art, good_desc(art, policy=2)) == -1                    # LIST without a list
    assert _call_off(art, good_desc(art, policy=1, sink_tokens=-1)) == -2
    assert _call_off(art, good_desc(art, split=17)) == -2                    # cluster size > 16
    assert _call_off(art, good_desc(art, split=-18)) == -2                   # persistent clusters of at most 16 CTAs
    assert _call_off(art, good_desc(art, max_blocks_per_seq=1 << 24)) == -2   # a step number is 24 bits
    assert _call_off(art, good_desc(art, dtype=art.ART_DTYPE_F32, head_dim=64, split=-1)) == -3   # dynamic: bf16 only
    assert _call_off(art, good_desc(art, dtype=art.ART_DTYPE_F32, head_dim=64, split=3)) == -2   # fp32 path: power of two
    assert _call_off(art, good_desc(art), k=33) == -4                        # ART_ERR_ALIGN
    # multi-token queries (q_len, reading R15): m * G <= 8, a cluster schedule
    assert _call_off(art, good_desc(art, q_len=3)) == -2                     # 3 * 4 rows
    assert _call_off(art, good_desc(art, q_len=-1)) == -2
    assert _call_off(art, good_desc(art, q_len=3, dtype=art.ART_DTYPE_F32, head_dim=64, num_q_heads=6)) == -2   # 3 * 3 rows
    lib = art.load_library()
    th = art.ArtThresholds(tau=1e-5, phi=1e-3, patience=0, probe_dim=32)
    vp = C.c_void_p
    rc = lib.art_decode_attention(C.byref(good_desc(art)), vp(16), vp(32), vp(48), vp(64), None, vp(80), C.byref(th),
                                  vp(96), vp(112), None, 0, None)
    assert rc == -2                                                          # patience < 1
    th = art.ArtThresholds(tau=float("nan"), phi=1e-3, patience=5, probe_dim=32)
    rc = lib.art_decode_attention(C.byref(good_desc(art)), vp(16), vp(32), vp(48), vp(64), None, vp(80), C.byref(th),
                                  vp(96), vp(112), None, 0, None)
    assert rc == -2                                                          # NaN threshold
    th = art.ArtThresholds(tau=1e-5, phi=1e-3, patience=5, probe_dim=48)
    rc = lib.art_decode_attention(C.byref(good_desc(art)), vp(16), vp(32), vp(48), vp(64), None, vp(80), C.byref(th),
                                  vp(96), vp(112), None, 0, None)
    assert rc == -2


def test_no_gpu_means_loud_failure_not_fallback(art):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    rc = _call_off(art, good_desc(art))
    assert rc in (-6, -7)                                                    # ART_ERR_ARCH / ART_ERR_CUDA
    assert art.art_workspace_bytes(good_desc(art)) > 0


def test_static_scratch_sizes_and_limit_need_no_device(art):
    """art_decode_attention_off_static rejects what does not fit its built-in array before any CUDA call."""
    import torch
    from workloads import generators as gen
    assert art.art_static_scratch_bytes() == 32 << 20
    w = gen.config(1, scale=1 / 8, batch=2)
    d = art.make_desc(w)
    assert art.art_static_scratch_needed(d) == 2 * 8 * 16 * 4 * 130 * 4
    big = art.ArtDesc(batch=128, num_q_heads=32, num_kv_heads=8, head_dim=128, block_tokens=64, dtype=art.ART_DTYPE_BF16,
                      max_blocks_per_seq=8)
    assert art.art_static_scratch_needed(big) > art.art_static_scratch_bytes()
    lib = art.load_library()
    x = torch.zeros(64)                                             # never dereferenced: the call fails on the size
    rc = lib.art_decode_attention_off_static(C.byref(big), x.data_ptr(), x.data_ptr(), x.data_ptr(), x.data_ptr(), None,
                                             x.data_ptr(), x.data_ptr(), x.data_ptr(), None)
    assert rc == -8 and "scratch" in art.art_status_string(rc)
    bad = art.ArtDesc(batch=1, num_q_heads=4, num_kv_heads=1, head_dim=64, block_tokens=64, dtype=art.ART_DTYPE_F32)
    assert lib.art_decode_attention_off_static(C.byref(bad), *([x.data_ptr()] * 4), None, *([x.data_ptr()] * 3), None) == -3
