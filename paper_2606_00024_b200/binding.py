"""ctypes binding of include/art_decode.h: same names, argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI.  PyTorch is used for
device memory and streams.  If ``libart_decode.so`` is missing this module raises at import
time; it never falls back to another implementation.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_NAME = "libart_decode.so"

ART_PATIENCE_INF = 2**31 - 1
ART_SPLIT_DYNAMIC = -1


def art_split_persistent(cl: int) -> int:
    """ART_SPLIT_PERSISTENT(cl): art_desc_t.split for persistent clusters of cl CTAs."""
    return -1 - int(cl)

ART_DTYPE_F32, ART_DTYPE_BF16 = 0, 1
ART_LAYOUT_HND, ART_LAYOUT_NHD = 0, 1
ART_POLICY_DENSE, ART_POLICY_SINK_WINDOW, ART_POLICY_LIST = 0, 1, 2


class ArtDesc(C.Structure):
    """art_desc_t (include/art_decode.h)."""
    _fields_ = [
        ("batch", C.c_int32), ("num_q_heads", C.c_int32), ("num_kv_heads", C.c_int32),
        ("head_dim", C.c_int32), ("block_tokens", C.c_int32), ("dtype", C.c_int32),
        ("kv_layout", C.c_int32), ("policy", C.c_int32), ("max_blocks_per_seq", C.c_int32),
        ("sink_tokens", C.c_int32), ("window_tokens", C.c_int32), ("max_eligible", C.c_int32),
        ("sm_scale", C.c_float), ("split", C.c_int32), ("q_len", C.c_int32), ("num_pages", C.c_int32),
        ("eligible_counts", C.c_void_p), ("blocks_loaded", C.c_void_p),
    ]


class ArtThresholds(C.Structure):
    """art_thresholds_t (include/art_decode.h)."""
    _fields_ = [("tau", C.c_float), ("phi", C.c_float), ("patience", C.c_int32), ("probe_dim", C.c_int32)]


class ArtError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: status {status} ({art_status_string(status)})")


def lib_path() -> str:
    """The in-tree library; ART_LIB_PATH selects another build of it (the -DART_DEBUG one of tests/test_gpu_debug_build.py)."""
    return os.environ.get("ART_LIB_PATH") or os.path.join(_HERE, _LIB_NAME)


_lib = None


def load_library():
    """dlopen the in-tree library and declare the prototypes of every exported symbol."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise ImportError(f"{path} not built: run `python -m paper_2606_00024_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    lib = C.CDLL(path)
    vp, i32p, f32p = C.c_void_p, C.c_void_p, C.c_void_p
    lib.art_decode_attention.restype = C.c_int
    lib.art_decode_attention.argtypes = [C.POINTER(ArtDesc), vp, vp, vp, i32p, i32p, i32p,
                                         C.POINTER(ArtThresholds), f32p, i32p, vp, C.c_size_t, vp]
    lib.art_decode_attention_off.restype = C.c_int
    lib.art_decode_attention_off.argtypes = [C.POINTER(ArtDesc), vp, vp, vp, i32p, i32p, i32p,
                                             f32p, i32p, vp, C.c_size_t, vp]
    lib.art_decode_attention_off_static.restype = C.c_int
    lib.art_decode_attention_off_static.argtypes = [C.POINTER(ArtDesc), vp, vp, vp, i32p, i32p, i32p, f32p, i32p, vp]
    lib.art_static_scratch_bytes.restype = C.c_size_t
    lib.art_static_scratch_bytes.argtypes = []
    lib.art_static_scratch_needed.restype = C.c_size_t
    lib.art_static_scratch_needed.argtypes = [C.POINTER(ArtDesc)]
    lib.art_decode_attention_host.restype = C.c_int
    lib.art_decode_attention_host.argtypes = [C.POINTER(ArtDesc), vp, vp, vp, i32p, i32p, i32p,
                                              C.POINTER(ArtThresholds), f32p, i32p, vp, C.c_size_t, vp]
    lib.art_topk_blocks.restype = C.c_int
    lib.art_topk_blocks.argtypes = [C.POINTER(ArtDesc), vp, vp, i32p, i32p, C.c_int32, f32p, i32p, i32p, vp]
    lib.art_workspace_bytes.restype = C.c_size_t
    lib.art_workspace_bytes.argtypes = [C.POINTER(ArtDesc)]
    lib.art_query_split.restype = C.c_int
    lib.art_query_split.argtypes = [C.POINTER(ArtDesc), C.c_int]
    lib.art_query_clusters.restype = C.c_int
    lib.art_query_clusters.argtypes = [C.POINTER(ArtDesc), C.c_int]
    lib.art_hbm_read_probe.restype = C.c_int
    lib.art_hbm_read_probe.argtypes = [vp, C.c_size_t, vp]
    lib.art_status_string.restype = C.c_char_p
    lib.art_status_string.argtypes = [C.c_int]
    lib.art_version.restype = C.c_int
    lib.art_version.argtypes = []
    _lib = lib
    return lib


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def art_version() -> int:
    return load_library().art_version()


def art_status_string(status: int) -> str:
    return load_library().art_status_string(int(status)).decode()


def art_workspace_bytes(desc: ArtDesc) -> int:
    return int(load_library().art_workspace_bytes(C.byref(desc)))


def art_query_split(desc: ArtDesc, art_on=True) -> int:
    """Cluster size the library picks; art_on: False / True / 2 (full-output detector)."""
    return int(load_library().art_query_split(C.byref(desc), int(art_on)))


def art_query_clusters(desc: ArtDesc, art_on=True) -> int:
    return int(load_library().art_query_clusters(C.byref(desc), int(art_on)))


_ws_cache = {}


def _workspace_for(desc: ArtDesc, device) -> torch.Tensor:
    """Device scratch of art_workspace_bytes(desc), cached per device (grown on demand).  The library never
    allocates; the caller (here: the binding, with torch) owns the memory.  One scratch per device: calls on
    DIFFERENT streams that may overlap (dynamic scheduler, host entry point) must pass their own `workspace`."""
    need = max(art_workspace_bytes(desc), 256)
    key = (device.type, device.index)
    ws = _ws_cache.get(key)
    if ws is None or ws.numel() < need:
        ws = torch.empty(need, dtype=torch.uint8, device=device)
        _ws_cache[key] = ws
    return ws


def art_decode_attention(desc, q, k_cache, v_cache, block_table, eligible_blocks, seq_lens, thresholds,
                         out, stop_block, workspace=None, stream=None) -> None:
    """ART-on.  All tensors are CUDA tensors except desc/thresholds (ctypes structs)."""
    if workspace is None:
        workspace = _workspace_for(desc, q.device)
    ws_ptr, ws_bytes = (_ptr(workspace), workspace.numel() * workspace.element_size())
    rc = load_library().art_decode_attention(
        C.byref(desc), _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(block_table), _ptr(eligible_blocks),
        _ptr(seq_lens), C.byref(thresholds), _ptr(out), _ptr(stop_block), ws_ptr, ws_bytes, _stream_ptr(stream))
    if rc != 0:
        raise ArtError(rc, "art_decode_attention")


def art_decode_attention_off(desc, q, k_cache, v_cache, block_table, eligible_blocks, seq_lens,
                             out, stop_block, workspace=None, stream=None) -> None:
    """ART-off (same kernel, detector compiled out)."""
    if workspace is None:
        workspace = _workspace_for(desc, q.device)
    ws_ptr, ws_bytes = (_ptr(workspace), workspace.numel() * workspace.element_size())
    rc = load_library().art_decode_attention_off(
        C.byref(desc), _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(block_table), _ptr(eligible_blocks),
        _ptr(seq_lens), _ptr(out), _ptr(stop_block), ws_ptr, ws_bytes, _stream_ptr(stream))
    if rc != 0:
        raise ArtError(rc, "art_decode_attention_off")


def art_decode_attention_off_static(desc, q, k_cache, v_cache, block_table, eligible_blocks, seq_lens,
                                    out, stop_block, stream=None) -> None:
    """ART-off on persistent clusters with the library's built-in scratch array: no workspace, no allocation
    (include/art_decode.h).  Calls that overlap on the GPU race on that array."""
    rc = load_library().art_decode_attention_off_static(
        C.byref(desc), _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(block_table), _ptr(eligible_blocks),
        _ptr(seq_lens), _ptr(out), _ptr(stop_block), _stream_ptr(stream))
    if rc != 0:
        raise ArtError(rc, "art_decode_attention_off_static")


def art_static_scratch_bytes() -> int:
    return int(load_library().art_static_scratch_bytes())


def art_static_scratch_needed(desc: ArtDesc) -> int:
    return int(load_library().art_static_scratch_needed(C.byref(desc)))


def art_decode_attention_host(desc, q_host, k_cache, v_cache, block_table_host, eligible_blocks_host,
                              seq_lens_host, thresholds, out_host, stop_block_host, workspace, stream=None) -> None:
    """End-to-end entry: per-step inputs / outputs are (pinned) HOST tensors, KV caches stay on the device.
    thresholds=None selects ART-off.  The call synchronises the stream before returning."""
    th = C.byref(thresholds) if thresholds is not None else None
    rc = load_library().art_decode_attention_host(
        C.byref(desc), _ptr(q_host), _ptr(k_cache), _ptr(v_cache), _ptr(block_table_host),
        _ptr(eligible_blocks_host), _ptr(seq_lens_host), th, _ptr(out_host), _ptr(stop_block_host),
        _ptr(workspace), workspace.numel() * workspace.element_size(), _stream_ptr(stream))
    if rc != 0:
        raise ArtError(rc, "art_decode_attention_host")


def art_hbm_read_probe(buf, stream=None) -> None:
    """Read-only streaming pass over a CUDA tensor (measurement aid, include/art_decode.h)."""
    rc = load_library().art_hbm_read_probe(_ptr(buf), buf.numel() * buf.element_size(), _stream_ptr(stream))
    if rc != 0:
        raise ArtError(rc, "art_hbm_read_probe")


def art_topk_blocks(desc, q, k_cache, block_table, seq_lens, top_k, block_scores, eligible_blocks, eligible_counts,
                    stream=None) -> None:
    """Importance-first block list of the scored base policy, built on the device (include/art_decode.h)."""
    rc = load_library().art_topk_blocks(C.byref(desc), _ptr(q), _ptr(k_cache), _ptr(block_table), _ptr(seq_lens),
                                        int(top_k), _ptr(block_scores), _ptr(eligible_blocks), _ptr(eligible_counts),
                                        _stream_ptr(stream))
    if rc != 0:
        raise ArtError(rc, "art_topk_blocks")


# ------------------------------------------------------------------ convenience (argument marshalling only)

def make_desc(w, *, split: int = 0, blocks_loaded=None, eligible_counts=None, sm_scale: float = 0.0) -> ArtDesc:
    """Fill an art_desc_t from a workload-like object (fields as in workloads.generators.Workload).
    A 4-D w.q is [B, m, Hq, d]: m query tokens per sequence (art_desc_t.q_len)."""
    ec = eligible_counts if eligible_counts is not None else w.eligible_counts
    return ArtDesc(
        batch=w.batch, num_q_heads=w.num_q_heads, num_kv_heads=w.num_kv_heads, head_dim=w.head_dim,
        block_tokens=64, dtype=ART_DTYPE_F32 if w.dtype == torch.float32 else ART_DTYPE_BF16,
        kv_layout=w.layout, policy=w.policy, max_blocks_per_seq=int(w.block_table.shape[1]),
        sink_tokens=w.sink_tokens, window_tokens=w.window_tokens,
        max_eligible=0 if w.eligible_blocks is None else int(w.eligible_blocks.shape[2]),
        sm_scale=sm_scale, split=split, q_len=int(w.q.shape[1]) if w.q.dim() == 4 else 0,
        num_pages=int(w.k_cache.shape[0]),
        eligible_counts=None if ec is None else ec.data_ptr(),
        blocks_loaded=None if blocks_loaded is None else blocks_loaded.data_ptr())


def run_workload(w, *, art: bool = True, split: int = 0, tau=None, phi=None, patience=None, probe_dim=None,
                 want_loaded: bool = False, stream=None, sm_scale: float = 0.0):
    """Allocate outputs and run one decode step on a CUDA-resident workload.
    Returns (out [B,Hq,d] (or [B,m,Hq,d]) fp32, stop_block [B,Hkv] int32, blocks_loaded or None)."""
    dev = w.q.device
    out = torch.empty(tuple(w.q.shape), dtype=torch.float32, device=dev)
    stop = torch.empty((w.batch, w.num_kv_heads), dtype=torch.int32, device=dev)
    loaded = torch.zeros((w.batch, w.num_kv_heads), dtype=torch.int32, device=dev) if want_loaded else None
    desc = make_desc(w, split=split, blocks_loaded=loaded, sm_scale=sm_scale)
    if art:
        th = ArtThresholds(tau=w.tau if tau is None else tau, phi=w.phi if phi is None else phi,
                           patience=w.patience if patience is None else patience,
                           probe_dim=w.probe_dim if probe_dim is None else probe_dim)
        art_decode_attention(desc, w.q, w.k_cache, w.v_cache, w.block_table, w.eligible_blocks, w.seq_lens,
                             th, out, stop, stream=stream)
    else:
        art_decode_attention_off(desc, w.q, w.k_cache, w.v_cache, w.block_table, w.eligible_blocks,
                                 w.seq_lens, out, stop, stream=stream)
    return out, stop, loaded


load_library()
