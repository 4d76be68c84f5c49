"""B200-native ART decode attention (arXiv 2606.00024): C-ABI CUDA library + thin binding.

The product path is the sm_100a shared library built from ``csrc/``; this package only
marshals arguments.  There is no CPU fallback: importing ``binding`` without the built
library raises.
"""
from .binding import (  # noqa: F401
    ArtDesc, ArtThresholds, ART_PATIENCE_INF, ART_SPLIT_DYNAMIC, art_split_persistent, ART_DTYPE_F32, ART_DTYPE_BF16, ART_LAYOUT_HND, ART_LAYOUT_NHD,
    ART_POLICY_DENSE, ART_POLICY_SINK_WINDOW, ART_POLICY_LIST, ArtError, art_decode_attention,
    art_decode_attention_off, art_decode_attention_off_static, art_static_scratch_bytes, art_static_scratch_needed, art_decode_attention_host, art_topk_blocks, art_workspace_bytes, art_query_split, art_query_clusters, art_hbm_read_probe,
    art_status_string, art_version, lib_path, load_library, make_desc, run_workload,
)
