"""B200-native performer hot path of Wan-Streamer v0.2 (arxiv/paper_2607_04443).

KV-cache write, Ulysses-local seq<->head relayouts and block-causal unit attention as
hand-written sm_100a CUDA kernels behind a C ABI (include/ws.h).  This package is the thin
Python binding: argument marshalling only.  There is no CPU fallback -- every call raises
if libws.so is missing or the device is not a CUDA device.
"""
from .binding import (  # noqa: F401
    WsError, lib_path, load, version, status_string,
    kv_cache_write, seq_to_head, head_to_seq, seq_to_head_multi, head_to_seq_multi,
    block_causal_attn, block_causal_attn_workspace_bytes, block_causal_attn_seq_layout,
    block_causal_attn_static_ws, STATIC_WORKSPACE_BYTES,
    kv_cache_write_fp8, block_causal_attn_fp8kv,
    kv_cache_write_ring, block_causal_attn_ring, ring_state,
    ulysses_push_seq_to_head, block_causal_attn_push_out, kv_slice_broadcast_write,
    unit_forward_host, unit_forward_host_staging_bytes, kernel_launch_count, attn_schedule, EXPORTS,
    DTYPE_BF16, DTYPE_F32, ABI_VERSION,
)
