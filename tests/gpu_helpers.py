"""Glue for the GPU parity tests: numpy (oracle side) <-> torch CUDA tensors (library side).
Holds no arithmetic of the method."""
from __future__ import annotations

import numpy as np
import torch

import paper_2607_04443_b200 as ws
from paper_2607_04443_b200 import workloads as wl


def to_dev(x: np.ndarray, dtype: str) -> torch.Tensor:
    """float32 numpy values (exact BF16 when dtype == 'bf16') -> CUDA tensor of that dtype."""
    if dtype == "bf16":
        bits = wl.bf16_bits(x).view(np.int16)
        return torch.from_numpy(bits).cuda().view(torch.bfloat16)
    return torch.from_numpy(np.ascontiguousarray(x, np.float32)).cuda()


def to_host(t: torch.Tensor) -> np.ndarray:
    """CUDA tensor -> float32/float64-exact numpy array."""
    if t.dtype == torch.bfloat16:
        bits = t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
        return wl.bf16_from_bits(bits)
    return t.detach().cpu().numpy()


def raw_bytes(t: torch.Tensor) -> np.ndarray:
    return t.contiguous().view(torch.uint8).cpu().numpy().reshape(-1)


def workspace_for(Lq, H, d, kv_total, dtype=torch.bfloat16) -> torch.Tensor:
    n = ws.block_causal_attn_workspace_bytes(Lq, H, d, kv_total, dtype)
    return torch.empty(n, dtype=torch.uint8, device="cuda")


def gpu_attention(q, k_cache, v_cache, cache_len, k_new, v_new, q_block_end, kv_visible, scale, dtype="bf16", want_lse=True):
    """numpy in -> (out float32 numpy [Lq,H,d], lse float32 numpy [H,Lq]) through ws_block_causal_attn."""
    tq = to_dev(q, dtype)
    tkc, tvc = to_dev(k_cache, dtype), to_dev(v_cache, dtype)
    tkn = to_dev(k_new, dtype) if k_new is not None and len(k_new) else None
    tvn = to_dev(v_new, dtype) if v_new is not None and len(v_new) else None
    Lq, H, d = q.shape
    Ln = 0 if tkn is None else tkn.shape[0]
    out = torch.full_like(tq, float("nan"))
    lse = torch.full((H, Lq), float("nan"), dtype=torch.float32, device="cuda") if want_lse else None
    wsp = workspace_for(Lq, H, d, cache_len + Ln, tq.dtype)
    ws.block_causal_attn(out, tq, tkc, tvc, cache_len, tkn, tvn, list(q_block_end), list(kv_visible), scale, wsp, lse=lse)
    torch.cuda.synchronize()
    return to_host(out), (lse.cpu().numpy() if want_lse else None)
