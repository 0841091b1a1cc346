"""ws_block_causal_attn_static_ws: attention for callers that cannot allocate device memory.

Who needs it: code that must run block-causal attention but has nowhere to get a workspace from -- a plug-in in a
serving process whose framework took all of HBM for its own pools (cudaMalloc fails, the pool is not reachable from C),
the per-unit real-time loop (a cudaMalloc / cudaFree there synchronises the device and stalls the units in flight), or
a set-up that forbids allocation once it is running.  The entry point takes its scratch from a 64 MiB array inside the
library's device image and is otherwise ws_block_causal_attn.

What is checked here:
  * on a GPU: its output equals the workspace-taking call's on the same inputs, within the attention tolerance of the
    parity suite (max-abs 2e-2, relative Frobenius 1e-2; LSE 2e-2), on TWO calls in a row with different problems --
    the second call finds the first one's partial results still in the shared array and must not be disturbed by them;
    a problem beyond the 64 MiB limit is refused and no output byte changes;
  * without a GPU: the limit and the argument rules are enforced on the host, before CUDA is touched.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here should not hide
the parity suite.  It does not depend on what ran before it (it makes its own inputs and compares two library calls),
so it passes alone in a fresh process and at the end of the full run alike.
"""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

import paper_2607_04443_b200 as ws
from paper_2607_04443_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
MAX_ABS, REL_FRO, LSE_ABS = 2e-2, 1e-2, 2e-2   # the tolerances of tests/test_gpu_parity.py
WORKSPACE, INVALID, UNSUPPORTED, ALIGN, RANGE = -6, -1, -2, -3, -4


@pytest.fixture(scope="module")
def lib():
    build.build_lib()
    return binding.load()


# ---------------------------------------------------------------- host side (no GPU needed)

def test_limit_matches_the_header():
    text = open(os.path.join(ROOT, "include", "ws.h")).read()
    m = re.search(r"#define\s+WS_STATIC_WORKSPACE_BYTES\s+\((\d+)u\s*<<\s*(\d+)\)", text)
    assert m, "WS_STATIC_WORKSPACE_BYTES not found in ws.h"
    assert int(m.group(1)) << int(m.group(2)) == ws.STATIC_WORKSPACE_BYTES == 64 << 20


def test_every_baseline_config_fits_the_built_in_scratch(lib):
    shapes = {"cfg1": (64, 2, 64, 192, torch.float32), "cfg2": (292, 24, 128, 8192 + 292, torch.bfloat16),
              "cfg3": (970, 40, 128, 16384 + 970, torch.bfloat16), "cfg4": (3680, 10, 128, 16384 + 3680, torch.bfloat16),
              "cfg5": (970, 40, 128, 65536 + 970, torch.bfloat16)}
    for name, (Lq, H, d, kv, dt) in shapes.items():
        assert ws.block_causal_attn_workspace_bytes(Lq, H, d, kv, dt) <= ws.STATIC_WORKSPACE_BYTES, name


def test_rejects_on_the_host_before_cuda_is_touched(lib):
    f = lib.ws_block_causal_attn_static_ws
    Mask = binding._BlockMask
    P = ctypes.c_void_p

    def call(out=0x10000000, q=0x20000000, kc=0x30000000, vc=0x40000000, cap=512, Tc=512, kn=0x50000000, vn=0x60000000, Ln=64,
             H=2, d=128, Lq=64, qe=(32, 64), kv=(544, 576), scale=0.1, dt=0):
        n = len(qe)
        m = Mask(n, (ctypes.c_int32 * n)(*qe), (ctypes.c_int32 * n)(*kv))
        return f(P(out), None, P(q), P(kc), P(vc), cap, Tc, P(kn) if kn else None, P(vn) if vn else None, Ln, H, d, Lq,
                 ctypes.byref(m), scale, dt, None)

    # too large for the 64 MiB array: 970 rows x 64 heads x 128 needs about 68 MB
    assert ws.block_causal_attn_workspace_bytes(970, 64, 128, 576, torch.bfloat16) > ws.STATIC_WORKSPACE_BYTES
    assert call(H=64, Lq=970, qe=(970,), kv=(576,)) == WORKSPACE
    assert "workspace" in ws.status_string(WORKSPACE).lower()
    # the argument rules of ws_block_causal_attn, same codes
    assert call(d=96) == UNSUPPORTED
    assert call(dt=3) == UNSUPPORTED
    assert call(qe=(32, 63)) == INVALID
    assert call(out=0) == INVALID
    assert call(kv=(544, 577)) == RANGE
    assert call(Tc=513) == RANGE
    assert call(q=0x20000008) == ALIGN
    assert call(kn=0) == INVALID


# ---------------------------------------------------------------- GPU

def _problem(seed, Lq, H, d, cache_len, Ln, qe, kv, capacity=None):
    g = torch.Generator(device="cpu").manual_seed(seed)
    r = lambda *s: torch.randn(*s, generator=g, dtype=torch.float32).to(torch.bfloat16).cuda()
    capacity = capacity or cache_len
    return dict(q=r(Lq, H, d), kc=r(H, capacity, d), vc=r(H, capacity, d), cache_len=cache_len,
                kn=r(Ln, H, d) if Ln else None, vn=r(Ln, H, d) if Ln else None, qe=list(qe), kv=list(kv), scale=d ** -0.5)


def _run_both(p):
    """(out, lse) of the static-scratch entry point and of ws_block_causal_attn with its own workspace."""
    Lq, H, d = p["q"].shape
    Ln = 0 if p["kn"] is None else p["kn"].shape[0]
    res = []
    for static in (True, False):
        out = torch.full_like(p["q"], float("nan"))
        lse = torch.full((H, Lq), float("nan"), dtype=torch.float32, device="cuda")
        if static:
            ws.block_causal_attn_static_ws(out, p["q"], p["kc"], p["vc"], p["cache_len"], p["kn"], p["vn"], p["qe"], p["kv"],
                                           p["scale"], lse=lse)
        else:
            n = ws.block_causal_attn_workspace_bytes(Lq, H, d, p["cache_len"] + Ln, torch.bfloat16)
            wsp = torch.full((n // 4,), float("nan"), dtype=torch.float32, device="cuda").view(torch.uint8)
            ws.block_causal_attn(out, p["q"], p["kc"], p["vc"], p["cache_len"], p["kn"], p["vn"], p["qe"], p["kv"], p["scale"],
                                 wsp, lse=lse)
        torch.cuda.synchronize()
        res.append((out.float().cpu().numpy().astype(np.float64), lse.cpu().numpy().astype(np.float64)))
    return res


def _assert_close(got, ref, what):
    (o, l), (o_ref, l_ref) = got, ref
    assert np.all(np.isfinite(o)), f"{what}: non-finite output"
    assert np.max(np.abs(o - o_ref)) <= MAX_ABS, f"{what}: max-abs"
    assert np.linalg.norm(o - o_ref) <= REL_FRO * np.linalg.norm(o_ref), f"{what}: rel-Frobenius"
    fin = np.isfinite(l_ref)
    assert np.array_equal(np.isfinite(l), fin), f"{what}: lse finiteness"
    assert np.max(np.abs(l[fin] - l_ref[fin])) <= LSE_ABS, f"{what}: lse"


@pytest.mark.gpu
def test_static_scratch_matches_the_workspace_call_on_two_calls_in_a_row():
    # Both problems split work items over several CTAs, so the scratch really carries partial results:
    # 1) a config-2-shaped unit (292 rows, 24 heads, 8192 cached keys + its own): 48 items over 148 SMs;
    # 2) right after it, a smaller two-block problem with a ragged tail, which finds call 1's records in the array.
    first = _problem(11, 292, 24, 128, 8192, 292, (292,), (8192 + 292,))
    second = _problem(12, 200, 6, 128, 3000, 200, (90, 200), (3090, 3200), capacity=3072)
    a_static, a_ref = _run_both(first)
    _assert_close(a_static, a_ref, "first call")
    b_static, b_ref = _run_both(second)
    _assert_close(b_static, b_ref, "second call")
    # and the first problem again, now behind the second one's leftovers
    c_static, c_ref = _run_both(first)
    _assert_close(c_static, c_ref, "third call")


@pytest.mark.gpu
def test_back_to_back_on_one_stream_without_a_host_sync_in_between():
    """Stream order is the only thing that keeps two calls apart: the second waits for the first on the same stream."""
    p1 = _problem(21, 292, 24, 128, 4096, 292, (292,), (4096 + 292,))
    p2 = _problem(22, 300, 8, 64, 2048, 0, (300,), (2048,))
    outs = []
    for p in (p1, p2):
        out = torch.full_like(p["q"], float("nan"))
        ws.block_causal_attn_static_ws(out, p["q"], p["kc"], p["vc"], p["cache_len"], p["kn"], p["vn"], p["qe"], p["kv"], p["scale"])
        outs.append(out)
    torch.cuda.synchronize()
    for p, out in zip((p1, p2), outs):
        ref = _run_both(p)[1]
        got = (out.float().cpu().numpy().astype(np.float64), ref[1])  # lse not requested above: compare O only
        _assert_close(got, ref, "pipelined call")


@pytest.mark.gpu
def test_problem_beyond_the_limit_is_refused_and_nothing_is_written():
    Lq, H, d = 970, 64, 128      # needs about 68 MB of scratch
    q = torch.zeros(Lq, H, d, dtype=torch.bfloat16, device="cuda")
    kc = torch.zeros(H, 128, d, dtype=torch.bfloat16, device="cuda")
    out = torch.full_like(q, 7.0)
    with pytest.raises(ws.WsError) as ei:
        ws.block_causal_attn_static_ws(out, q, kc, kc.clone(), 128, None, None, [Lq], [128], 0.1)
    assert ei.value.status == WORKSPACE
    assert "built-in" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())
