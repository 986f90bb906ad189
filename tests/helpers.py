"""Shared helpers of the GPU parity tests: move seeded inputs to the device, run the CUDA path
through the C ABI binding, compare with the oracle under the gates DESIGN.md states."""
from __future__ import annotations

import numpy as np
import torch

import d2sd_synth as synth

# Float gates (BASELINE.json north_star; stricter ones from DESIGN.md "Tolerances").
OUT_ATOL, OUT_RTOL = 2e-2, 1e-2      # |gpu - ref| <= atol + rtol*|ref| per element (bf16 out)
LSE_ATOL = 1e-3                      # natural-log LSE, absolute
ROW_REL_L2 = 1e-2                    # per (node, head) relative L2 error of the bf16 output
STATE_REL_L2 = 5e-3                  # per-row relative L2 of the fp32 prefix-only / tree-only states


def bf16_cuda(bits: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16).cuda()


def i32_cuda(a: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a).astype(np.int32, copy=False)).cuda()


def mask_cuda(mask_u32: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(mask_u32).view(np.int32)).cuda()


def oracle_tree(oracle, cfg, step):
    pl, r = oracle.select_prefixes(step["conf"], cfg.K)
    tree = oracle.build_tree(step["draft1"], step["draft2"], pl, step["ctx_len"], cfg.T_cap)
    return pl, r, tree


def gpu_attention(d2sd, cfg, step, tree, ti, kv, **kw):
    """Run d2sd_cascade_verify_attn on the oracle-built tree (so that stage (c) is tested in
    isolation).  Returns (out fp32 numpy, lse numpy, dbg numpy or None)."""
    dbg = kw.pop("dbg", False)
    B, T, Hq, d = ti["q"].shape
    dbg_t = torch.full((2, B, T, Hq, d + 1), float("nan"), dtype=torch.float32, device="cuda") if dbg else None
    out0 = torch.full((B, T, Hq, d), float("nan"), dtype=torch.bfloat16, device="cuda")
    lse0 = torch.full((B, T, Hq), float("nan"), dtype=torch.float32, device="cuda")
    out, lse = d2sd.cascade_verify_attn(
        bf16_cuda(ti["q"]), bf16_cuda(kv["k_cache"]), bf16_cuda(kv["v_cache"]),
        None if kv["kv_indptr"] is None else i32_cuda(kv["kv_indptr"]),
        None if kv["kv_indices"] is None else i32_cuda(kv["kv_indices"]),
        i32_cuda(step["ctx_len"]), bf16_cuda(ti["tree_k"]), bf16_cuda(ti["tree_v"]),
        mask_cuda(tree["mask"]), i32_cuda(tree["tree_len"]), int(step["ctx_len"].max()),
        page_size=kv["page_size"], out=out0, lse=lse0, dbg_state=dbg_t, **kw)
    torch.cuda.synchronize()
    return (out.float().cpu().numpy(), lse.cpu().numpy(), None if dbg_t is None else dbg_t.cpu().numpy())


def check_rows(got_o, got_lse, ref_o, ref_lse, what="", row_gate=ROW_REL_L2, elementwise=True):
    """got_o/ref_o [..., d], got_lse/ref_lse [...]: the gates above, with a useful message."""
    got_o = np.asarray(got_o, np.float64)
    assert np.isfinite(got_o).all(), f"{what}: non-finite output"
    if elementwise:
        bad = np.abs(got_o - ref_o) > OUT_ATOL + OUT_RTOL * np.abs(ref_o)
        assert not bad.any(), f"{what}: {bad.sum()} elements outside atol/rtol, max err {np.abs(got_o - ref_o).max():.3e}"
    num = np.linalg.norm(got_o - ref_o, axis=-1)
    den = np.linalg.norm(ref_o, axis=-1)
    rel = num / np.maximum(den, 1e-30)
    assert (rel <= row_gate).all(), f"{what}: row rel-L2 max {rel.max():.3e} > {row_gate}"
    if got_lse is not None:
        fin = np.isfinite(ref_lse)
        err = np.abs(np.asarray(got_lse, np.float64)[fin] - ref_lse[fin])
        assert err.size == 0 or err.max() <= LSE_ATOL, f"{what}: LSE max err {err.max():.3e}"
        assert np.array_equal(np.isneginf(got_lse), np.isneginf(ref_lse)), f"{what}: -inf LSE pattern differs"
    return float(rel.max())


def valid_rows(tree_len, T_cap):
    """Boolean [B,T_cap] of real tree nodes."""
    return np.arange(T_cap)[None, :] < np.asarray(tree_len)[:, None]
