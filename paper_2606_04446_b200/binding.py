"""ctypes binding of libd2sd.so: the calls of include/d2sd.h with torch tensors as buffers.

Argument marshalling only -- every step of the path runs in the library's CUDA kernels.  Output
tensors are allocated here with torch (device memory is PyTorch's job) unless the caller passes
preallocated ones; all work is enqueued on torch's current CUDA stream, so the calls can be
captured into a ``torch.cuda.CUDAGraph``.
"""
from __future__ import annotations

import ctypes
import os
from typing import Dict, Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libd2sd.so")
_lib = None


class D2sdError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"d2sd status {status}: {message}")
        self.status = status


class _AttnParams(ctypes.Structure):
    _fields_ = [("B", ctypes.c_int32), ("T_cap", ctypes.c_int32), ("Hq", ctypes.c_int32),
                ("Hkv", ctypes.c_int32), ("d", ctypes.c_int32), ("sm_scale", ctypes.c_float),
                ("page_size", ctypes.c_int32), ("max_ctx_len", ctypes.c_int32),
                ("kv_rows", ctypes.c_int64), ("num_splits", ctypes.c_int32), ("impl", ctypes.c_int32),
                ("phases", ctypes.c_int32)]


class _CommitParams(ctypes.Structure):
    _fields_ = [("B", ctypes.c_int32), ("gamma", ctypes.c_int32), ("T_cap", ctypes.c_int32),
                ("Hkv", ctypes.c_int32), ("d", ctypes.c_int32), ("n_layers", ctypes.c_int32),
                ("page_size", ctypes.c_int32), ("kv_rows", ctypes.c_int64),
                ("tree_layer_stride", ctypes.c_int64), ("cache_layer_stride", ctypes.c_int64),
                ("F", ctypes.c_int32)]


def lib_path() -> str:
    return _LIB_PATH


def lib() -> ctypes.CDLL:
    """Load libd2sd.so (fails loudly when it has not been built: there is no fallback path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_2606_04446_b200.build` "
                              "(or __graft_entry__.build()); the D2SD path has no CPU fallback")
        L = ctypes.CDLL(_LIB_PATH)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        L.d2sd_last_error.restype = ctypes.c_char_p
        L.d2sd_version.restype = ctypes.c_char_p
        L.d2sd_select_prefixes.restype = i32
        L.d2sd_select_prefixes.argtypes = [vp, i32, i32, i32, vp, vp, vp]
        L.d2sd_build_tree.restype = i32
        L.d2sd_build_tree.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp]
        L.d2sd_cascade_workspace_bytes.restype = ctypes.c_size_t
        L.d2sd_cascade_workspace_bytes.argtypes = [ctypes.POINTER(_AttnParams)]
        L.d2sd_cascade_workspace_init.restype = i32
        L.d2sd_cascade_workspace_init.argtypes = [ctypes.POINTER(_AttnParams), vp, ctypes.c_size_t, vp]
        L.d2sd_cascade_verify_attn.restype = i32
        L.d2sd_cascade_verify_attn.argtypes = [ctypes.POINTER(_AttnParams)] + [vp] * 14 + [ctypes.c_size_t, vp]
        L.d2sd_accept_workspace_bytes.restype = ctypes.c_size_t
        L.d2sd_accept_workspace_bytes.argtypes = [i32, i32, i32]
        L.d2sd_accept.restype = i32
        L.d2sd_accept.argtypes = [vp, i64, i32, vp, vp, vp, vp, i32, i32, i32, vp, vp, vp, vp, vp, vp,
                                  ctypes.c_size_t, vp]
        L.d2sd_accept_static_max_bytes.restype = ctypes.c_size_t
        L.d2sd_accept_static_max_bytes.argtypes = []
        L.d2sd_accept_static.restype = i32
        L.d2sd_accept_static.argtypes = [vp, i64, i32, vp, vp, vp, vp, i32, i32, i32, vp, vp, vp, vp, vp, vp]
        L.d2sd_confidence_workspace_bytes.restype = ctypes.c_size_t
        L.d2sd_confidence_workspace_bytes.argtypes = [i32, i32, i32]
        L.d2sd_draft_confidence.restype = i32
        L.d2sd_draft_confidence.argtypes = [vp, i64, i32, vp, i32, i32, vp, vp, vp, ctypes.c_size_t, vp]
        L.d2sd_commit_workspace_bytes.restype = ctypes.c_size_t
        L.d2sd_commit_workspace_bytes.argtypes = [i32]
        L.d2sd_commit_kv.restype = i32
        L.d2sd_commit_kv.argtypes = ([ctypes.POINTER(_CommitParams)] + [vp] * 10 + [i32] + [vp] * 6 +
                                     [ctypes.c_size_t, vp])
        L.d2sd_select_third.restype = i32
        L.d2sd_select_third.argtypes = [vp, vp, i32, i32, i32, vp, vp, vp]
        L.d2sd_build_tree3.restype = i32
        L.d2sd_build_tree3.argtypes = [vp] * 6 + [i32] * 4 + [vp] * 8
        _lib = L
    return _lib


def version() -> str:
    return lib().d2sd_version().decode()


def last_error() -> str:
    return lib().d2sd_last_error().decode()


def t_cap(gamma: int, K: int) -> int:
    """Largest possible tree: gamma + K(gamma-1) - K(K-1)/2 (include/d2sd.h)."""
    return gamma + K * (gamma - 1) - K * (K - 1) // 2


def _check(status: int) -> None:
    if status != 0:
        raise D2sdError(status, last_error())


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    return None if t is None else t.data_ptr()


def _dev(t: torch.Tensor, dtype: torch.dtype, name: str) -> torch.Tensor:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of {dtype}, got "
                        f"{getattr(t, 'dtype', type(t))} on {getattr(t, 'device', '?')}")
    return t


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _out(t: Optional[torch.Tensor], shape, dtype, device, name: str) -> torch.Tensor:
    if t is None:
        return torch.empty(shape, dtype=dtype, device=device)
    _dev(t, dtype, name)
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: shape {tuple(t.shape)} != {tuple(shape)}")
    return t


# ------------------------------------------------------------------------------------------ (a)

def select_prefixes(conf: torch.Tensor, K: int, prefix_len: Optional[torch.Tensor] = None,
                    r_out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """d2sd_select_prefixes: conf fp32 [B,gamma] -> prefix_len int32 [B,K] (ascending)."""
    _dev(conf, torch.float32, "conf")
    B, gamma = conf.shape
    prefix_len = _out(prefix_len, (B, K), torch.int32, conf.device, "prefix_len")
    if r_out is not None:
        _out(r_out, (B, gamma - 1), torch.float64, conf.device, "r_out")
    _check(lib().d2sd_select_prefixes(_ptr(conf), B, gamma, K, _ptr(prefix_len), _ptr(r_out), _stream()))
    return prefix_len


# ------------------------------------------------------------------------------------------ (b)

def build_tree(draft1: torch.Tensor, draft2: torch.Tensor, prefix_len: torch.Tensor, ctx_len: torch.Tensor,
               T_cap: Optional[int] = None, out: Optional[Dict[str, torch.Tensor]] = None) -> Dict[str, torch.Tensor]:
    """d2sd_build_tree -> dict(tokens, parent, depth, pos_id [B,T_cap]; branch_off [B,K+1];
    mask uint32-as-int32 [B,T_cap,W]; tree_len [B])."""
    _dev(draft1, torch.int32, "draft1")
    B, gamma = draft1.shape
    K = prefix_len.shape[1]
    _dev(prefix_len, torch.int32, "prefix_len")
    _dev(draft2, torch.int32, "draft2")
    _dev(ctx_len, torch.int32, "ctx_len")
    if tuple(draft2.shape) != (B, K, gamma):
        raise ValueError(f"draft2: shape {tuple(draft2.shape)} != {(B, K, gamma)}")
    if T_cap is None:
        T_cap = t_cap(gamma, K)
    W = (T_cap + 31) // 32
    dev = draft1.device
    out = dict(out) if out else {}
    for name in ("tokens", "parent", "depth", "pos_id"):
        out[name] = _out(out.get(name), (B, T_cap), torch.int32, dev, name)
    out["branch_off"] = _out(out.get("branch_off"), (B, K + 1), torch.int32, dev, "branch_off")
    out["mask"] = _out(out.get("mask"), (B, T_cap, W), torch.int32, dev, "mask")  # uint32 bit pattern
    out["tree_len"] = _out(out.get("tree_len"), (B,), torch.int32, dev, "tree_len")
    _check(lib().d2sd_build_tree(_ptr(draft1), _ptr(draft2), _ptr(prefix_len), _ptr(ctx_len), B, gamma, K,
                                 T_cap, _ptr(out["tokens"]), _ptr(out["parent"]), _ptr(out["depth"]),
                                 _ptr(out["pos_id"]), _ptr(out["branch_off"]), _ptr(out["mask"]),
                                 _ptr(out["tree_len"]), _stream()))
    return out


# ------------------------------------------------------------------------------------------ (c)

def _params(q, tree_k, page_size, max_ctx_len, kv_rows, sm_scale, num_splits, impl, phases=0) -> _AttnParams:
    B, T_cap, Hq, d = q.shape
    return _AttnParams(B=B, T_cap=T_cap, Hq=Hq, Hkv=tree_k.shape[2], d=d,
                       sm_scale=float(sm_scale or 0.0), page_size=page_size, max_ctx_len=int(max_ctx_len),
                       kv_rows=int(kv_rows), num_splits=num_splits, impl=impl, phases=phases)


def cascade_workspace_bytes(B: int, T_cap: int, Hq: int, Hkv: int, d: int, max_ctx_len: int,
                            page_size: int = 0, kv_rows: int = 0, num_splits: int = 0, impl: int = 0) -> int:
    p = _AttnParams(B=B, T_cap=T_cap, Hq=Hq, Hkv=Hkv, d=d, sm_scale=0.0, page_size=page_size,
                    max_ctx_len=max_ctx_len, kv_rows=kv_rows, num_splits=num_splits, impl=impl, phases=0)
    n = lib().d2sd_cascade_workspace_bytes(ctypes.byref(p))
    if n == 0:
        raise D2sdError(-1, last_error())
    return int(n)


def cascade_workspace(B: int, T_cap: int, Hq: int, Hkv: int, d: int, max_ctx_len: int, device="cuda",
                      page_size: int = 0, kv_rows: int = 0, num_splits: int = 0, impl: int = 0) -> torch.Tensor:
    """Allocate a workspace for these params and initialise it (d2sd_cascade_workspace_init)."""
    p = _AttnParams(B=B, T_cap=T_cap, Hq=Hq, Hkv=Hkv, d=d, sm_scale=0.0, page_size=page_size,
                    max_ctx_len=max_ctx_len, kv_rows=kv_rows, num_splits=num_splits, impl=impl, phases=0)
    n = lib().d2sd_cascade_workspace_bytes(ctypes.byref(p))
    if n == 0:
        raise D2sdError(-1, last_error())
    ws = torch.empty(int(n), dtype=torch.uint8, device=device)
    _check(lib().d2sd_cascade_workspace_init(ctypes.byref(p), _ptr(ws), int(n), _stream()))
    return ws


def cascade_verify_attn(q: torch.Tensor, k_cache: torch.Tensor, v_cache: torch.Tensor,
                        kv_indptr: Optional[torch.Tensor], kv_indices: Optional[torch.Tensor],
                        ctx_len: torch.Tensor, tree_k: torch.Tensor, tree_v: torch.Tensor, mask: torch.Tensor,
                        tree_len: torch.Tensor, max_ctx_len: int, *, page_size: int = 0,
                        sm_scale: Optional[float] = None, num_splits: int = 0, impl: int = 0,
                        phases: int = 0, out: Optional[torch.Tensor] = None, lse: Optional[torch.Tensor] = None,
                        return_lse: bool = True, dbg_state: Optional[torch.Tensor] = None,
                        workspace: Optional[torch.Tensor] = None):
    """d2sd_cascade_verify_attn.  q bf16 [B,T_cap,Hq,d]; contiguous k/v_cache [rows,Hkv,d] or paged
    pool [P,16,Hkv,d]; returns (out bf16 [B,T_cap,Hq,d], lse fp32 [B,T_cap,Hq] or None)."""
    bf = torch.bfloat16
    _dev(q, bf, "q"); _dev(k_cache, bf, "k_cache"); _dev(v_cache, bf, "v_cache")
    _dev(tree_k, bf, "tree_k"); _dev(tree_v, bf, "tree_v")
    _dev(mask, torch.int32, "mask"); _dev(ctx_len, torch.int32, "ctx_len"); _dev(tree_len, torch.int32, "tree_len")
    if kv_indptr is not None:
        _dev(kv_indptr, torch.int32, "kv_indptr")
    if kv_indices is not None:
        _dev(kv_indices, torch.int32, "kv_indices")
    B, T_cap, Hq, d = q.shape
    kv_rows = k_cache.shape[0] * (k_cache.shape[1] if page_size else 1)
    p = _params(q, tree_k, page_size, max_ctx_len, kv_rows, sm_scale, num_splits, impl, phases)
    need = lib().d2sd_cascade_workspace_bytes(ctypes.byref(p))
    if need == 0:
        raise D2sdError(-1, last_error())
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=q.device)
        _check(lib().d2sd_cascade_workspace_init(ctypes.byref(p), _ptr(workspace), need, _stream()))
    out = _out(out, (B, T_cap, Hq, d), bf, q.device, "out")
    if lse is None and return_lse:
        lse = torch.empty((B, T_cap, Hq), dtype=torch.float32, device=q.device)
    if dbg_state is not None:
        _out(dbg_state, (2, B, T_cap, Hq, d + 1), torch.float32, q.device, "dbg_state")
    _check(lib().d2sd_cascade_verify_attn(
        ctypes.byref(p), _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(kv_indptr), _ptr(kv_indices),
        _ptr(ctx_len), _ptr(tree_k), _ptr(tree_v), _ptr(mask), _ptr(tree_len), _ptr(out), _ptr(lse),
        _ptr(dbg_state), _ptr(workspace), workspace.numel() * workspace.element_size(), _stream()))
    return out, lse


# ------------------------------------------------------------------------------------------ (d)

def accept_workspace_bytes(B: int, T_cap: int, V: int) -> int:
    return int(lib().d2sd_accept_workspace_bytes(B, T_cap, V))


def accept(logits: torch.Tensor, tokens: torch.Tensor, parent: torch.Tensor, depth: torch.Tensor,
           tree_len: torch.Tensor, gamma: int, out: Optional[Dict[str, torch.Tensor]] = None,
           workspace: Optional[torch.Tensor] = None) -> Dict[str, torch.Tensor]:
    """d2sd_accept: logits bf16 [B,T_cap,V] -> dict(argmax [B,T_cap], accept_len, bonus, best_node [B],
    path [B,gamma])."""
    if not (logits.is_cuda and logits.dtype == torch.bfloat16 and logits.dim() == 3 and logits.stride(2) == 1
            and logits.stride(0) == logits.shape[1] * logits.stride(1)):
        raise TypeError("logits: expected CUDA bf16 [B,T_cap,V] with unit inner stride and uniform row stride")
    B, T_cap, V = logits.shape
    for t, n in ((tokens, "tokens"), (parent, "parent"), (depth, "depth"), (tree_len, "tree_len")):
        _dev(t, torch.int32, n)
    dev = logits.device
    out = dict(out) if out else {}
    out["argmax"] = _out(out.get("argmax"), (B, T_cap), torch.int32, dev, "argmax")
    for name in ("accept_len", "bonus", "best_node"):
        out[name] = _out(out.get(name), (B,), torch.int32, dev, name)
    out["path"] = _out(out.get("path"), (B, gamma), torch.int32, dev, "path")
    need = accept_workspace_bytes(B, T_cap, V)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=dev)
    _check(lib().d2sd_accept(_ptr(logits), logits.stride(1), V, _ptr(tokens), _ptr(parent), _ptr(depth),
                             _ptr(tree_len), B, gamma, T_cap, _ptr(out["argmax"]), _ptr(out["accept_len"]),
                             _ptr(out["path"]), _ptr(out["bonus"]), _ptr(out["best_node"]), _ptr(workspace),
                             workspace.numel() * workspace.element_size(), _stream()))
    return out


def accept_static_max_bytes() -> int:
    return int(lib().d2sd_accept_static_max_bytes())


def accept_static(logits: torch.Tensor, tokens: torch.Tensor, parent: torch.Tensor, depth: torch.Tensor,
                  tree_len: torch.Tensor, gamma: int, out: Dict[str, torch.Tensor]) -> Dict[str, torch.Tensor]:
    """d2sd_accept_static: d2sd_accept with the library's built-in scratch.  Allocates nothing: the caller
    passes every output (out: argmax [B,T_cap], accept_len, bonus, best_node [B], path [B,gamma], int32)."""
    if not (logits.is_cuda and logits.dtype == torch.bfloat16 and logits.dim() == 3 and logits.stride(2) == 1
            and logits.stride(0) == logits.shape[1] * logits.stride(1)):
        raise TypeError("logits: expected CUDA bf16 [B,T_cap,V] with unit inner stride and uniform row stride")
    B, T_cap, V = logits.shape
    for t, n in ((tokens, "tokens"), (parent, "parent"), (depth, "depth"), (tree_len, "tree_len")):
        _dev(t, torch.int32, n)
    dev = logits.device
    for name, shape in (("argmax", (B, T_cap)), ("accept_len", (B,)), ("bonus", (B,)), ("best_node", (B,)),
                        ("path", (B, gamma))):
        if out.get(name) is None:
            raise TypeError(f"accept_static: out[{name!r}] must be given (this entry point allocates nothing)")
        _out(out[name], shape, torch.int32, dev, name)
    _check(lib().d2sd_accept_static(_ptr(logits), logits.stride(1), V, _ptr(tokens), _ptr(parent), _ptr(depth),
                                    _ptr(tree_len), B, gamma, T_cap, _ptr(out["argmax"]), _ptr(out["accept_len"]),
                                    _ptr(out["path"]), _ptr(out["bonus"]), _ptr(out["best_node"]), _stream()))
    return out


# ------------------------------------------------------------------------- the steps around the path

def t_cap3(gamma: int, K: int) -> int:
    """Largest depth-3 tree (include/d2sd.h, d2sd_build_tree3)."""
    return t_cap(gamma, K) + K * (gamma - 2) - K * (K - 1) // 2


def confidence_workspace_bytes(B: int, gamma: int, V: int) -> int:
    return int(lib().d2sd_confidence_workspace_bytes(B, gamma, V))


def draft_confidence(logits: torch.Tensor, anchor: torch.Tensor, draft: Optional[torch.Tensor] = None,
                     conf: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None):
    """d2sd_draft_confidence: drafter logits bf16 [B,gamma-1,V], anchor int32 [B] ->
    (draft int32 [B,gamma], conf fp32 [B,gamma]), slot 0 = (anchor, 1)."""
    if not (logits.is_cuda and logits.dtype == torch.bfloat16 and logits.dim() == 3 and logits.stride(2) == 1
            and logits.stride(0) == logits.shape[1] * logits.stride(1)):
        raise TypeError("logits: expected CUDA bf16 [B,gamma-1,V] with unit inner stride and uniform row stride")
    B, gm1, V = logits.shape
    gamma = gm1 + 1
    _dev(anchor, torch.int32, "anchor")
    draft = _out(draft, (B, gamma), torch.int32, logits.device, "draft")
    conf = _out(conf, (B, gamma), torch.float32, logits.device, "conf")
    if workspace is None:
        workspace = torch.empty(confidence_workspace_bytes(B, gamma, V), dtype=torch.uint8, device=logits.device)
    _check(lib().d2sd_draft_confidence(_ptr(logits), logits.stride(1), V, _ptr(anchor), B, gamma, _ptr(draft),
                                       _ptr(conf), _ptr(workspace), workspace.numel(), _stream()))
    return draft, conf


def commit_kv(tree_k: torch.Tensor, tree_v: torch.Tensor, path: torch.Tensor, accept_len: torch.Tensor,
              ctx_len: torch.Tensor, k_cache: torch.Tensor, v_cache: torch.Tensor,
              kv_indptr: Optional[torch.Tensor], kv_indices: Optional[torch.Tensor], page_size: int = 0, *,
              free_pages: Optional[torch.Tensor] = None, free_head: Optional[torch.Tensor] = None,
              ctx_len_out: Optional[torch.Tensor] = None, dropped: Optional[torch.Tensor] = None,
              feat: Optional[torch.Tensor] = None, feat_out: Optional[torch.Tensor] = None,
              workspace: Optional[torch.Tensor] = None):
    """d2sd_commit_kv.  tree_k/tree_v bf16 [n_layers,B,T_cap,Hkv,d]; caches bf16 [n_layers,rows,Hkv,d]
    (paged: rows = pages*page_size), updated IN PLACE; returns (ctx_len_out, dropped[, feat_out])."""
    bf = torch.bfloat16
    for t, n in ((tree_k, "tree_k"), (tree_v, "tree_v"), (k_cache, "k_cache"), (v_cache, "v_cache")):
        _dev(t, bf, n)
    for t, n in ((path, "path"), (accept_len, "accept_len"), (ctx_len, "ctx_len")):
        _dev(t, torch.int32, n)
    n_layers, B, T_cap, Hkv, d = tree_k.shape
    gamma = path.shape[1]
    kv_rows = k_cache.shape[1]
    if k_cache.shape[0] != n_layers or tuple(k_cache.shape[2:]) != (Hkv, d):
        raise ValueError(f"k_cache: shape {tuple(k_cache.shape)} does not match [n_layers, rows, {Hkv}, {d}]")
    dev = tree_k.device
    ctx_len_out = _out(ctx_len_out, (B,), torch.int32, dev, "ctx_len_out")
    dropped = _out(dropped, (B,), torch.int32, dev, "dropped")
    F = 0
    if feat is not None:
        _dev(feat, bf, "feat")
        F = feat.shape[2]
        feat_out = _out(feat_out, (B, gamma, F), bf, dev, "feat_out")
    p = _CommitParams(B=B, gamma=gamma, T_cap=T_cap, Hkv=Hkv, d=d, n_layers=n_layers, page_size=page_size,
                      kv_rows=kv_rows, tree_layer_stride=B * T_cap * Hkv * d, cache_layer_stride=kv_rows * Hkv * d, F=F)
    need = int(lib().d2sd_commit_workspace_bytes(B))
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=dev)
    _check(lib().d2sd_commit_kv(ctypes.byref(p), _ptr(tree_k), _ptr(tree_v), _ptr(path), _ptr(accept_len), _ptr(ctx_len),
                                _ptr(k_cache), _ptr(v_cache), _ptr(kv_indptr), _ptr(kv_indices), _ptr(free_pages),
                                0 if free_pages is None else free_pages.numel(), _ptr(free_head), _ptr(ctx_len_out),
                                _ptr(dropped), _ptr(feat), _ptr(feat_out), _ptr(workspace), workspace.numel(), _stream()))
    return (ctx_len_out, dropped) if feat is None else (ctx_len_out, dropped, feat_out)


def select_third(conf2: torch.Tensor, prefix_len: torch.Tensor, third_len: Optional[torch.Tensor] = None,
                 r3_out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """d2sd_select_third: conf2 fp32 [B,K,gamma], prefix_len int32 [B,K] -> third_len int32 [B,K] (-1 = none)."""
    _dev(conf2, torch.float32, "conf2")
    _dev(prefix_len, torch.int32, "prefix_len")
    B, K, gamma = conf2.shape
    third_len = _out(third_len, (B, K), torch.int32, conf2.device, "third_len")
    if r3_out is not None:
        _out(r3_out, (B, K, gamma - 1), torch.float64, conf2.device, "r3_out")
    _check(lib().d2sd_select_third(_ptr(conf2), _ptr(prefix_len), B, gamma, K, _ptr(third_len), _ptr(r3_out), _stream()))
    return third_len


def build_tree3(draft1: torch.Tensor, draft2: torch.Tensor, draft3: torch.Tensor, prefix_len: torch.Tensor,
                third_len: torch.Tensor, ctx_len: torch.Tensor, T_cap: Optional[int] = None) -> Dict[str, torch.Tensor]:
    """d2sd_build_tree3 -> the dict of build_tree with branch_off [B,2K+1]."""
    B, gamma = draft1.shape
    K = prefix_len.shape[1]
    for t, n in ((draft1, "draft1"), (draft2, "draft2"), (draft3, "draft3"), (prefix_len, "prefix_len"),
                 (third_len, "third_len"), (ctx_len, "ctx_len")):
        _dev(t, torch.int32, n)
    if T_cap is None:
        T_cap = t_cap3(gamma, K)
    W = (T_cap + 31) // 32
    dev = draft1.device
    out = {name: torch.empty((B, T_cap), dtype=torch.int32, device=dev) for name in ("tokens", "parent", "depth", "pos_id")}
    out["branch_off"] = torch.empty((B, 2 * K + 1), dtype=torch.int32, device=dev)
    out["mask"] = torch.empty((B, T_cap, W), dtype=torch.int32, device=dev)
    out["tree_len"] = torch.empty((B,), dtype=torch.int32, device=dev)
    _check(lib().d2sd_build_tree3(_ptr(draft1), _ptr(draft2), _ptr(draft3), _ptr(prefix_len), _ptr(third_len),
                                  _ptr(ctx_len), B, gamma, K, T_cap, _ptr(out["tokens"]), _ptr(out["parent"]),
                                  _ptr(out["depth"]), _ptr(out["pos_id"]), _ptr(out["branch_off"]), _ptr(out["mask"]),
                                  _ptr(out["tree_len"]), _stream()))
    return out
