"""ctypes front end of the CPU oracle (``d2sd_oracle.c``).

TEST INFRASTRUCTURE, NOT PRODUCT: only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.  It never
imports the CUDA package and the CUDA package never imports it.

Every function takes and returns numpy arrays; bf16 tensors are ``uint16`` bit patterns.
The arithmetic lives in the C file (each function there cites the PAPER.md passage it follows);
this file only marshals arguments.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "d2sd_oracle.c")
_LIB = os.path.join(_HERE, "libd2sd_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, no fast-math, no FP contraction, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-fno-fast-math", "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.d2sd_oracle_num_threads.restype = ctypes.c_int32
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _c(a, dtype) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


def num_threads() -> int:
    return int(_load().d2sd_oracle_num_threads())


def select_prefixes(conf: np.ndarray, K: int) -> Tuple[np.ndarray, np.ndarray]:
    """conf fp32 [B,gamma] -> (prefix_len int32 [B,K] ascending, r fp64 [B,gamma-1])."""
    conf = _c(conf, np.float32)
    B, gamma = conf.shape
    assert 0 <= K <= gamma - 1 and gamma >= 2
    prefix_len = np.zeros((B, K), dtype=np.int32)
    r = np.zeros((B, gamma - 1), dtype=np.float64)
    _load().d2sd_oracle_select(_p(conf), ctypes.c_int32(B), ctypes.c_int32(gamma), ctypes.c_int32(K),
                               _p(prefix_len), _p(r))
    return prefix_len, r


def build_tree(draft1: np.ndarray, draft2: np.ndarray, prefix_len: np.ndarray, ctx_len: np.ndarray,
               T_cap: int) -> dict:
    draft1 = _c(draft1, np.int32)
    B, gamma = draft1.shape
    prefix_len = _c(prefix_len, np.int32).reshape(B, -1)
    K = prefix_len.shape[1]
    draft2 = _c(draft2, np.int32).reshape(B, K, gamma)
    ctx_len = _c(ctx_len, np.int32)
    W = (T_cap + 31) // 32
    out = {
        "tokens": np.zeros((B, T_cap), np.int32), "parent": np.zeros((B, T_cap), np.int32),
        "depth": np.zeros((B, T_cap), np.int32), "pos_id": np.zeros((B, T_cap), np.int32),
        "branch_off": np.zeros((B, K + 1), np.int32), "mask": np.zeros((B, T_cap, W), np.uint32),
        "tree_len": np.zeros((B,), np.int32),
    }
    _load().d2sd_oracle_build_tree(_p(draft1), _p(draft2), _p(prefix_len), _p(ctx_len),
                                   ctypes.c_int32(B), ctypes.c_int32(gamma), ctypes.c_int32(K),
                                   ctypes.c_int32(T_cap), _p(out["tokens"]), _p(out["parent"]),
                                   _p(out["depth"]), _p(out["pos_id"]), _p(out["branch_off"]),
                                   _p(out["mask"]), _p(out["tree_len"]))
    return out


WHICH = {"full": 0, "prefix": 1, "tree": 2}


def _attn_common(q, k_cache, v_cache, kv_indptr, kv_indices, page_size, ctx_len, tree_k, tree_v, mask):
    q = _c(q, np.uint16)
    B, T_cap, Hq, d = q.shape
    tree_k = _c(tree_k, np.uint16)
    tree_v = _c(tree_v, np.uint16)
    Hkv = tree_k.shape[2]
    k_cache = _c(k_cache, np.uint16)
    v_cache = _c(v_cache, np.uint16)
    kv_indptr = None if kv_indptr is None else _c(kv_indptr, np.int32)
    kv_indices = None if kv_indices is None else _c(kv_indices, np.int32)
    ctx_len = _c(ctx_len, np.int32)
    mask = _c(mask, np.uint32)
    W = mask.shape[-1]
    assert mask.shape == (B, T_cap, W) and W == (T_cap + 31) // 32
    assert (page_size > 0) == (kv_indices is not None)
    return q, k_cache, v_cache, kv_indptr, kv_indices, ctx_len, tree_k, tree_v, mask, (B, T_cap, W, Hq, Hkv, d)


def attention(q, k_cache, v_cache, kv_indptr, kv_indices, page_size, ctx_len, tree_k, tree_v, mask,
              tree_len, sm_scale: Optional[float] = None, which: str = "full"):
    """Explicit masked softmax attention for every (b, t<tree_len[b], h).
    Returns (out fp64 [B,T_cap,Hq,d], lse fp64 [B,T_cap,Hq]); padding rows are NaN."""
    (q, k_cache, v_cache, kv_indptr, kv_indices, ctx_len, tree_k, tree_v, mask,
     (B, T_cap, W, Hq, Hkv, d)) = _attn_common(q, k_cache, v_cache, kv_indptr, kv_indices, page_size,
                                               ctx_len, tree_k, tree_v, mask)
    tree_len = _c(tree_len, np.int32)
    if sm_scale is None:
        sm_scale = 1.0 / np.sqrt(float(d))
    out = np.full((B, T_cap, Hq, d), np.nan, np.float64)
    lse = np.full((B, T_cap, Hq), np.nan, np.float64)
    _load().d2sd_oracle_attention(
        ctypes.c_int32(WHICH[which]), _p(q), _p(k_cache), _p(v_cache), _p(kv_indptr), _p(kv_indices),
        ctypes.c_int32(page_size), _p(ctx_len), _p(tree_k), _p(tree_v), _p(mask), _p(tree_len),
        ctypes.c_int32(B), ctypes.c_int32(T_cap), ctypes.c_int32(W), ctypes.c_int32(Hq),
        ctypes.c_int32(Hkv), ctypes.c_int32(d), ctypes.c_double(sm_scale), _p(out), _p(lse))
    return out, lse


def attention_rows(q, k_cache, v_cache, kv_indptr, kv_indices, page_size, ctx_len, tree_k, tree_v,
                   mask, sel, sm_scale: Optional[float] = None, which: str = "full"):
    """Same definition for a list of (b,t,h) triples ``sel`` [n,3] -> (out [n,d], lse [n])."""
    (q, k_cache, v_cache, kv_indptr, kv_indices, ctx_len, tree_k, tree_v, mask,
     (B, T_cap, W, Hq, Hkv, d)) = _attn_common(q, k_cache, v_cache, kv_indptr, kv_indices, page_size,
                                               ctx_len, tree_k, tree_v, mask)
    sel = _c(sel, np.int32).reshape(-1, 3)
    if sm_scale is None:
        sm_scale = 1.0 / np.sqrt(float(d))
    n = sel.shape[0]
    out = np.zeros((n, d), np.float64)
    lse = np.zeros((n,), np.float64)
    _load().d2sd_oracle_attention_rows(
        ctypes.c_int32(WHICH[which]), _p(q), _p(k_cache), _p(v_cache), _p(kv_indptr), _p(kv_indices),
        ctypes.c_int32(page_size), _p(ctx_len), _p(tree_k), _p(tree_v), _p(mask),
        ctypes.c_int32(T_cap), ctypes.c_int32(W), ctypes.c_int32(Hq), ctypes.c_int32(Hkv),
        ctypes.c_int32(d), ctypes.c_double(sm_scale), _p(sel), ctypes.c_int64(n), _p(out), _p(lse))
    return out, lse


def argmax(logits: np.ndarray, tree_len: np.ndarray) -> np.ndarray:
    """logits bf16 bits [B,T_cap,V] -> first-index argmax int32 [B,T_cap] (-1 on padding rows)."""
    logits = _c(logits, np.uint16)
    B, T_cap, V = logits.shape
    tree_len = _c(tree_len, np.int32)
    a = np.zeros((B, T_cap), np.int32)
    _load().d2sd_oracle_argmax(_p(logits), ctypes.c_int64(V), ctypes.c_int32(V), _p(tree_len),
                               ctypes.c_int32(B), ctypes.c_int32(T_cap), _p(a))
    return a


def accept_walk(argmax_: np.ndarray, tokens, parent, depth, tree_len, gamma: int) -> dict:
    a = _c(argmax_, np.int32)
    B, T_cap = a.shape
    tokens, parent, depth = _c(tokens, np.int32), _c(parent, np.int32), _c(depth, np.int32)
    tree_len = _c(tree_len, np.int32)
    out = {"accept_len": np.zeros((B,), np.int32), "path": np.zeros((B, gamma), np.int32),
           "bonus": np.zeros((B,), np.int32), "best_node": np.zeros((B,), np.int32)}
    _load().d2sd_oracle_accept_walk(_p(a), _p(tokens), _p(parent), _p(depth), _p(tree_len),
                                    ctypes.c_int32(B), ctypes.c_int32(gamma), ctypes.c_int32(T_cap),
                                    _p(out["accept_len"]), _p(out["path"]), _p(out["bonus"]),
                                    _p(out["best_node"]))
    return out


def accept(logits: np.ndarray, tokens, parent, depth, tree_len, gamma: int) -> dict:
    a = argmax(logits, tree_len)
    out = accept_walk(a, tokens, parent, depth, tree_len, gamma)
    out["argmax"] = a
    return out


# ------------------------------------------------------------------------------- next rows

def confidence(logits: np.ndarray, anchor: np.ndarray):
    """f3, Eq. 3.  logits bf16 bits [B,gamma-1,V], anchor int32 [B] ->
    (draft int32 [B,gamma], conf fp64 [B,gamma]); slot 0 = (anchor, 1)."""
    logits = _c(logits, np.uint16)
    B, gm1, V = logits.shape
    gamma = gm1 + 1
    anchor = _c(anchor, np.int32)
    draft = np.zeros((B, gamma), np.int32)
    conf = np.zeros((B, gamma), np.float64)
    _load().d2sd_oracle_confidence(_p(logits), ctypes.c_int64(V), ctypes.c_int32(V), _p(anchor),
                                   ctypes.c_int32(B), ctypes.c_int32(gamma), _p(draft), _p(conf))
    return draft, conf


def commit_kv(tree_k, tree_v, path, accept_len, ctx_len, k_cache, v_cache, kv_indptr, kv_indices,
              page_size: int, free_pages=None, free_head: int = 0):
    """f1.  tree_k/tree_v bf16 bits [n_layers,B,T_cap,Hkv,d]; caches
    [n_layers,rows,Hkv,d] (paged: rows = pages*page_size).  Returns a dict with the NEW k_cache,
    v_cache, kv_indices (copies; inputs untouched), ctx_len, dropped, free_head."""
    tree_k, tree_v = _c(tree_k, np.uint16), _c(tree_v, np.uint16)
    n_layers, B, T_cap, Hkv, d = tree_k.shape
    k_cache, v_cache = _c(k_cache, np.uint16).copy(), _c(v_cache, np.uint16).copy()
    assert k_cache.shape[0] == n_layers and k_cache.shape[2:] == (Hkv, d)
    kv_rows = k_cache.shape[1]
    path = _c(path, np.int32)
    gamma = path.shape[1]
    accept_len, ctx_len = _c(accept_len, np.int32), _c(ctx_len, np.int32)
    kv_indptr = None if kv_indptr is None else _c(kv_indptr, np.int32)
    kv_indices = None if kv_indices is None else _c(kv_indices, np.int32).copy()
    free_pages = None if free_pages is None else _c(free_pages, np.int32)
    head = np.array([free_head], np.int32)
    ctx_out = np.zeros((B,), np.int32)
    dropped = np.zeros((B,), np.int32)
    _load().d2sd_oracle_commit_kv(
        _p(tree_k), _p(tree_v), ctypes.c_int64(B * T_cap * Hkv * d), _p(path), _p(accept_len), _p(ctx_len),
        _p(k_cache), _p(v_cache), ctypes.c_int64(kv_rows * Hkv * d), ctypes.c_int64(kv_rows), _p(kv_indptr),
        _p(kv_indices), ctypes.c_int32(page_size), _p(free_pages),
        ctypes.c_int32(0 if free_pages is None else free_pages.size), _p(head), ctypes.c_int32(B),
        ctypes.c_int32(gamma), ctypes.c_int32(T_cap), ctypes.c_int32(Hkv), ctypes.c_int32(d),
        ctypes.c_int32(n_layers), _p(ctx_out), _p(dropped))
    return {"k_cache": k_cache, "v_cache": v_cache, "kv_indices": kv_indices, "ctx_len": ctx_out,
            "dropped": dropped, "free_head": int(head[0])}


def gather_path(feat, path, accept_len):
    """f1.  feat bf16 bits [B,T_cap,F] -> [B,gamma,F] rows of the accepted path, zero padded."""
    feat = _c(feat, np.uint16)
    B, T_cap, F = feat.shape
    path = _c(path, np.int32)
    gamma = path.shape[1]
    out = np.zeros((B, gamma, F), np.uint16)
    _load().d2sd_oracle_gather_path(_p(feat), _p(path), _p(_c(accept_len, np.int32)), ctypes.c_int32(B),
                                    ctypes.c_int32(gamma), ctypes.c_int32(T_cap), ctypes.c_int32(F), _p(out))
    return out


def select_third(conf2, prefix_len):
    """f2.  conf2 fp32 [B,K,gamma], prefix_len [B,K] -> (third_len int32 [B,K] (-1 = none),
    r3 fp64 [B,K,gamma-1])."""
    conf2 = _c(conf2, np.float32)
    B, K, gamma = conf2.shape
    prefix_len = _c(prefix_len, np.int32).reshape(B, K)
    third = np.zeros((B, K), np.int32)
    r3 = np.zeros((B, K, gamma - 1), np.float64)
    _load().d2sd_oracle_select_third(_p(conf2), _p(prefix_len), ctypes.c_int32(B), ctypes.c_int32(gamma),
                                     ctypes.c_int32(K), _p(third), _p(r3))
    return third, r3


def build_tree3(draft1, draft2, draft3, prefix_len, third_len, ctx_len, T_cap: int) -> dict:
    """f2: the depth-3 tree (two-level tree + third-level continuations); branch_off [B,2K+1]."""
    draft1 = _c(draft1, np.int32)
    B, gamma = draft1.shape
    prefix_len = _c(prefix_len, np.int32).reshape(B, -1)
    K = prefix_len.shape[1]
    draft2 = _c(draft2, np.int32).reshape(B, K, gamma)
    draft3 = _c(draft3, np.int32).reshape(B, K, gamma)
    third_len = _c(third_len, np.int32).reshape(B, K)
    ctx_len = _c(ctx_len, np.int32)
    W = (T_cap + 31) // 32
    out = {
        "tokens": np.zeros((B, T_cap), np.int32), "parent": np.zeros((B, T_cap), np.int32),
        "depth": np.zeros((B, T_cap), np.int32), "pos_id": np.zeros((B, T_cap), np.int32),
        "branch_off": np.zeros((B, 2 * K + 1), np.int32), "mask": np.zeros((B, T_cap, W), np.uint32),
        "tree_len": np.zeros((B,), np.int32),
    }
    _load().d2sd_oracle_build_tree3(_p(draft1), _p(draft2), _p(draft3), _p(prefix_len), _p(third_len),
                                    _p(ctx_len), ctypes.c_int32(B), ctypes.c_int32(gamma), ctypes.c_int32(K),
                                    ctypes.c_int32(T_cap), _p(out["tokens"]), _p(out["parent"]),
                                    _p(out["depth"]), _p(out["pos_id"]), _p(out["branch_off"]),
                                    _p(out["mask"]), _p(out["tree_len"]))
    return out
