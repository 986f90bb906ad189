"""Seeded synthetic inputs for the D2SD verification hot path.

This module is shared by the tests, ``bench.py`` and ``__graft_entry__.smoke()``.
It holds NONE of the method's arithmetic (no r(i), no top-K, no tree build, no
attention, no argmax): it only draws random tensors of the shapes, sizes and
value distributions of BASELINE.json's five configs and lays them out in memory.
Neither ``oracle/`` nor the CUDA path is imported here.

The inputs stand in for the paper's Qwen3-8B workloads (gamma=16,
K=4 default; model only named, head shapes from BASELINE.json); the paper's
datasets, weights and drafters are not available, only their shapes are used.
The recipe is restated in DESIGN.md ("Input recipe").

bf16 tensors are carried as ``numpy.uint16`` bit patterns (round-to-nearest-even
from fp32) so that the CPU oracle and the GPU see bit-identical values.
"""
from __future__ import annotations

import dataclasses
from typing import Dict, List, Optional

import numpy as np

BASE_SEED = 26060444  # seed = 26060444 + config number

# Fixed ids for the per-tensor random streams (spawn order never changes).
_STREAM = {
    "conf": 1, "draft1": 2, "draft2": 3, "ctx_len": 4, "q": 5, "tree_k": 6,
    "tree_v": 7, "k_cache": 8, "v_cache": 9, "page_perm": 10, "logits": 11,
    "plant_u": 12, "pool_fill": 13,
}


@dataclasses.dataclass(frozen=True)
class Config:
    """One BASELINE.json config (shapes only)."""
    number: int
    name: str
    B: int            # requests
    layers: int       # attention layers per verification step
    gamma: int        # block size (position 0 = anchor)
    K: int            # re-anchored branches
    V: int            # vocabulary
    ctx: tuple        # (lo, hi) inclusive range the context lengths are drawn from
    paged: bool
    page_size: int = 16
    Hq: int = 32
    Hkv: int = 8
    d: int = 128

    @property
    def seed(self) -> int:
        return BASE_SEED + self.number

    @property
    def T_cap(self) -> int:
        return t_cap(self.gamma, self.K)

    @property
    def W(self) -> int:
        return (self.T_cap + 31) // 32


def t_cap(gamma: int, K: int) -> int:
    """Largest possible tree size: gamma trunk nodes + the K shortest distinct prefixes."""
    return gamma + K * (gamma - 1) - K * (K - 1) // 2


def t_cap3(gamma: int, K: int) -> int:
    """Largest depth-3 tree (third cascade level): t_cap plus, per branch, a third-level continuation
    anchored one token into the branch's tail (gamma-2-i nodes for prefix i)."""
    return t_cap(gamma, K) + K * (gamma - 2) - K * (K - 1) // 2


CONFIGS: Dict[int, Config] = {
    1: Config(1, "tiny", B=1, layers=1, gamma=16, K=2, V=1024, ctx=(256, 256), paged=False),
    2: Config(2, "qwen3-8b-step", B=1, layers=36, gamma=16, K=4, V=151936, ctx=(4096, 4096), paged=False),
    3: Config(3, "long-context", B=1, layers=36, gamma=16, K=4, V=151936, ctx=(32768, 32768), paged=False),
    4: Config(4, "wide-tree", B=1, layers=1, gamma=32, K=8, V=151936, ctx=(8192, 8192), paged=False),
    5: Config(5, "batched-paged", B=16, layers=1, gamma=16, K=4, V=151936, ctx=(1024, 16384), paged=True),
}


def custom(number: int, **kw) -> Config:
    """A config with overridden fields (reduced-size parity cases); seed follows ``number``."""
    base = dict(number=number, name="custom", B=1, layers=1, gamma=16, K=4, V=1024,
                ctx=(256, 256), paged=False)
    base.update(kw)
    return Config(**base)


def _rng(cfg: Config, stream: str, sub: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([cfg.seed, _STREAM[stream], sub])))


# --------------------------------------------------------------------------- bf16 carriers

def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit pattern, round-to-nearest-even (finite inputs)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def _normal_bf16(rng: np.random.Generator, shape, scale: float = 1.0, chunk: int = 1 << 24) -> np.ndarray:
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.uint16)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        x = rng.standard_normal(e - s, dtype=np.float32)
        if scale != 1.0:
            x *= np.float32(scale)
        out[s:e] = f32_to_bf16_bits(x)
    return out.reshape(shape)


# --------------------------------------------------------------------------- step-level inputs

def make_step_inputs(cfg: Config) -> Dict[str, np.ndarray]:
    """conf fp32 [B,gamma] ~ U(0,1) (slot 0 = anchor, ignored by the method), draft ids
    ~ U[0,V), ctx_len int32 [B] ~ U{lo..hi}."""
    conf = _rng(cfg, "conf").random((cfg.B, cfg.gamma), dtype=np.float32)
    draft1 = _rng(cfg, "draft1").integers(0, cfg.V, size=(cfg.B, cfg.gamma), dtype=np.int32)
    draft2 = _rng(cfg, "draft2").integers(0, cfg.V, size=(cfg.B, max(cfg.K, 1), cfg.gamma), dtype=np.int32)
    draft2 = draft2[:, :cfg.K, :].copy()
    lo, hi = cfg.ctx
    ctx_len = _rng(cfg, "ctx_len").integers(lo, hi + 1, size=(cfg.B,), dtype=np.int32)
    return {"conf": conf, "draft1": draft1, "draft2": draft2, "ctx_len": ctx_len}


def make_tree_inputs(cfg: Config, layer: int = 0, q_scale: float = 1.0) -> Dict[str, np.ndarray]:
    """Q [B,T_cap,Hq,d], tree K/V [B,T_cap,Hkv,d], bf16 bits, N(0,1) (Q optionally scaled:
    the 'peaked' set of SURVEY.md §8(c) uses q_scale=4)."""
    T = cfg.T_cap
    return {
        "q": _normal_bf16(_rng(cfg, "q", layer), (cfg.B, T, cfg.Hq, cfg.d), q_scale),
        "tree_k": _normal_bf16(_rng(cfg, "tree_k", layer), (cfg.B, T, cfg.Hkv, cfg.d)),
        "tree_v": _normal_bf16(_rng(cfg, "tree_v", layer), (cfg.B, T, cfg.Hkv, cfg.d)),
    }


def make_kv_cache(cfg: Config, ctx_len: np.ndarray, layer: int = 0,
                  pool_fill_nan: bool = False) -> Dict[str, Optional[np.ndarray]]:
    """Committed KV prefix for one layer, N(0,1) bf16.

    contiguous: k_cache/v_cache [sum L_b, Hkv, d], kv_indptr [B+1] token offsets.
    paged:      pool [P, page, Hkv, d] with P = ceil(1.25 * sum pages); page ids are a random
                permutation; kv_indptr [B+1] offsets into kv_indices; the tail page of each
                request is partially filled.  Slots no request owns hold N(0,1) values too, or
                NaN when ``pool_fill_nan`` (robustness case: they must never reach an output).
    """
    ctx_len = np.asarray(ctx_len, dtype=np.int64)
    if not cfg.paged:
        total = int(ctx_len.sum())
        indptr = np.zeros(cfg.B + 1, dtype=np.int32)
        indptr[1:] = np.cumsum(ctx_len)
        k = _normal_bf16(_rng(cfg, "k_cache", layer), (total, cfg.Hkv, cfg.d))
        v = _normal_bf16(_rng(cfg, "v_cache", layer), (total, cfg.Hkv, cfg.d))
        return {"k_cache": k, "v_cache": v, "kv_indptr": indptr, "kv_indices": None, "page_size": 0}
    ps = cfg.page_size
    pages = (ctx_len + ps - 1) // ps
    n_used = int(pages.sum())
    P = max(1, (n_used * 5 + 3) // 4)
    perm = _rng(cfg, "page_perm", layer).permutation(P).astype(np.int32)
    indices = perm[:n_used].copy()
    indptr = np.zeros(cfg.B + 1, dtype=np.int32)
    indptr[1:] = np.cumsum(pages)
    k = _normal_bf16(_rng(cfg, "k_cache", layer), (P, ps, cfg.Hkv, cfg.d))
    v = _normal_bf16(_rng(cfg, "v_cache", layer), (P, ps, cfg.Hkv, cfg.d))
    if pool_fill_nan:
        owned = np.zeros((P, ps), dtype=bool)
        for b in range(cfg.B):
            L = int(ctx_len[b])
            pg = indices[indptr[b]:indptr[b + 1]]
            owned[pg, :] = True
            if L % ps:
                owned[pg[-1], L % ps:] = False
        k[~owned] = 0x7FC0  # bf16 quiet NaN
        v[~owned] = 0x7FC0
    return {"k_cache": k, "v_cache": v, "kv_indptr": indptr, "kv_indices": indices, "page_size": ps}


def make_logits(cfg: Config, rows: Optional[int] = None) -> np.ndarray:
    """Target logits bf16 bits [B,T_cap,V] ~ N(0,1)."""
    T = cfg.T_cap if rows is None else rows
    return _normal_bf16(_rng(cfg, "logits"), (cfg.B, T, cfg.V))


PLANT_VALUE_BITS = 0x4180  # bf16(16.0): exact, above any N(0,1) sample


def plant_acceptance(cfg: Config, logits: np.ndarray, conf: np.ndarray, tokens: np.ndarray,
                     parent: np.ndarray, depth: np.ndarray, tree_len: np.ndarray,
                     force: Optional[float] = None) -> int:
    """Planted acceptance: with random logits and ids nothing is ever accepted.

    The tree (tokens/parent/depth/tree_len) is an INPUT here: a real target model consumes the
    tree and emits these logits.  Using the paper's calibration claim Pr(accept_k | prefix) ~= c_k
    (PAPER.md:91), for every non-root node n draw u ~ U(0,1) and, if u < conf[depth[n]], make the
    target "predict" it: logits[parent[n], tokens[n]] = 16.0.  Nodes are visited in index order; a
    parent that already carries a plant is skipped.  ``force`` replaces every u (0.0 = plant all
    first children, 1.0 = plant none).  Modifies ``logits`` in place; returns the number of plants.
    """
    rng = _rng(cfg, "plant_u")
    n_plants = 0
    for b in range(cfg.B):
        T = int(tree_len[b])
        u = rng.random(cfg.T_cap)
        planted = np.zeros(cfg.T_cap, dtype=bool)
        for n in range(1, T):
            p = int(parent[b, n])
            un = u[n] if force is None else force
            if planted[p] or not (un < float(conf[b, int(depth[b, n])])):
                continue
            logits[b, p, int(tokens[b, n])] = PLANT_VALUE_BITS
            planted[p] = True
            n_plants += 1
    return n_plants


def sample_rows(cfg: Config, tree_len: np.ndarray, n: int, salt: int = 0) -> np.ndarray:
    """n distinct-ish (b, t, h) triples with t < tree_len[b], for sampled parity at full size."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([cfg.seed, 99, salt])))
    out = np.empty((n, 3), dtype=np.int32)
    for i in range(n):
        b = int(rng.integers(0, cfg.B))
        out[i] = (b, int(rng.integers(0, int(tree_len[b]))), int(rng.integers(0, cfg.Hq)))
    return out
