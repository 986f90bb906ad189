"""Pins of the oracle functions of the "next" rows (f1 KV commit, f2 third cascade
level, f3 confidence extraction) against things that are NOT the oracle (no GPU): torch.softmax in
fp64, closed forms, exact rational arithmetic, an independent page walk, the two-cycle invariant,
brute force over the 2K+1 flat candidate sequences.  Pin names P10..P12 follow DESIGN.md.
"""
import math
from fractions import Fraction

import numpy as np
import pytest
import torch

import d2sd_synth as synth


def _bits(x):
    return synth.f32_to_bf16_bits(np.asarray(x, np.float32))


def _f(bits):
    return synth.bf16_bits_to_f32(bits).astype(np.float64)


# ----------------------------------------------------------------------------- P10 confidence (f3)

def test_P10_confidence_vs_torch_softmax(oracle):
    """PAPER.md:87-89 Eq. 3: c_k = max_v softmax(logits_k)(v), t_k = argmax -- torch.softmax fp64."""
    rng = np.random.default_rng(310)
    for B, gamma, V, scale in ((3, 6, 50, 1.0), (2, 16, 1024, 3.0), (1, 4, 151936, 1.0), (2, 2, 7, 10.0)):
        logits = _bits(rng.standard_normal((B, gamma - 1, V)) * scale)
        anchor = rng.integers(0, V, (B,), dtype=np.int32)
        draft, conf = oracle.confidence(logits, anchor)
        p = torch.softmax(torch.from_numpy(_f(logits)), dim=-1)
        ref_c, ref_t = p.max(dim=-1)
        np.testing.assert_allclose(conf[:, 1:], ref_c.numpy(), rtol=1e-12)
        assert np.array_equal(draft[:, 1:], np.argmax(_f(logits), axis=-1))  # numpy: first occurrence
        assert np.array_equal(draft[:, 0], anchor) and (conf[:, 0] == 1.0).all()
        assert ((conf > 0) & (conf <= 1)).all()


def test_P10_confidence_closed_forms_and_ties(oracle):
    V = 1000
    lg = np.zeros((1, 3, V), np.float32)
    lg[0, 1, 17] = 2.0                      # one entry a, the rest 0: c = e^a / (e^a + V - 1)
    lg[0, 2, [5, 900]] = 3.0                # tie of two maxima: first index, c = e^3 / (2 e^3 + V - 2)
    draft, conf = oracle.confidence(_bits(lg), np.array([42], np.int32))
    assert draft[0].tolist() == [42, 0, 17, 5]          # constant row: first index 0
    np.testing.assert_allclose(conf[0, 1], 1.0 / V, rtol=1e-13)
    np.testing.assert_allclose(conf[0, 2], math.e ** 2 / (math.e ** 2 + V - 1), rtol=1e-13)
    np.testing.assert_allclose(conf[0, 3], math.e ** 3 / (2 * math.e ** 3 + V - 2), rtol=1e-13)
    lg = np.zeros((1, 1, 8), np.float32)
    lg[0, 0, 3] = -0.0                      # -0 == +0: still index 0
    lg[0, 0, :] -= 0.0
    assert oracle.confidence(_bits(lg), np.array([0], np.int32))[0][0, 1] == 0
    lg = np.full((1, 1, 64), -30.0, np.float32)
    lg[0, 0, 63] = 30.0                     # saturated: c -> 1, sum is 1 + 63 e^-60
    _, conf = oracle.confidence(_bits(lg), np.array([0], np.int32))
    np.testing.assert_allclose(conf[0, 1], 1.0 / (1.0 + 63 * math.exp(-60.0)), rtol=1e-15)


def test_P10_confidence_feeds_selection(oracle):
    """Eq. 3 -> Eq. 4/5 chain: the confidences (rounded to the fp32 the stage-(a) call takes) select the
    same prefixes as an exact-rational ranking of the same fp32 values."""
    rng = np.random.default_rng(311)
    gamma, K, V = 8, 3, 64
    logits = _bits(rng.standard_normal((20, gamma - 1, V)) * 4.0)
    _, conf = oracle.confidence(logits, np.zeros(20, np.int32))
    conf32 = conf.astype(np.float32)
    pl, _ = oracle.select_prefixes(conf32, K)
    for b in range(20):
        c = [Fraction(float(x)) for x in conf32[b]]
        r, P = [], Fraction(1)
        for i in range(gamma - 1):
            r.append(P * (1 - c[i + 1]))
            P *= c[i + 1]
        assert pl[b].tolist() == sorted(sorted(range(gamma - 1), key=lambda i: (-r[i], i))[:K])


# ----------------------------------------------------------------------------- P11 KV commit (f1)

def _cycle_case(oracle, rng, gamma, K, L, B, paged, ps=4, n_layers=2, Hq=4, Hkv=2, d=8, spare_pages=True):
    """One verification cycle at toy size: tree, per-layer tree K/V, caches with room to grow."""
    conf = rng.random((B, gamma), dtype=np.float32)
    pl, _ = oracle.select_prefixes(conf, K)
    V = 50
    d1 = rng.integers(0, V, (B, gamma), dtype=np.int32)
    d2 = rng.integers(0, V, (B, K, gamma), dtype=np.int32)
    ctx = rng.integers(L[0], L[1] + 1, (B,), dtype=np.int32)
    T_cap = synth.t_cap(gamma, K)
    tr = oracle.build_tree(d1, d2, pl, ctx, T_cap)
    tk = _bits(rng.standard_normal((n_layers, B, T_cap, Hkv, d)))
    tv = _bits(rng.standard_normal((n_layers, B, T_cap, Hkv, d)))
    q = _bits(rng.standard_normal((n_layers, B, T_cap, Hq, d)))
    cap = ctx + gamma + 2                   # room for a whole accepted block and a little more
    if paged:
        pages_cap = (cap + ps - 1) // ps
        P = int(pages_cap.sum()) + 5
        perm = rng.permutation(P).astype(np.int32)
        indptr = np.concatenate([[0], np.cumsum(pages_cap)]).astype(np.int32)
        indices = perm[:int(pages_cap.sum())].copy()
        free = perm[int(pages_cap.sum()):].copy()
        kc = _bits(rng.standard_normal((n_layers, P * ps, Hkv, d)))
        vc = _bits(rng.standard_normal((n_layers, P * ps, Hkv, d)))
        kv = dict(k_cache=kc, v_cache=vc, kv_indptr=indptr, kv_indices=indices, page_size=ps, free=free)
    else:
        indptr = np.concatenate([[0], np.cumsum(cap)]).astype(np.int32)
        kc = _bits(rng.standard_normal((n_layers, int(cap.sum()), Hkv, d)))
        vc = _bits(rng.standard_normal((n_layers, int(cap.sum()), Hkv, d)))
        kv = dict(k_cache=kc, v_cache=vc, kv_indptr=indptr, kv_indices=None, page_size=0, free=None)
    # acceptance: a random logits table with plants so that walks are non-trivial
    logits = _bits(rng.standard_normal((B, T_cap, V)))
    for b in range(B):
        for n in range(1, int(tr["tree_len"][b])):
            if rng.random() < 0.7:
                logits[b, tr["parent"][b, n], tr["tokens"][b, n]] = synth.PLANT_VALUE_BITS
    acc = oracle.accept(logits, tr["tokens"], tr["parent"], tr["depth"], tr["tree_len"], gamma)
    return dict(ctx=ctx, tr=tr, tk=tk, tv=tv, q=q, kv=kv, acc=acc, T_cap=T_cap, gamma=gamma)


def _rows_of(kv, indices, layer, b, n_rows):
    """Independent restatement of the addressing: the first n_rows cache rows of request b."""
    if kv["page_size"]:
        ps = kv["page_size"]
        pg = indices[kv["kv_indptr"][b]:kv["kv_indptr"][b + 1]]
        rows = (pg[:, None].astype(np.int64) * ps + np.arange(ps)[None, :]).reshape(-1)[:n_rows]
    else:
        rows = kv["kv_indptr"][b] + np.arange(n_rows)
    return rows


@pytest.mark.parametrize("paged", [False, True])
def test_P11_commit_bruteforce_and_untouched(oracle, paged):
    """rows L..L+accept_len of every layer's cache == tree rows of path[0..accept_len];
    every other byte of the caches is unchanged; ctx_len grows by accept_len + 1."""
    rng = np.random.default_rng(320 + paged)
    c = _cycle_case(oracle, rng, 8, 3, (0, 13), B=4, paged=paged)
    kv, acc = c["kv"], c["acc"]
    res = oracle.commit_kv(c["tk"], c["tv"], acc["path"], acc["accept_len"], c["ctx"], kv["k_cache"],
                           kv["v_cache"], kv["kv_indptr"], kv["kv_indices"], kv["page_size"])
    assert np.array_equal(res["ctx_len"], c["ctx"] + acc["accept_len"] + 1) and (res["dropped"] == 0).all()
    assert acc["accept_len"].max() >= 1, "case must accept something"
    touched = np.zeros(kv["k_cache"].shape[:2], bool)
    for layer in range(c["tk"].shape[0]):
        for b in range(4):
            L, n = int(c["ctx"][b]), int(acc["accept_len"][b]) + 1
            rows = _rows_of(kv, kv["kv_indices"], layer, b, L + n)
            nodes = acc["path"][b, :n]
            assert (nodes >= 0).all() and nodes[0] == 0
            assert np.array_equal(res["k_cache"][layer, rows[L:]], c["tk"][layer, b, nodes])
            assert np.array_equal(res["v_cache"][layer, rows[L:]], c["tv"][layer, b, nodes])
            touched[layer, rows[L:]] = True
    assert np.array_equal(res["k_cache"][~touched], kv["k_cache"][~touched])
    assert np.array_equal(res["v_cache"][~touched], kv["v_cache"][~touched])
    if paged:
        assert np.array_equal(res["kv_indices"], kv["kv_indices"])  # no free list: table untouched


@pytest.mark.parametrize("paged", [False, True])
def test_P11_two_cycle_invariant(oracle, paged):
    """The pin VERDICT asks for: attention of cycle n over prefix U accepted path == prefix-only attention
    of the same query over the committed cache of cycle n+1 (truncated behind the query's own position).
    The attention oracle is pinned on its own (P3, P5, P6); the commit is what this test pins."""
    rng = np.random.default_rng(330 + paged)
    c = _cycle_case(oracle, rng, 6, 2, (3, 9), B=3, paged=paged, n_layers=2)
    kv, acc, tr = c["kv"], c["acc"], c["tr"]
    res = oracle.commit_kv(c["tk"], c["tv"], acc["path"], acc["accept_len"], c["ctx"], kv["k_cache"],
                           kv["v_cache"], kv["kv_indptr"], kv["kv_indices"], kv["page_size"])
    for layer in range(2):
        before = oracle.attention(c["q"][layer], kv["k_cache"][layer], kv["v_cache"][layer], kv["kv_indptr"],
                                  kv["kv_indices"], kv["page_size"], c["ctx"], c["tk"][layer], c["tv"][layer],
                                  tr["mask"], tr["tree_len"])
        for b in range(3):
            for j in range(int(acc["accept_len"][b]) + 1):
                node = int(acc["path"][b, j])
                ctx_j = c["ctx"].copy()
                ctx_j[b] = c["ctx"][b] + j + 1      # committed rows up to and including path[j]
                sel = np.array([[b, node, h] for h in range(c["q"].shape[3])], np.int32)
                o, l = oracle.attention_rows(c["q"][layer], res["k_cache"][layer], res["v_cache"][layer],
                                             kv["kv_indptr"], res["kv_indices"], kv["page_size"], ctx_j,
                                             c["tk"][layer], c["tv"][layer], tr["mask"], sel, which="prefix")
                np.testing.assert_allclose(o, before[0][b, node], rtol=1e-12, atol=1e-13)
                np.testing.assert_allclose(l, before[1][b, node], rtol=1e-12, atol=1e-13)
    # and the chain continues: a second commit appends behind the first
    res2 = oracle.commit_kv(c["tk"], c["tv"], acc["path"], np.zeros_like(acc["accept_len"]), res["ctx_len"],
                            res["k_cache"], res["v_cache"], kv["kv_indptr"], res["kv_indices"], kv["page_size"])
    assert np.array_equal(res2["ctx_len"], res["ctx_len"] + 1)
    for b in range(3):
        row = _rows_of(kv, res2["kv_indices"], 0, b, int(res2["ctx_len"][b]))[-1]
        assert np.array_equal(res2["k_cache"][0, row], c["tk"][0, b, 0])


def test_P11_capacity_free_list_and_drops(oracle):
    """Reading G25: pages come from the free list in request order; what does not fit is dropped from the
    END of the path and reported."""
    rng = np.random.default_rng(340)
    gamma, ps, Hkv, d = 6, 4, 1, 4
    B, T_cap = 3, synth.t_cap(gamma, 0)
    ctx = np.array([4, 7, 2], np.int32)                 # pages in use: 1, 2, 1
    indptr = np.array([0, 3, 5, 8], np.int32)           # segment capacity: 3, 2, 3 pages
    indices = np.array([10, -1, -1, 11, 12, 13, -1, -1], np.int32)
    free = np.array([20, 21, 22], np.int32)
    path = np.tile(np.arange(gamma, dtype=np.int32), (B, 1))
    accept_len = np.array([4, 3, 5], np.int32)          # wants 5, 4, 6 rows
    tk = _bits(rng.standard_normal((1, B, T_cap, Hkv, d)))
    tv = _bits(rng.standard_normal((1, B, T_cap, Hkv, d)))
    kc = _bits(rng.standard_normal((1, 30 * ps, Hkv, d)))
    res = oracle.commit_kv(tk, tv, path, accept_len, ctx, kc, kc.copy(), indptr, indices, ps, free_pages=free)
    # request 0: rows 4..8 -> pages 1,2 of its segment: takes 20, 21.  request 1: rows 7..10 need page 2 of a
    # 2-page segment: capacity 8 rows -> 1 row fits, 3 dropped, no page taken.  request 2: rows 2..7 -> one more
    # page: takes 22.
    assert res["kv_indices"].tolist() == [10, 20, 21, 11, 12, 13, 22, -1]
    assert res["free_head"] == 3
    assert res["ctx_len"].tolist() == [9, 8, 8] and res["dropped"].tolist() == [0, 3, 0]
    assert np.array_equal(res["k_cache"][0, 20 * ps:20 * ps + 4], tk[0, 0, :4])     # positions 4..7
    assert np.array_equal(res["k_cache"][0, 21 * ps], tk[0, 0, 4])                  # position 8
    assert np.array_equal(res["k_cache"][0, 12 * ps + 3], tk[0, 1, 0])              # position 7 of request 1
    assert np.array_equal(res["k_cache"][0, 13 * ps + 2:13 * ps + 4], tk[0, 2, :2]) # positions 2,3
    assert np.array_equal(res["k_cache"][0, 22 * ps:22 * ps + 4], tk[0, 2, 2:6])    # positions 4..7
    # exhausted free list: the third request gets nothing and keeps only what its own page holds
    res = oracle.commit_kv(tk, tv, path, accept_len, ctx, kc, kc.copy(), indptr, indices, ps, free_pages=free[:2])
    assert res["ctx_len"].tolist() == [9, 8, 4] and res["dropped"].tolist() == [0, 3, 4] and res["free_head"] == 2
    # contiguous: the request's row range is the capacity
    res = oracle.commit_kv(tk, tv, path, accept_len, ctx, kc, kc.copy(), np.array([0, 8, 16, 24], np.int32), None, 0)
    assert res["ctx_len"].tolist() == [8, 8, 8] and res["dropped"].tolist() == [1, 3, 0]


def test_P11_gather_path(oracle):
    rng = np.random.default_rng(350)
    B, gamma, T_cap, F = 3, 5, 9, 6
    feat = _bits(rng.standard_normal((B, T_cap, F)))
    path = np.array([[0, 1, 2, -1, -1], [0, 5, 6, 7, 8], [0, -1, -1, -1, -1]], np.int32)
    al = np.array([2, 4, 0], np.int32)
    out = oracle.gather_path(feat, path, al)
    for b in range(B):
        for j in range(gamma):
            want = feat[b, path[b, j]] if j <= al[b] else np.zeros(F, np.uint16)
            assert np.array_equal(out[b, j], want)


# ----------------------------------------------------------------------------- P12 third level (f2)

def _exact_third(conf2_row, i, gamma):
    """Exact-rational Eq. 4 on the tail of a branch with prefix i (reading G22):
    candidates j' = 1..n-1, value (prod_{k<=j'} c_{i+k}) (1 - c_{i+j'+1})."""
    c = [Fraction(float(x)) for x in conf2_row]
    n = gamma - 1 - i
    out = {}
    for jp in range(1, n):
        P = Fraction(1)
        for k in range(1, jp + 1):
            P *= c[i + k]
        out[jp] = P * (1 - c[i + jp + 1])
    return out


def test_P12_select_third_vs_exact(oracle):
    rng = np.random.default_rng(360)
    for gamma, K in ((4, 2), (6, 4), (8, 3), (16, 4), (32, 8)):
        B = 40
        conf = rng.random((B, gamma), dtype=np.float32)
        pl, _ = oracle.select_prefixes(conf, K)
        conf2 = rng.random((B, K, gamma), dtype=np.float32)
        conf2[0] = rng.choice(np.array([0.0, 0.25, 0.5, 1.0], np.float32), (K, gamma))  # ties and zeros
        conf2[1] = 1.0                                                                   # every r = 0: pure tie-break
        third, r3 = oracle.select_third(conf2, pl)
        for b in range(B):
            for k in range(K):
                i = int(pl[b, k])
                ex = _exact_third(conf2[b, k], i, gamma)
                if not ex:                       # n_b = 1: nothing to extend ("up to" 2K+1 candidates)
                    assert i == gamma - 2 and third[b, k] == -1
                    continue
                best = min(ex, key=lambda jp: (-ex[jp], jp))
                assert third[b, k] == i + best
                assert i + 1 <= third[b, k] <= gamma - 2      # the set {1..gamma-2} of :228
                for jp, v in ex.items():
                    assert abs(r3[b, k, jp] - float(v)) <= 1e-15
                # telescoping over the whole tail: sum_{j'>=0} r(j') + prod = 1, with r(0) = 1 - c_{i+1}
                tail = conf2[b, k, i + 1:].astype(np.float64)
                assert abs((1 - tail[0]) + r3[b, k].sum() + np.prod(tail) - 1.0) <= 1e-12


def _rand_tree3(oracle, rng, gamma, K, B=3, V=1000, L=(0, 50), third=None):
    conf = rng.random((B, gamma), dtype=np.float32)
    pl, _ = oracle.select_prefixes(conf, K)
    conf2 = rng.random((B, K, gamma), dtype=np.float32)
    th, _ = oracle.select_third(conf2, pl)
    if third is not None:
        th = np.full_like(th, third)
    d1 = rng.integers(0, V, (B, gamma), dtype=np.int32)
    d2 = rng.integers(0, V, (B, K, gamma), dtype=np.int32)
    d3 = rng.integers(0, V, (B, K, gamma), dtype=np.int32)
    ctx = rng.integers(L[0], L[1] + 1, (B,), dtype=np.int32)
    T_cap = synth.t_cap3(gamma, K)
    return pl, th, d1, d2, d3, ctx, T_cap, oracle.build_tree3(d1, d2, d3, pl, th, ctx, T_cap)


def _row_bits(row):
    return [a for a in range(32 * len(row)) if (int(row[a // 32]) >> (a % 32)) & 1]


def test_P12_build_tree3_invariants_and_candidates(oracle):
    """Structure the paper fixes: T = gamma + sum (gamma-1-i) + sum (gamma-1-j); 2K+1 root-to-leaf
    candidates (fewer where a branch has no child), each a full block; candidate tokens by position are
    draft1[..i] ++ draft2[k][i+1..j] ++ draft3[k][j+1..]; mask row = ancestors by the parent array."""
    rng = np.random.default_rng(370)
    for gamma, K in ((4, 2), (6, 4), (16, 4), (16, 15), (32, 8), (3, 1)):
        pl, th, d1, d2, d3, ctx, T_cap, tr = _rand_tree3(oracle, rng, gamma, K, B=4)
        for b in range(4):
            T = int(tr["tree_len"][b])
            want_T = gamma + sum(gamma - 1 - int(i) for i in pl[b]) + sum(gamma - 1 - int(j) for j in th[b] if j >= 0)
            assert T == want_T <= T_cap
            par, dep, tok, boff = tr["parent"][b], tr["depth"][b], tr["tokens"][b], tr["branch_off"][b]
            assert boff[0] == gamma and boff[2 * K] == T and (np.diff(boff) >= 0).all()
            for n in range(T):
                bits = _row_bits(tr["mask"][b, n])
                assert len(bits) == dep[n] + 1 and max(bits) == n
                if n:
                    assert 0 <= par[n] < n and dep[n] == dep[par[n]] + 1
                    assert bits == sorted(_row_bits(tr["mask"][b, par[n]]) + [n])
                assert tr["pos_id"][b, n] == ctx[b] + dep[n]
            assert (tok[T:] == -1).all() and (tr["mask"][b, T:] == 0).all()
            leaves = sorted(set(range(T)) - set(par[:T].tolist()))
            n_third = int((th[b] >= 0).sum())
            assert len(leaves) == 1 + K + n_third <= 2 * K + 1
            seqs = set()
            for leaf in leaves:
                nodes = []
                a = leaf
                while a >= 0:
                    nodes.append(a)
                    a = par[a]
                nodes = nodes[::-1]
                assert len(nodes) == gamma           # every candidate runs to the block end
                seqs.add(tuple(int(tok[x]) for x in nodes))
            want = {tuple(int(x) for x in d1[b])}
            for k in range(K):
                i, j = int(pl[b, k]), int(th[b, k])
                want.add(tuple(int(x) for x in np.concatenate([d1[b, :i + 1], d2[b, k, i + 1:]])))
                if j >= 0:
                    want.add(tuple(int(x) for x in np.concatenate([d1[b, :i + 1], d2[b, k, i + 1:j + 1], d3[b, k, j + 1:]])))
            assert seqs == want


def test_P12_no_third_level_is_the_two_level_tree(oracle):
    rng = np.random.default_rng(380)
    gamma, K = 16, 4
    pl, th, d1, d2, d3, ctx, T_cap, tr3 = _rand_tree3(oracle, rng, gamma, K, third=-1)
    tr2 = oracle.build_tree(d1, d2, pl, ctx, T_cap)
    for name in ("tokens", "parent", "depth", "pos_id", "mask", "tree_len"):
        assert np.array_equal(tr3[name], tr2[name]), name
    assert np.array_equal(tr3["branch_off"][:, :K], tr2["branch_off"][:, :K])
    assert (tr3["branch_off"][:, K:] == tr2["tree_len"][:, None]).all()


def test_P12_flat_candidate_attention(oracle):
    """The 2K+1 candidates as FLAT sequences: causal attention over [prefix ++ sequence] (torch SDPA, fp64)
    == the depth-3 tree output at the node holding that position (the P3 pin on the deeper tree)."""
    rng = np.random.default_rng(390)
    gamma, K, L, Hq, Hkv, d = 6, 3, 5, 4, 2, 8
    pl, th, d1, d2, d3, ctx, T_cap, tr = _rand_tree3(oracle, rng, gamma, K, B=2, L=(L, L))
    B = 2
    q = _bits(rng.standard_normal((B, T_cap, Hq, d)))
    tk = _bits(rng.standard_normal((B, T_cap, Hkv, d)))
    tv = _bits(rng.standard_normal((B, T_cap, Hkv, d)))
    indptr = np.array([0, L, 2 * L], np.int32)
    kc = _bits(rng.standard_normal((2 * L, Hkv, d)))
    vc = _bits(rng.standard_normal((2 * L, Hkv, d)))
    out, lse = oracle.attention(q, kc, vc, indptr, None, 0, ctx, tk, tv, tr["mask"], tr["tree_len"])
    G, scale = Hq // Hkv, 1.0 / math.sqrt(d)
    assert (th >= 0).any()
    for b in range(B):
        T = int(tr["tree_len"][b])
        par = tr["parent"][b]
        for leaf in sorted(set(range(T)) - set(par[:T].tolist())):
            nodes, a = [], leaf
            while a >= 0:
                nodes.append(a)
                a = par[a]
            nodes = nodes[::-1]
            for h in range(Hq):
                g = h // G
                Kseq = np.concatenate([_f(kc[indptr[b]:indptr[b] + L, g]), _f(tk[b, nodes, g])])
                Vseq = np.concatenate([_f(vc[indptr[b]:indptr[b] + L, g]), _f(tv[b, nodes, g])])
                Qseq = _f(q[b, nodes, h])
                allow = np.concatenate([np.ones((gamma, L), bool), np.tril(np.ones((gamma, gamma), bool))], 1)
                ref = torch.nn.functional.scaled_dot_product_attention(
                    torch.from_numpy(Qseq)[None], torch.from_numpy(Kseq)[None], torch.from_numpy(Vseq)[None],
                    attn_mask=torch.from_numpy(allow)[None], scale=scale)[0].numpy()
                np.testing.assert_allclose(out[b, nodes, h], ref, rtol=1e-12, atol=1e-13)
