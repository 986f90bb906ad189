"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test checks oracle/ against something that is NOT the oracle: exact rational arithmetic,
closed forms, special cases, brute force over the paper's K+1 flat candidate sequences, torch's
scaled_dot_product_attention in fp64, numpy.argmax.  Pin names P1..P9 follow DESIGN.md.
"""
import itertools
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


# ----------------------------------------------------------------------------- golden (paper)

def _golden():
    import os
    rows = []
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_shapes.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                name, g, k, v = line.split()
                rows.append((name, int(g), int(k), int(v)))
    return rows


def test_golden_paper_shapes(oracle):
    """counts the paper states for its figures."""
    for name, gamma, K, value in _golden():
        conf = np.linspace(0.9, 0.1, gamma, dtype=np.float32)[None]
        pl, r = oracle.select_prefixes(conf, K)
        if name == "n_prefix_candidates":
            # Fig. 2b (:115): K of the `value` candidate prefix lengths {0..gamma-2} are selected, all distinct and
            # in range, and the tree then holds gamma + sum_{i in S} (gamma-1-i) tokens (:107)
            assert len(set(pl[0].tolist())) == K and K < value
            assert set(pl[0].tolist()) <= set(range(value))
            tree = oracle.build_tree(np.zeros((1, gamma), np.int32), np.zeros((1, K, gamma), np.int32),
                                     pl, np.zeros(1, np.int32), synth.t_cap(gamma, K))
            assert int(tree["tree_len"][0]) == gamma + sum(gamma - 1 - int(i) for i in pl[0])
        elif name == "n_candidates":
            # "the K+1 candidates" (:124): the flattened tree has exactly K+1 root-to-leaf paths, each of them a
            # full block of gamma positions (every candidate runs to the block end, :107)
            tree = oracle.build_tree(np.zeros((1, gamma), np.int32), np.zeros((1, K, gamma), np.int32),
                                     pl, np.zeros(1, np.int32), synth.t_cap(gamma, K))
            T = int(tree["tree_len"][0])
            par = tree["parent"][0, :T]
            leaves = sorted(set(range(T)) - set(par.tolist()))
            assert len(leaves) == value
            assert all(int(tree["depth"][0, n]) == gamma - 1 for n in leaves)
        elif name.startswith("redraft_len_i"):
            i = int(name[len("redraft_len_i"):])
            pl = np.array([[i]], np.int32)
            tree = oracle.build_tree(np.zeros((1, gamma), np.int32), np.zeros((1, 1, gamma), np.int32),
                                     pl, np.zeros(1, np.int32), synth.t_cap(gamma, 1))
            assert int(tree["tree_len"][0]) - gamma == value


# ----------------------------------------------------------------------------- P1 / P2 select

def _exact_r(c):
    """Eq. 4 in exact rational arithmetic: r(i) = prod_{k<=i} c_k * (1 - c_{i+1})."""
    cf = [Fraction(float(x)) for x in c]
    out, P = [], Fraction(1)
    for i in range(len(c) - 1):
        out.append(P * (1 - cf[i + 1]))
        P *= cf[i + 1]
    return out, P


def test_P1_select_telescoping_and_exact(oracle):
    rng = np.random.default_rng(1)
    for gamma in (2, 3, 8, 16, 32, 64):
        conf = rng.random((50, gamma), dtype=np.float32)
        _, r = oracle.select_prefixes(conf, min(4, gamma - 1))
        assert (r >= 0).all()
        for b in range(conf.shape[0]):
            exact, prod = _exact_r(conf[b])
            # telescoping closed form (exact): sum_i r(i) + prod_k c_k = 1
            assert sum(exact) + prod == 1
            assert abs(math.fsum(r[b]) + float(prod) - 1.0) < 1e-15 * gamma
            for i, e in enumerate(exact):  # each r(i) within a few ulp of the exact rational
                assert abs(r[b, i] - float(e)) <= 4 * gamma * np.spacing(float(e)) + 1e-300


def test_P2_select_special_cases(oracle):
    gamma, K = 16, 4
    half = np.full((1, gamma), 0.5, np.float32)
    pl, r = oracle.select_prefixes(half, K)
    assert np.array_equal(r[0], 2.0 ** -(np.arange(gamma - 1) + 1.0))
    assert pl.tolist() == [[0, 1, 2, 3]]
    c = np.full((1, gamma), 0.7, np.float32)
    c[0, 1] = 0.0  # c_1 = 0: r(0)=1, all others exactly 0 -> ties broken towards smaller i
    pl, r = oracle.select_prefixes(c, K)
    assert r[0, 0] == 1.0 and (r[0, 1:] == 0).all() and pl.tolist() == [[0, 1, 2, 3]]
    c = np.zeros((1, gamma), np.float32)
    c[0, 1:4] = 1.0  # c = (.,1,1,1,0,...): exactly 3 accepted with probability 1
    pl, r = oracle.select_prefixes(c, 1)
    assert r[0, 3] == 1.0 and r[0].sum() == 1.0 and pl.tolist() == [[3]]
    # the anchor slot conf[.,0] is ignored (G9)
    a = np.random.default_rng(3).random((4, gamma), dtype=np.float32)
    b = a.copy()
    b[:, 0] = 0.123
    assert np.array_equal(oracle.select_prefixes(a, K)[0], oracle.select_prefixes(b, K)[0])
    # K = 0 is legal (G8) and K = gamma-1 returns every prefix length
    assert oracle.select_prefixes(a, 0)[0].shape == (4, 0)
    assert oracle.select_prefixes(a, gamma - 1)[0].tolist() == [list(range(gamma - 1))] * 4


def test_P2_select_exhaustive_grid_vs_exact_sort(oracle):
    vals = [0.0, 0.25, 0.5, 0.75, 1.0]
    for gamma in (2, 3, 4, 5, 6):
        grid = np.array(list(itertools.product(vals, repeat=gamma - 1)), np.float32)
        conf = np.concatenate([np.full((len(grid), 1), 0.5, np.float32), grid], axis=1)
        for K in range(0, gamma):
            pl, _ = oracle.select_prefixes(conf, K)
            for b in range(len(conf)):
                exact, _ = _exact_r(conf[b])
                want = sorted(sorted(range(gamma - 1), key=lambda i: (-exact[i], i))[:K])
                assert pl[b].tolist() == want, (gamma, K, conf[b])


def test_select_random_vs_exact_ranking(oracle):
    rng = np.random.default_rng(7)
    for gamma, K in ((16, 2), (16, 4), (32, 8)):
        conf = rng.random((300, gamma), dtype=np.float32)
        pl, _ = oracle.select_prefixes(conf, K)
        for b in range(conf.shape[0]):
            exact, _ = _exact_r(conf[b])
            want = sorted(sorted(range(gamma - 1), key=lambda i: (-exact[i], i))[:K])
            assert pl[b].tolist() == want


# ----------------------------------------------------------------------------- P4 build invariants

def _rand_tree(oracle, rng, gamma, K, B=3, V=1000, L=(0, 50)):
    conf = rng.random((B, gamma), dtype=np.float32)
    pl, _ = oracle.select_prefixes(conf, K)
    d1 = rng.integers(0, V, (B, gamma), dtype=np.int32)
    d2 = rng.integers(0, V, (B, K, gamma), dtype=np.int32)
    ctx = rng.integers(L[0], L[1] + 1, (B,), dtype=np.int32)
    T_cap = synth.t_cap(gamma, K)
    return conf, pl, d1, d2, ctx, T_cap, oracle.build_tree(d1, d2, pl, ctx, T_cap)


def _row_bits(row):
    return [a for a in range(32 * len(row)) if (int(row[a // 32]) >> (a % 32)) & 1]


def test_P4_build_invariants(oracle):
    rng = np.random.default_rng(11)
    for gamma, K in ((2, 0), (2, 1), (4, 2), (6, 4), (16, 0), (16, 2), (16, 4), (32, 8), (16, 15), (64, 3)):
        conf, pl, d1, d2, ctx, T_cap, tr = _rand_tree(oracle, rng, gamma, K)
        for b in range(d1.shape[0]):
            T = int(tr["tree_len"][b])
            assert T == gamma + sum(gamma - 1 - int(i) for i in pl[b]) <= T_cap
            boff = tr["branch_off"][b]
            assert boff[0] == gamma and boff[K] == T and (np.diff(boff) > 0).all()
            par, dep, tok = tr["parent"][b], tr["depth"][b], tr["tokens"][b]
            assert par[0] == -1 and dep[0] == 0
            assert np.array_equal(tok[:gamma], d1[b])
            for n in range(T):
                bits = _row_bits(tr["mask"][b, n])
                assert len(bits) == dep[n] + 1 and max(bits) == n
                if n > 0:
                    assert 0 <= par[n] < n and dep[n] == dep[par[n]] + 1
                    assert bits == _row_bits(tr["mask"][b, par[n]]) + [n]
                assert tr["pos_id"][b, n] == ctx[b] + dep[n]
            for n in range(gamma):  # trunk block is lower-triangular
                assert _row_bits(tr["mask"][b, n]) == list(range(n + 1))
            for k in range(K):      # closed form: trunk range 0..i_b plus branch range off_b..n
                i = int(pl[b, k])
                for n in range(boff[k], boff[k + 1]):
                    assert _row_bits(tr["mask"][b, n]) == list(range(i + 1)) + list(range(boff[k], n + 1))
                    assert tok[n] == d2[b, k, i + 1 + (n - boff[k])]
            # padding rows
            assert (tok[T:] == -1).all() and (par[T:] == -1).all() and (dep[T:] == 0).all()
            assert (tr["pos_id"][b, T:] == 0).all() and (tr["mask"][b, T:] == 0).all()


# ----------------------------------------------------------------------------- P3 / P5 / P6 attention

def _small_attn_case(oracle, rng, gamma, K, L, Hq=4, Hkv=2, d=8, B=2, paged=False, ps=4):
    conf, pl, d1, d2, ctx, T_cap, tr = _rand_tree(oracle, rng, gamma, K, B=B, L=(L, L))
    q = _bits(rng.standard_normal((B, T_cap, Hq, d)))
    tk = _bits(rng.standard_normal((B, T_cap, Hkv, d)))
    tv = _bits(rng.standard_normal((B, T_cap, Hkv, d)))
    if paged:
        pages = (ctx + ps - 1) // ps
        P = int(pages.sum()) + 3
        perm = rng.permutation(P).astype(np.int32)
        indices = perm[:int(pages.sum())]
        indptr = np.concatenate([[0], np.cumsum(pages)]).astype(np.int32)
        kc = _bits(rng.standard_normal((P, ps, Hkv, d)))
        vc = _bits(rng.standard_normal((P, ps, Hkv, d)))
        kv = dict(k_cache=kc, v_cache=vc, kv_indptr=indptr, kv_indices=indices, page_size=ps)
    else:
        indptr = np.concatenate([[0], np.cumsum(ctx)]).astype(np.int32)
        kc = _bits(rng.standard_normal((int(ctx.sum()), Hkv, d)))
        vc = _bits(rng.standard_normal((int(ctx.sum()), Hkv, d)))
        kv = dict(k_cache=kc, v_cache=vc, kv_indptr=indptr, kv_indices=None, page_size=0)
    return pl, ctx, T_cap, tr, q, tk, tv, kv


def _prefix_rows(kv, b, L, g):
    """Independent restatement of the KV addressing (contiguous rows or page table)."""
    if kv["page_size"]:
        ps = kv["page_size"]
        pg = kv["kv_indices"][kv["kv_indptr"][b]:kv["kv_indptr"][b + 1]]
        k = kv["k_cache"][pg].reshape(-1, *kv["k_cache"].shape[2:])[:L, g]
        v = kv["v_cache"][pg].reshape(-1, *kv["v_cache"].shape[2:])[:L, g]
    else:
        s = kv["kv_indptr"][b]
        k, v = kv["k_cache"][s:s + L, g], kv["v_cache"][s:s + L, g]
    return _f(k), _f(v)


@pytest.mark.parametrize("gamma,K,L,paged", [(4, 2, 5, False), (6, 4, 7, False), (6, 4, 0, False),
                                             (8, 3, 9, True), (4, 0, 6, False)])
def test_P3_flat_candidate_bruteforce(oracle, gamma, K, L, paged):
    """the K+1 candidates as FLAT sequences, ordinary causal attention over
    [prefix ++ sequence] per candidate (torch SDPA, fp64) == the tree output at the node holding
    that position.  Shapes of Fig. 1b (gamma=4,K=2) and Fig. 2b (gamma=6,K=4)."""
    rng = np.random.default_rng(100 + gamma * 10 + K)
    Hq, Hkv, d = 4, 2, 8
    pl, ctx, T_cap, tr, q, tk, tv, kv = _small_attn_case(oracle, rng, gamma, K, L, Hq, Hkv, d, paged=paged)
    out, lse = oracle.attention(q, kv["k_cache"], kv["v_cache"], kv["kv_indptr"], kv["kv_indices"],
                                kv["page_size"], ctx, tk, tv, tr["mask"], tr["tree_len"])
    G = Hq // Hkv
    scale = 1.0 / math.sqrt(d)
    for b in range(q.shape[0]):
        # node index of (candidate, position), restated from the layout reading G13
        offs, off = [], gamma
        for k in range(K):
            offs.append(off)
            off += gamma - 1 - int(pl[b, k])
        cands = [list(range(gamma))]
        for k in range(K):
            i = int(pl[b, k])
            cands.append(list(range(i + 1)) + [offs[k] + (p - i - 1) for p in range(i + 1, gamma)])
        for nodes in cands:
            for h in range(Hq):
                g = h // G
                kp, vp = _prefix_rows(kv, b, L, g)
                Kseq = np.concatenate([kp, _f(tk[b, nodes, g])])
                Vseq = np.concatenate([vp, _f(tv[b, nodes, g])])
                Qseq = _f(q[b, nodes, h])
                allow = np.concatenate([np.ones((gamma, L), bool), np.tril(np.ones((gamma, gamma), bool))], 1)
                ref = torch.nn.functional.scaled_dot_product_attention(
                    torch.from_numpy(Qseq)[None], torch.from_numpy(Kseq)[None], torch.from_numpy(Vseq)[None],
                    attn_mask=torch.from_numpy(allow)[None], scale=scale)[0].numpy()
                s = (Qseq @ Kseq.T) * scale
                s[~allow] = -np.inf
                ref_lse = torch.logsumexp(torch.from_numpy(s), dim=1).numpy()
                np.testing.assert_allclose(out[b, nodes, h], ref, rtol=1e-12, atol=1e-13)
                np.testing.assert_allclose(lse[b, nodes, h], ref_lse, rtol=1e-12, atol=1e-13)


def test_P5_cascade_merge_invariant(oracle):
    """merge(prefix state, tree state) == single-pass attention over prefix U allowed tree keys."""
    rng = np.random.default_rng(5)
    for L, paged in ((0, False), (1, False), (37, False), (50, True)):
        pl, ctx, T_cap, tr, q, tk, tv, kv = _small_attn_case(oracle, rng, 8, 3, L, paged=paged)
        args = (q, kv["k_cache"], kv["v_cache"], kv["kv_indptr"], kv["kv_indices"], kv["page_size"],
                ctx, tk, tv, tr["mask"], tr["tree_len"])
        of, lf = oracle.attention(*args, which="full")
        op, lp = oracle.attention(*args, which="prefix")
        ot, lt = oracle.attention(*args, which="tree")
        for b in range(q.shape[0]):
            T = int(tr["tree_len"][b])
            m = np.maximum(lp[b, :T], lt[b, :T])
            wp, wt = np.exp(lp[b, :T] - m), np.exp(lt[b, :T] - m)
            merged = (wp[..., None] * op[b, :T] + wt[..., None] * ot[b, :T]) / (wp + wt)[..., None]
            np.testing.assert_allclose(merged, of[b, :T], rtol=1e-12, atol=1e-13)
            np.testing.assert_allclose(m + np.log(wp + wt), lf[b, :T], rtol=1e-12, atol=1e-13)
            if L == 0:  # empty prefix (G16): state (0, -inf) and the full result is the tree state
                assert np.isneginf(lp[b, :T]).all() and (op[b, :T] == 0).all()
                np.testing.assert_array_equal(of[b, :T], ot[b, :T])
            assert np.isnan(of[b, T:]).all()  # padding rows untouched


def test_P5_split_associativity(oracle):
    """Splitting the prefix anywhere and LSE-merging the parts reproduces the prefix-only state."""
    rng = np.random.default_rng(6)
    L = 40
    pl, ctx, T_cap, tr, q, tk, tv, kv = _small_attn_case(oracle, rng, 6, 2, L, B=1)
    base = (q, kv["k_cache"], kv["v_cache"], None, None, 0)
    rest = (tk, tv, tr["mask"], tr["tree_len"])
    op, lp = oracle.attention(*base, ctx, *rest, which="prefix")
    T = int(tr["tree_len"][0])
    for cut in (1, 13, 39):
        o1, l1 = oracle.attention(q, kv["k_cache"][:cut], kv["v_cache"][:cut], None, None, 0,
                                  np.array([cut], np.int32), *rest, which="prefix")
        o2, l2 = oracle.attention(q, kv["k_cache"][cut:], kv["v_cache"][cut:], None, None, 0,
                                  np.array([L - cut], np.int32), *rest, which="prefix")
        m = np.maximum(l1[0, :T], l2[0, :T])
        w1, w2 = np.exp(l1[0, :T] - m), np.exp(l2[0, :T] - m)
        merged = (w1[..., None] * o1[0, :T] + w2[..., None] * o2[0, :T]) / (w1 + w2)[..., None]
        np.testing.assert_allclose(merged, op[0, :T], rtol=1e-12, atol=1e-13)


def test_P6_chain_equals_sdpa(oracle):
    """K=0: the tree is the draft-1 chain -> plain causal attention with a fully visible prefix."""
    rng = np.random.default_rng(8)
    gamma, L, Hq, Hkv, d = 8, 100, 8, 2, 16
    pl, ctx, T_cap, tr, q, tk, tv, kv = _small_attn_case(oracle, rng, gamma, 0, L, Hq, Hkv, d, B=1)
    out, lse = oracle.attention(q, kv["k_cache"], kv["v_cache"], kv["kv_indptr"], None, 0, ctx, tk, tv,
                                tr["mask"], tr["tree_len"])
    G = Hq // Hkv
    Kall = np.concatenate([_f(kv["k_cache"]), _f(tk[0])]).transpose(1, 0, 2).repeat(G, axis=0)
    Vall = np.concatenate([_f(kv["v_cache"]), _f(tv[0])]).transpose(1, 0, 2).repeat(G, axis=0)
    Q = _f(q[0]).transpose(1, 0, 2)
    allow = np.concatenate([np.ones((gamma, L), bool), np.tril(np.ones((gamma, gamma), bool))], 1)
    ref = torch.nn.functional.scaled_dot_product_attention(
        torch.from_numpy(Q), torch.from_numpy(Kall), torch.from_numpy(Vall),
        attn_mask=torch.from_numpy(allow)).numpy().transpose(1, 0, 2)
    np.testing.assert_allclose(out[0], ref, rtol=1e-12, atol=1e-13)


def test_attention_rows_matches_full(oracle):
    rng = np.random.default_rng(9)
    pl, ctx, T_cap, tr, q, tk, tv, kv = _small_attn_case(oracle, rng, 8, 3, 21, paged=True)
    args = (q, kv["k_cache"], kv["v_cache"], kv["kv_indptr"], kv["kv_indices"], kv["page_size"], ctx,
            tk, tv, tr["mask"])
    for which in ("full", "prefix", "tree"):
        of, lf = oracle.attention(*args, tr["tree_len"], which=which)
        sel = np.array([(b, t, h) for b in range(2) for t in range(int(tr["tree_len"][b])) for h in (0, 3)], np.int32)
        o, l = oracle.attention_rows(*args, sel, which=which)
        np.testing.assert_array_equal(o, of[sel[:, 0], sel[:, 1], sel[:, 2]])
        np.testing.assert_array_equal(l, lf[sel[:, 0], sel[:, 1], sel[:, 2]])


def test_sm_scale_and_uniform_values(oracle):
    """Closed forms: all-equal keys -> O = mean of V rows, LSE = s + ln(n); scale enters linearly."""
    gamma, L, Hq, Hkv, d = 4, 16, 2, 1, 8
    tr = oracle.build_tree(np.zeros((1, gamma), np.int32), np.zeros((1, 0, gamma), np.int32),
                           np.zeros((1, 0), np.int32), np.array([L], np.int32), gamma)
    q = _bits(np.ones((1, gamma, Hq, d)))
    kc = _bits(np.full((L, Hkv, d), 0.5))
    rng = np.random.default_rng(2)
    vc = _bits(rng.standard_normal((L, Hkv, d)))
    tk = _bits(np.full((1, gamma, Hkv, d), 0.5))
    tv = _bits(rng.standard_normal((1, gamma, Hkv, d)))
    for scale in (0.25, 1.0):
        out, lse = oracle.attention(q, kc, vc, None, None, 0, np.array([L], np.int32), tk, tv, tr["mask"],
                                    tr["tree_len"], sm_scale=scale)
        for t in range(gamma):
            n = L + t + 1
            want = (_f(vc[:, 0]).sum(0) + _f(tv[0, :t + 1, 0]).sum(0)) / n
            np.testing.assert_allclose(out[0, t, 0], want, rtol=1e-13, atol=1e-14)
            assert abs(lse[0, t, 1] - (0.5 * d * scale + math.log(n))) < 1e-13


# ----------------------------------------------------------------------------- P7 / P8 / P9 accept

def test_P9_argmax_first_index_and_ties(oracle):
    rng = np.random.default_rng(12)
    B, T, V = 2, 5, 3000
    logits = _bits(rng.standard_normal((B, T, V)))
    tl = np.array([T, 3], np.int32)
    logits[0, 1, 17] = 0x4180
    logits[0, 1, 2999] = 0x4180     # planted tie: first index wins
    logits[0, 1, 900] = 0x4180
    logits[0, 2, :] = 0x8000        # all -0.0 ...
    logits[0, 2, 5] = 0x0000        # ... and one +0.0: IEEE-equal -> index 0
    logits[1, 0, :] = 0xC000        # constant row -> index 0
    logits[1, 1, V - 1] = 0x4200    # maximum at the last index
    a = oracle.argmax(logits, tl)
    ref = np.argmax(synth.bf16_bits_to_f32(logits), axis=-1)  # numpy: first occurrence
    for b in range(B):
        assert np.array_equal(a[b, :tl[b]], ref[b, :tl[b]])
        assert (a[b, tl[b]:] == -1).all()
    assert a[0, 1] == 17 and a[0, 2] == 0 and a[1, 0] == 0 and a[1, 1] == V - 1


def _linear_accept(seq_tokens, seq_pred):
    """PAPER.md:69 linear rule: accept draft tokens up to (not including) the first mismatch.
    seq_pred[p] = target's prediction after position p."""
    n = 0
    for p in range(1, len(seq_tokens)):
        if seq_tokens[p] != seq_pred[p - 1]:
            break
        n += 1
    return n


def test_P7_P8_accept_vs_flat_candidates(oracle):
    rng = np.random.default_rng(13)
    V = 12  # tiny vocabulary: frequent accidental matches, duplicate siblings (G12, G17)
    for gamma, K in ((4, 2), (6, 4), (16, 4), (16, 0), (8, 7)):
        for trial in range(40):
            conf, pl, d1, d2, ctx, T_cap, tr = _rand_tree(oracle, rng, gamma, K, B=2, V=V)
            a = rng.integers(0, V, (2, T_cap), dtype=np.int32)
            if trial % 4 == 0:  # walk some way down by construction
                for b in range(2):
                    for n in range(1, int(tr["tree_len"][b])):
                        if rng.random() < 0.8:
                            a[b, tr["parent"][b, n]] = tr["tokens"][b, n]
            res = oracle.accept_walk(a, tr["tokens"], tr["parent"], tr["depth"], tr["tree_len"], gamma)
            for b in range(2):
                offs, off = [], gamma
                for k in range(K):
                    offs.append(off)
                    off += gamma - 1 - int(pl[b, k])
                cands = [list(range(gamma))]
                for k in range(K):
                    i = int(pl[b, k])
                    cands.append(list(range(i + 1)) + [offs[k] + (p - i - 1) for p in range(i + 1, gamma)])
                lens = [_linear_accept([tr["tokens"][b, n] for n in nodes], [a[b, n] for n in nodes])
                        for nodes in cands]
                best = max(lens)
                assert res["accept_len"][b] == best           # P8: max over candidates
                if K == 0:
                    assert res["accept_len"][b] == lens[0]    # P7: K=0 is the linear rule
                # winning node: smallest node index among candidates reaching the best length (G17)
                want_node = min(nodes[best] for nodes, ln in zip(cands, lens) if ln == best)
                assert res["best_node"][b] == want_node
                assert res["bonus"][b] == a[b, want_node]
                path = res["path"][b]
                assert (path[best + 1:] == -1).all() and path[0] == 0 and path[best] == want_node
                for j in range(1, best + 1):
                    assert tr["parent"][b, path[j]] == path[j - 1]


def test_P7_accept_special_cases(oracle):
    rng = np.random.default_rng(14)
    gamma, K, V = 16, 4, 50000
    conf, pl, d1, d2, ctx, T_cap, tr = _rand_tree(oracle, rng, gamma, K, B=1, V=V)
    T = int(tr["tree_len"][0])
    # every node's token equals the target argmax at its parent -> full acceptance, trunk leaf wins
    a = np.zeros((1, T_cap), np.int32)
    tok = tr["tokens"].copy()
    for n in range(1, T):
        tok[0, n] = 7  # all drafts identical => every child equals a[parent] = 7
    a[:] = 7
    res = oracle.accept_walk(a, tok, tr["parent"], tr["depth"], tr["tree_len"], gamma)
    assert res["accept_len"][0] == gamma - 1 and res["best_node"][0] == gamma - 1
    assert res["path"][0].tolist() == list(range(gamma))
    # nothing matches -> accept_len 0, bonus = argmax at the root
    a = np.full((1, T_cap), V + 5, np.int32)
    a[0, 0] = 4242
    res = oracle.accept_walk(a, tr["tokens"], tr["parent"], tr["depth"], tr["tree_len"], gamma)
    assert res["accept_len"][0] == 0 and res["bonus"][0] == 4242 and res["best_node"][0] == 0
    assert res["path"][0].tolist() == [0] + [-1] * (gamma - 1)
    # an unaccepted parent blocks its matching child
    a = np.full((1, T_cap), -7, np.int32)
    a[0, 1] = tr["tokens"][0, 2]
    res = oracle.accept_walk(a, tr["tokens"], tr["parent"], tr["depth"], tr["tree_len"], gamma)
    assert res["accept_len"][0] == 0


def test_plant_acceptance_forces(oracle):
    """Generator harness: force=0 plants every first child -> long walks; force=1 plants nothing."""
    cfg = synth.CONFIGS[1]
    st = synth.make_step_inputs(cfg)
    pl, _ = oracle.select_prefixes(st["conf"], cfg.K)
    tr = oracle.build_tree(st["draft1"], st["draft2"], pl, st["ctx_len"], cfg.T_cap)
    conf1 = np.ones_like(st["conf"])
    logits = synth.make_logits(cfg)
    n = synth.plant_acceptance(cfg, logits, conf1, tr["tokens"], tr["parent"], tr["depth"], tr["tree_len"], force=0.0)
    assert n > 0
    res = oracle.accept(logits, tr["tokens"], tr["parent"], tr["depth"], tr["tree_len"], cfg.gamma)
    assert res["accept_len"][0] == cfg.gamma - 1
    logits = synth.make_logits(cfg)
    assert synth.plant_acceptance(cfg, logits, st["conf"], tr["tokens"], tr["parent"], tr["depth"],
                                  tr["tree_len"], force=1.0) == 0
