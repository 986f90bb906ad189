"""GPU parity of the steps around the hot path: confidence extraction (f3), KV commit
(f1), third cascade level (f2) -- the CUDA path through the C ABI against the CPU oracle.

Integers, indices and copied bytes are bit-exact.  The confidences are fp32 sums of ex2.approx
exponentials: relative gate 2e-5 against the fp64 oracle (151 936 terms,
each exponential within 2^-22, tree sums in fp32); the SELECTION built on them is then checked
bit-exactly with the GPU-produced confidences fed to both sides.
"""
import numpy as np
import pytest
import torch

import d2sd_synth as synth
from helpers import bf16_cuda, check_rows, gpu_attention, i32_cuda, mask_cuda, valid_rows

pytestmark = pytest.mark.gpu
CONF_RTOL = 2e-5


@pytest.fixture(scope="module")
def d2sd():
    import paper_2606_04446_b200 as m
    m.lib()
    assert torch.cuda.is_available()
    return m


def _bits(x):
    return synth.f32_to_bf16_bits(np.asarray(x, np.float32))


# ------------------------------------------------------------------------------------------ f3

@pytest.mark.parametrize("B,gamma,V,scale,stride", [(1, 16, 151936, 1.0, None), (16, 16, 151936, 4.0, None),
                                                     (3, 6, 1000, 8.0, None), (2, 2, 7, 1.0, None),
                                                     (2, 8, 16385, 2.0, 16391), (1, 4, 32768, 1.0, 32776)])
def test_confidence_parity(d2sd, oracle, B, gamma, V, scale, stride):
    rng = np.random.default_rng(5000 + V + gamma)
    lg = rng.standard_normal((B, gamma - 1, V)).astype(np.float32) * scale
    if V >= 1000:
        lg[0, 0, [V - 1, 17]] = 20.0                # tie of two maxima, the later one in the last chunk
        lg[0, 1 % (gamma - 1), :] = 0.0             # constant row: c = 1/V, token 0
    bits = _bits(lg)
    anchor = rng.integers(0, V, (B,), dtype=np.int32)
    ref_d, ref_c = oracle.confidence(bits, anchor)
    t = bf16_cuda(bits)
    if stride is not None:                            # padded / misaligned row stride
        big = torch.zeros((B, gamma - 1, stride), dtype=torch.bfloat16, device="cuda")
        big[:, :, :V] = t
        t = big[:, :, :V]
    draft, conf = d2sd.draft_confidence(t, i32_cuda(anchor))
    torch.cuda.synchronize()
    assert np.array_equal(draft.cpu().numpy(), ref_d), "draft tokens (argmax) not bit-exact"
    c = conf.cpu().numpy().astype(np.float64)
    assert (c[:, 0] == 1.0).all()
    np.testing.assert_allclose(c, ref_c, rtol=CONF_RTOL, atol=0)
    # the selection on the GPU-produced confidences, same fp32 values on both sides: bit-exact
    K = min(4, gamma - 1)
    pl_ref, _ = oracle.select_prefixes(conf.cpu().numpy(), K)
    pl = d2sd.select_prefixes(conf, K)
    torch.cuda.synchronize()
    assert np.array_equal(pl.cpu().numpy(), pl_ref)


# ------------------------------------------------------------------------------------------ f1

def _commit_inputs(oracle, cfg, n_layers, rng, paged, spare=2, feat_F=0):
    """A verification cycle at reduced size with room to grow: oracle tree + planted acceptance."""
    st = synth.make_step_inputs(cfg)
    pl, _ = oracle.select_prefixes(st["conf"], cfg.K)
    tree = oracle.build_tree(st["draft1"], st["draft2"], pl, st["ctx_len"], cfg.T_cap)
    logits = synth.make_logits(cfg)
    synth.plant_acceptance(cfg, logits, st["conf"], tree["tokens"], tree["parent"], tree["depth"], tree["tree_len"], force=0.35)
    acc = oracle.accept(logits, tree["tokens"], tree["parent"], tree["depth"], tree["tree_len"], cfg.gamma)
    B, T_cap, Hkv, d = cfg.B, cfg.T_cap, cfg.Hkv, cfg.d
    tk = _bits(rng.standard_normal((n_layers, B, T_cap, Hkv, d)))
    tv = _bits(rng.standard_normal((n_layers, B, T_cap, Hkv, d)))
    ctx = st["ctx_len"].astype(np.int32)
    cap = ctx + cfg.gamma + spare
    if paged:
        ps = 16
        pages_cap = (cap + ps - 1) // ps
        P = int(pages_cap.sum()) + 12
        perm = rng.permutation(P).astype(np.int32)
        indptr = np.concatenate([[0], np.cumsum(pages_cap)]).astype(np.int32)
        indices = perm[:int(pages_cap.sum())].copy()
        free = perm[int(pages_cap.sum()):].copy()
        rows = P * ps
    else:
        ps, indices, free = 0, None, None
        indptr = np.concatenate([[0], np.cumsum(cap)]).astype(np.int32)
        rows = int(cap.sum())
    kc = _bits(rng.standard_normal((n_layers, rows, Hkv, d)))
    vc = _bits(rng.standard_normal((n_layers, rows, Hkv, d)))
    feat = _bits(rng.standard_normal((B, T_cap, feat_F))) if feat_F else None
    return dict(st=st, tree=tree, acc=acc, tk=tk, tv=tv, ctx=ctx, kc=kc, vc=vc, indptr=indptr, indices=indices,
                free=free, ps=ps, feat=feat)


def _run_commit(d2sd, c, use_free=False, accept_len=None, ctx=None, indices=None, kc=None, vc=None, head=0):
    al = c["acc"]["accept_len"] if accept_len is None else accept_len
    k = bf16_cuda(c["kc"] if kc is None else kc)
    v = bf16_cuda(c["vc"] if vc is None else vc)
    ind = c["indices"] if indices is None else indices
    ind_t = None if ind is None else i32_cuda(ind)
    ctx_t = i32_cuda(c["ctx"] if ctx is None else ctx)
    kw = {}
    if use_free:
        kw = dict(free_pages=i32_cuda(c["free"]), free_head=torch.tensor([head], dtype=torch.int32, device="cuda"))
    if c["feat"] is not None:
        kw["feat"] = bf16_cuda(c["feat"])
    res = d2sd.commit_kv(bf16_cuda(c["tk"]), bf16_cuda(c["tv"]), i32_cuda(c["acc"]["path"]), i32_cuda(al), ctx_t, k, v,
                         i32_cuda(c["indptr"]), ind_t, c["ps"], ctx_len_out=ctx_t, **kw)  # ctx_len updated IN PLACE
    torch.cuda.synchronize()
    out = dict(k=k.view(torch.int16).cpu().numpy().view(np.uint16), v=v.view(torch.int16).cpu().numpy().view(np.uint16),
               ctx=res[0].cpu().numpy(), dropped=res[1].cpu().numpy(),
               indices=None if ind_t is None else ind_t.cpu().numpy())
    if use_free:
        out["head"] = int(kw["free_head"].item())
    if c["feat"] is not None:
        out["feat"] = res[2].view(torch.int16).cpu().numpy().view(np.uint16)
    return out


@pytest.mark.parametrize("paged", [False, True])
@pytest.mark.parametrize("B,n_layers", [(1, 36), (16, 3)])
def test_commit_kv_byte_exact(d2sd, oracle, paged, B, n_layers):
    rng = np.random.default_rng(6000 + B + paged)
    cfg = synth.custom(96, B=B, gamma=16, K=4, ctx=(40, 300), paged=paged)
    c = _commit_inputs(oracle, cfg, n_layers, rng, paged, feat_F=256)
    assert c["acc"]["accept_len"].max() >= 1
    ref = oracle.commit_kv(c["tk"], c["tv"], c["acc"]["path"], c["acc"]["accept_len"], c["ctx"], c["kc"], c["vc"],
                           c["indptr"], c["indices"], c["ps"])
    got = _run_commit(d2sd, c)
    assert np.array_equal(got["ctx"], ref["ctx_len"]) and np.array_equal(got["dropped"], ref["dropped"])
    assert np.array_equal(got["k"], ref["k_cache"]) and np.array_equal(got["v"], ref["v_cache"])
    assert np.array_equal(got["feat"], oracle.gather_path(c["feat"], c["acc"]["path"], c["acc"]["accept_len"]))
    if paged:
        assert np.array_equal(got["indices"], ref["kv_indices"])


def test_commit_kv_free_list_and_drops(d2sd, oracle):
    """Pages from the free list in request order; a short list and full segments drop rows from the path's end."""
    rng = np.random.default_rng(6100)
    cfg = synth.custom(97, B=23, gamma=16, K=4, ctx=(1, 200), paged=True)
    c = _commit_inputs(oracle, cfg, 2, rng, True, spare=-9)   # some segments too small for a whole block
    # entries behind the pages in use are unassigned: poison them, the free list must provide
    ind = c["indices"].copy()
    for b in range(cfg.B):
        used = (int(c["ctx"][b]) + 15) // 16
        ind[c["indptr"][b] + used:c["indptr"][b + 1]] = -1
    c["free"] = c["free"][:9].copy()                           # only 9 pages to give, 2 of them already handed out
    al = np.full(cfg.B, cfg.gamma - 1, np.int32)              # everybody accepts the whole block
    path = np.tile(np.arange(cfg.gamma, dtype=np.int32), (cfg.B, 1))
    c["acc"] = dict(path=path, accept_len=al)
    ref = oracle.commit_kv(c["tk"], c["tv"], path, al, c["ctx"], c["kc"], c["vc"], c["indptr"], ind, 16,
                           free_pages=c["free"], free_head=2)
    got = _run_commit(d2sd, c, use_free=True, indices=ind, head=2)
    assert ref["dropped"].max() > 0 and (ref["dropped"] == 0).any()
    assert np.array_equal(got["ctx"], ref["ctx_len"]) and np.array_equal(got["dropped"], ref["dropped"])
    assert np.array_equal(got["indices"], ref["kv_indices"]) and got["head"] == ref["free_head"]
    assert np.array_equal(got["k"], ref["k_cache"]) and np.array_equal(got["v"], ref["v_cache"])


@pytest.mark.parametrize("paged", [False, True])
def test_two_cycles_chained_on_device(d2sd, oracle, paged):
    """Cycle n: select -> build -> attention -> accept -> commit, all on the device; cycle n+1 attends the
    committed cache.  Attention of cycle n+1 (GPU) == oracle attention over the oracle-committed cache, and
    the committed bytes are identical."""
    rng = np.random.default_rng(6200 + paged)
    cfg = synth.custom(98, B=4, gamma=16, K=4, ctx=(100, 900), paged=paged, V=1024)
    c = _commit_inputs(oracle, cfg, 1, rng, paged)
    st, tree = c["st"], c["tree"]
    # cycle n on the device
    pl = d2sd.select_prefixes(torch.from_numpy(st["conf"]).cuda(), cfg.K)
    tr = d2sd.build_tree(i32_cuda(st["draft1"]), i32_cuda(st["draft2"]), pl, i32_cuda(c["ctx"]), cfg.T_cap)
    logits = synth.make_logits(cfg)
    synth.plant_acceptance(cfg, logits, st["conf"], tree["tokens"], tree["parent"], tree["depth"], tree["tree_len"], force=0.35)
    acc = d2sd.accept(bf16_cuda(logits), tr["tokens"], tr["parent"], tr["depth"], tr["tree_len"], cfg.gamma)
    k, v = bf16_cuda(c["kc"]), bf16_cuda(c["vc"])
    ctx_t = i32_cuda(c["ctx"])
    ind_t = None if c["indices"] is None else i32_cuda(c["indices"])
    d2sd.commit_kv(bf16_cuda(c["tk"]), bf16_cuda(c["tv"]), acc["path"], acc["accept_len"], ctx_t, k, v,
                   i32_cuda(c["indptr"]), ind_t, c["ps"], ctx_len_out=ctx_t)
    torch.cuda.synchronize()
    ref = oracle.commit_kv(c["tk"], c["tv"], c["acc"]["path"], c["acc"]["accept_len"], c["ctx"], c["kc"], c["vc"],
                           c["indptr"], c["indices"], c["ps"])
    assert np.array_equal(ctx_t.cpu().numpy(), ref["ctx_len"])
    assert np.array_equal(k.view(torch.int16).cpu().numpy().view(np.uint16), ref["k_cache"])
    # cycle n+1: new tree inputs, attention over the committed cache (layer 0 of the [1,rows,Hkv,d] caches)
    cfg2 = synth.custom(99, B=4, gamma=16, K=4, ctx=(0, 0), paged=paged, V=1024)
    st2 = synth.make_step_inputs(cfg2)
    st2["ctx_len"] = ref["ctx_len"].copy()
    pl2, _ = oracle.select_prefixes(st2["conf"], cfg.K)
    tree2 = oracle.build_tree(st2["draft1"], st2["draft2"], pl2, st2["ctx_len"], cfg.T_cap)
    ti2 = synth.make_tree_inputs(cfg2)
    shape = (-1, 16, cfg.Hkv, cfg.d) if paged else (-1, cfg.Hkv, cfg.d)
    kv2 = dict(k_cache=k[0].view(torch.int16).cpu().numpy().view(np.uint16).reshape(shape),
               v_cache=v[0].view(torch.int16).cpu().numpy().view(np.uint16).reshape(shape),
               kv_indptr=c["indptr"], kv_indices=c["indices"], page_size=c["ps"])
    o, lse, _ = gpu_attention(d2sd, cfg2, st2, tree2, ti2, kv2)
    ro, rl = oracle.attention(ti2["q"], ref["k_cache"][0].reshape(shape), ref["v_cache"][0].reshape(shape), c["indptr"],
                              c["indices"], c["ps"], st2["ctx_len"], ti2["tree_k"], ti2["tree_v"], tree2["mask"],
                              tree2["tree_len"])
    vr = valid_rows(tree2["tree_len"], cfg.T_cap)
    check_rows(o[vr], lse[vr], ro[vr], rl[vr], "cycle n+1")


# ------------------------------------------------------------------------------------------ f2

@pytest.mark.parametrize("gamma,K", [(3, 1), (4, 2), (6, 4), (16, 4), (16, 15), (32, 8), (64, 3)])
def test_third_level_bit_exact(d2sd, oracle, gamma, K):
    rng = np.random.default_rng(7000 + gamma * 64 + K)
    B = 33
    conf = rng.random((B, gamma), dtype=np.float32)
    pl, _ = oracle.select_prefixes(conf, K)
    conf2 = rng.random((B, K, gamma), dtype=np.float32)
    conf2[0] = 1.0
    conf2[1] = rng.choice(np.array([0.0, 0.5, 1.0], np.float32), (K, gamma))
    th_ref, r3_ref = oracle.select_third(conf2, pl)
    r3 = torch.empty((B, K, gamma - 1), dtype=torch.float64, device="cuda")
    th = d2sd.select_third(torch.from_numpy(conf2).cuda(), i32_cuda(pl), r3_out=r3)
    torch.cuda.synchronize()
    assert np.array_equal(r3.cpu().numpy().view(np.uint64), r3_ref.view(np.uint64)), "r3 not bit-identical"
    assert np.array_equal(th.cpu().numpy(), th_ref)
    d1 = rng.integers(0, 151936, (B, gamma), dtype=np.int32)
    d2 = rng.integers(0, 151936, (B, K, gamma), dtype=np.int32)
    d3 = rng.integers(0, 151936, (B, K, gamma), dtype=np.int32)
    ctx = rng.integers(0, 40000, (B,), dtype=np.int32)
    for T_cap in (synth.t_cap3(gamma, K), synth.t_cap3(gamma, K) + 5):
        if T_cap > 1024:
            continue
        ref = oracle.build_tree3(d1, d2, d3, pl, th_ref, ctx, T_cap)
        got = d2sd.build_tree3(i32_cuda(d1), i32_cuda(d2), i32_cuda(d3), i32_cuda(pl), th, i32_cuda(ctx), T_cap)
        torch.cuda.synchronize()
        for name in ("tokens", "parent", "depth", "pos_id", "branch_off", "tree_len"):
            assert np.array_equal(got[name].cpu().numpy(), ref[name]), name
        assert np.array_equal(got["mask"].cpu().numpy().view(np.uint32), ref["mask"]), "mask"


def test_third_level_whole_path(d2sd, oracle):
    """Depth-3 tree through attention and acceptance: the three-range mask built on the device feeds
    d2sd_cascade_verify_attn and d2sd_accept unchanged ("jointly verifies in a single pass")."""
    rng = np.random.default_rng(7100)
    gamma, K, B, L = 16, 4, 2, 1500
    cfg = synth.custom(100, B=B, gamma=gamma, K=K, ctx=(L, L), V=1024)
    st = synth.make_step_inputs(cfg)
    pl, _ = oracle.select_prefixes(st["conf"], K)
    conf2 = rng.random((B, K, gamma), dtype=np.float32)
    d3 = rng.integers(0, cfg.V, (B, K, gamma), dtype=np.int32)
    T_cap = synth.t_cap3(gamma, K)
    th = d2sd.select_third(torch.from_numpy(conf2).cuda(), i32_cuda(pl))
    tr = d2sd.build_tree3(i32_cuda(st["draft1"]), i32_cuda(st["draft2"]), i32_cuda(d3), i32_cuda(pl), th,
                          i32_cuda(st["ctx_len"]), T_cap)
    torch.cuda.synchronize()
    th_ref, _ = oracle.select_third(conf2, pl)
    ref_tree = oracle.build_tree3(st["draft1"], st["draft2"], d3, pl, th_ref, st["ctx_len"], T_cap)
    assert int(ref_tree["tree_len"].max()) > synth.t_cap(gamma, K) - 10
    big = synth.custom(100, B=B, gamma=64, K=16, ctx=(L, L))
    ti = {k: v[:, :T_cap].copy() for k, v in synth.make_tree_inputs(big).items()}
    kv = synth.make_kv_cache(cfg, st["ctx_len"])
    tree_np = {"mask": tr["mask"].cpu().numpy().view(np.uint32), "tree_len": tr["tree_len"].cpu().numpy()}
    assert np.array_equal(tree_np["mask"], ref_tree["mask"])
    o, lse, _ = gpu_attention(d2sd, cfg, st, tree_np, ti, kv)
    ro, rl = oracle.attention(ti["q"], kv["k_cache"], kv["v_cache"], kv["kv_indptr"], None, 0, st["ctx_len"],
                              ti["tree_k"], ti["tree_v"], ref_tree["mask"], ref_tree["tree_len"])
    vr = valid_rows(ref_tree["tree_len"], T_cap)
    check_rows(o[vr], lse[vr], ro[vr], rl[vr], "depth-3 tree")
    logits = _bits(rng.standard_normal((B, T_cap, cfg.V)))
    for b in range(B):
        for n in range(1, int(ref_tree["tree_len"][b])):
            if rng.random() < 0.8:
                logits[b, ref_tree["parent"][b, n], ref_tree["tokens"][b, n]] = synth.PLANT_VALUE_BITS
    ref = oracle.accept(logits, ref_tree["tokens"], ref_tree["parent"], ref_tree["depth"], ref_tree["tree_len"], gamma)
    got = d2sd.accept(bf16_cuda(logits), tr["tokens"], tr["parent"], tr["depth"], tr["tree_len"], gamma)
    torch.cuda.synchronize()
    for name in ("argmax", "accept_len", "bonus", "best_node", "path"):
        assert np.array_equal(got[name].cpu().numpy(), ref[name]), name
