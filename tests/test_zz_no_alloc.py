"""d2sd_accept_static: the accept stage with the library's built-in scratch instead of a caller workspace
(include/d2sd.h).  Collected last on purpose (the run uses -x).  The new entry point is compared
with the existing path (d2sd_accept with a workspace) bit for bit -- every output of the stage is an integer --
on two calls in a row that share the scratch: the second call is a different, smaller problem, so the array
still holds the first call's chunk states when it runs."""
import ctypes

import numpy as np
import pytest
import torch

import d2sd_synth as synth
from helpers import bf16_cuda, i32_cuda

NAMES = ("argmax", "accept_len", "bonus", "best_node", "path")


@pytest.fixture(scope="module")
def d2sd():
    import paper_2606_04446_b200 as m
    m.lib()  # fails loudly if libd2sd.so is missing
    return m


def _case(d2sd, cfg):
    """Tree from the library's own select/build kernels, logits with planted acceptance, both accept paths."""
    st = synth.make_step_inputs(cfg)
    conf = torch.from_numpy(st["conf"]).cuda()
    pl = d2sd.select_prefixes(conf, cfg.K)
    tree = d2sd.build_tree(i32_cuda(st["draft1"]), i32_cuda(st["draft2"]), pl, i32_cuda(st["ctx_len"]), cfg.T_cap)
    torch.cuda.synchronize()
    host = {k: tree[k].cpu().numpy() for k in ("tokens", "parent", "depth", "tree_len")}
    logits = synth.make_logits(cfg)
    synth.plant_acceptance(cfg, logits, st["conf"], host["tokens"], host["parent"], host["depth"], host["tree_len"])
    lg = bf16_cuda(logits)
    args = (lg, tree["tokens"], tree["parent"], tree["depth"], tree["tree_len"], cfg.gamma)
    ref = d2sd.accept(*args)  # the existing path: caller workspace
    out = {"argmax": torch.full((cfg.B, cfg.T_cap), -7, dtype=torch.int32, device="cuda"),
           "path": torch.full((cfg.B, cfg.gamma), -7, dtype=torch.int32, device="cuda")}
    for name in ("accept_len", "bonus", "best_node"):
        out[name] = torch.full((cfg.B,), -7, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    got = d2sd.accept_static(*args, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the device's free memory"
    for name in NAMES:
        assert np.array_equal(got[name].cpu().numpy(), ref[name].cpu().numpy()), name
    return int(ref["accept_len"].sum())


@pytest.mark.gpu
def test_accept_static_matches_accept_on_two_calls_in_a_row(d2sd):
    big = synth.custom(90, B=4, gamma=16, K=4, V=151936)   # 4 x 70 rows x 10 chunks = 2800 chunk states
    small = synth.custom(91, B=2, gamma=8, K=3, V=20001)   # 2 x 26 rows x 2 chunks, ragged last chunk
    assert 4 * big.T_cap * 10 * 16 <= d2sd.accept_static_max_bytes()
    accepted = _case(d2sd, big)
    accepted += _case(d2sd, small)   # the scratch still holds the first call's states
    accepted += _case(d2sd, big)     # and back
    assert accepted > 0              # the planted acceptance made the walk do something


def test_accept_static_rejects_sizes_beyond_the_scratch(d2sd):
    """Rejected before anything is enqueued (no GPU needed): 64 x 1024 rows x 10 chunks x 16 B = 10 MiB."""
    L = d2sd.lib()
    vp = ctypes.c_void_p
    assert L.d2sd_accept_static_max_bytes() == 1 << 20
    st = L.d2sd_accept_static(vp(16), 151936, 151936, *([vp(16)] * 4), 64, 16, 1024, *([vp(16)] * 5), None)
    assert st == -2  # D2SD_ERR_UNSUPPORTED
    msg = d2sd.last_error()
    assert "d2sd_accept_static" in msg and "1048576" in msg and "d2sd_accept" in msg
