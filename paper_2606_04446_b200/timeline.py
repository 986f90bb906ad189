"""Per-CTA cycle breakdown of the fused cascade-attention kernel (a profiling aid, not part of the path).

    python -m paper_2606_04446_b200.timeline [config 1-4] [--ctas 0,5,17]

Builds a second copy of the library with -DD2SD_TIMELINE (libd2sd_timeline.so, in-tree), runs a few
layers of one single-request BASELINE.json config on random data with an L2 flush in between, and
prints the clock64 stamps the kernel recorded (attn_cascade_sm100.cu, TL / TLA / TLABS): prologue,
first MMA, start / end of the first 16 softmax units, epilogue, partial-state store, group wait,
merge, and the MMA issuer's wait accounting of slot 0.  Stamps are cycles since the CTA passed
griddepcontrol.wait; clock64 is per SM, so only differences inside one CTA mean anything.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import sys

import numpy as np
import torch

from . import binding, build

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(_HERE, "libd2sd_timeline.so")


def build_timeline_lib() -> str:
    newest = max(os.path.getmtime(f) for f in build.SOURCES + build.HEADERS)
    if not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        subprocess.check_call([os.environ.get("NVCC", "nvcc")] + build.NVCC_FLAGS + ["-DD2SD_TIMELINE"] +
                              build.SOURCES + ["-o", LIB])
    return LIB


def main(argv) -> None:
    cfg_no = int(argv[0]) if argv and argv[0].isdigit() else 2
    ctas = [0, 5, 17]
    if "--ctas" in argv:
        ctas = [int(x) for x in argv[argv.index("--ctas") + 1].split(",")]
    binding._LIB_PATH = build_timeline_lib()  # before the first call: the binding loads lazily
    binding._lib = None
    sys.path.insert(0, os.path.dirname(_HERE))  # the seeded input generators live at the repo root
    import d2sd_synth as synth
    from . import build_tree, cascade_verify_attn, cascade_workspace, select_prefixes

    cfg = synth.CONFIGS[cfg_no]
    assert cfg.B == 1 and not cfg.paged, "single-request contiguous configs only (1-4)"
    st = synth.make_step_inputs(cfg)
    i32 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).cuda()
    pl = select_prefixes(torch.from_numpy(st["conf"]).cuda(), cfg.K)
    tree = build_tree(i32(st["draft1"]), i32(st["draft2"]), pl, i32(st["ctx_len"]), cfg.T_cap)
    L = int(st["ctx_len"].max())
    q = torch.randn(1, cfg.T_cap, cfg.Hq, cfg.d, device="cuda").bfloat16()
    tk = torch.randn(1, cfg.T_cap, cfg.Hkv, cfg.d, device="cuda").bfloat16()
    tv = torch.randn_like(tk)
    layers = [(torch.randn(L, cfg.Hkv, cfg.d, device="cuda").bfloat16(),
               torch.randn(L, cfg.Hkv, cfg.d, device="cuda").bfloat16()) for _ in range(4)]
    ws = cascade_workspace(1, cfg.T_cap, cfg.Hq, cfg.Hkv, cfg.d, L, kv_rows=L)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(3):
        flush.zero_()
        for k, v in layers:
            cascade_verify_attn(q, k, v, None, None, i32(st["ctx_len"]), tk, tv, tree["mask"], tree["tree_len"], L,
                                workspace=ws)
    torch.cuda.synchronize()
    buf = np.zeros((256, 128), dtype=np.int64)
    assert ctypes.CDLL(LIB).d2sd_debug_timeline(buf.ctypes.data_as(ctypes.c_void_p)) == 0
    print(f"config {cfg_no}: T = {int(tree['tree_len'][0])}, L = {L}, {int((buf[:, 2] > 0).sum())} CTAs recorded "
          f"(index = blockIdx.x + gridDim.x * blockIdx.y)")
    for c in ctas:
        r = buf[c]
        if r[2] == 0:
            continue
        t0 = r[123]
        units = [(int(r[64 + 2 * n]), int(r[65 + 2 * n])) for n in range(16) if r[64 + 2 * n]]
        print(f"CTA {c}: prologue {r[0]}, all MMAs done {r[100]}, staged {r[102]}/{r[103]}, stored {r[101]}, "
              f"group complete {r[120]}, merge [lse {r[110] - t0}, rows {r[111] - t0}, done {r[113] - t0}], end {r[2]}")
        print(f"   softmax units (start, end): {units}")
        print("   MMA issuer of slot 0, cycles [tail, V wait, P wait, PV issue, commit, K wait, QK issue]: "
              f"{[int(x) for x in r[3:10]]}")


if __name__ == "__main__":
    main(sys.argv[1:])
