"""Host-side checks that need no GPU: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/d2sd.h declares; the argument validation that runs before any launch; the product
path has no CPU fallback and never touches oracle/."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def d2sd():
    from paper_2606_04446_b200 import build as b
    b.build()
    import paper_2606_04446_b200 as m
    return m


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "d2sd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(d2sd_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(d2sd):
    names = _declared_symbols()
    assert {"d2sd_select_prefixes", "d2sd_build_tree", "d2sd_cascade_verify_attn", "d2sd_accept",
            "d2sd_cascade_workspace_bytes", "d2sd_cascade_workspace_init", "d2sd_accept_workspace_bytes", "d2sd_last_error",
            "d2sd_version"} <= set(names)
    L = ctypes.CDLL(d2sd.lib_path())
    for n in names:
        assert hasattr(L, n), f"{n} declared in d2sd.h but not exported"


def test_version_and_workspace_queries(d2sd):
    assert "sm_100a" in d2sd.version()
    n = d2sd.cascade_workspace_bytes(1, 70, 32, 8, 128, 4096)
    assert n > 70 * 32 * 128 * 4 and n % 256 == 0
    assert d2sd.cascade_workspace_bytes(16, 70, 32, 8, 128, 16384, page_size=16) > n
    assert d2sd.accept_workspace_bytes(1, 70, 151936) >= 70 * 19 * 8
    for bad in (dict(d=64), dict(Hkv=7), dict(page_size=8), dict(T_cap=2000)):
        kw = dict(B=1, T_cap=70, Hq=32, Hkv=8, d=128, max_ctx_len=4096)
        kw.update(bad)
        with pytest.raises(d2sd.D2sdError):
            d2sd.cascade_workspace_bytes(**kw)
        assert d2sd.last_error()


def test_argument_validation_before_launch(d2sd):
    """Invalid arguments are rejected on the host, before any CUDA call (works without a GPU)."""
    L = d2sd.lib()
    vp = ctypes.c_void_p
    assert L.d2sd_select_prefixes(vp(16), 1, 1, 0, vp(16), None, None) == -1      # gamma < 2
    assert L.d2sd_select_prefixes(vp(16), 1, 16, 16, vp(16), None, None) == -1    # K > gamma-1
    assert L.d2sd_select_prefixes(None, 1, 16, 4, vp(16), None, None) == -1       # NULL conf
    assert b"conf" in L.d2sd_last_error()
    assert L.d2sd_select_prefixes(None, 0, 16, 4, None, None, None) == 0          # B = 0 is a no-op
    assert L.d2sd_build_tree(*([vp(16)] * 4), 1, 16, 4, 69, *([vp(16)] * 7), None) == -1   # T_cap too small
    assert L.d2sd_accept(vp(16), 100, 200, *([vp(16)] * 4), 1, 16, 70, *([vp(16)] * 6), 1 << 20, None) == -1


def test_product_path_is_isolated_from_the_oracle():
    """Neither side imports the other; the binding has no CPU fallback."""
    pkg = os.path.join(ROOT, "paper_2606_04446_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "d2sd_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2606_04446_b200" not in src.replace("under paper_2606_04446_b200/", "") or f.endswith(".c"), f
            assert not re.search(r"^\s*(from|import)\s+paper_2606_04446_b200", src, flags=re.M), f
            assert "#include \"d2sd.h\"" not in src and "common.cuh" not in src
    synth = open(os.path.join(ROOT, "d2sd_synth.py")).read()
    assert not re.search(r"^\s*(from|import)\s+(oracle|paper_2606_04446_b200)", synth, flags=re.M)


def test_missing_library_fails_loudly(monkeypatch, d2sd):
    from paper_2606_04446_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "_LIB_PATH", "/nonexistent/libd2sd.so")
    with pytest.raises(ImportError):
        binding.lib()
