"""The C-ABI library loads and exports every symbol include/nhplan.h declares (no compute without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2306_01301_b200 import build
    return ctypes.CDLL(build.build())


def declared_symbols():
    src = "".join(open(os.path.join(ROOT, "include", f)).read() for f in sorted(os.listdir(os.path.join(ROOT, "include"))) if f.endswith(".h"))
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nhp_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    names = declared_symbols()
    assert len(names) >= 14
    for name in names:
        assert hasattr(lib, name), name
    from paper_2306_01301_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_query_sizes_is_pure_host_arithmetic():
    from paper_2306_01301_b200 import binding
    s = binding.query_sizes(9, 9, binding.FLAG_SOFT)
    assert (s.V_bytes, s.C_bytes, s.S_bytes) == (4 << 27, (1 << 27) // 8, 1 << 27)
    assert 3 << 27 <= s.workspace_bytes < (3 << 27) + (16 << 20)          # three curve-major copies of S + the footprint tables
    s0 = binding.query_sizes(10, 9, 0)
    assert (s0.V_bytes, s0.C_bytes, s0.S_bytes) == (4 << 29, (1 << 29) // 8, 0)
    assert 0 < s0.workspace_bytes < 32 << 20                                # footprint tables only
    # the level volumes of the reachability planner are part of the workspace: (levels + 4) N_R / 8 bytes
    s1 = binding.query_sizes(10, 9, 0, max_reach_levels=10)
    assert s1.workspace_bytes - s0.workspace_bytes == 14 * (1 << 29) // 8
    # a larger footprint limit costs more table space, and the limit is clamped to the grid
    assert binding.query_sizes(9, 9, 0, max_footprint_radius=128).workspace_bytes > binding.query_sizes(9, 9, 0).workspace_bytes
    assert binding.query_sizes(5, 5, 0, max_footprint_radius=500).workspace_bytes == binding.query_sizes(5, 5, 0, max_footprint_radius=15).workspace_bytes
    with pytest.raises(binding.NhpError) as e:
        binding.query_sizes(3, 9, 0)
    assert e.value.code == -2


def test_create_rejects_bad_arguments_before_touching_the_device(lib):
    from paper_2306_01301_b200 import binding as b
    L = b.load_library()
    w = b.Weights((ctypes.c_uint32 * 6)(*[8192] * 6), (ctypes.c_uint32 * 6)(*[256] * 6), 10, 0)
    bufs = b.Buffers(0x1000, 0x2000, None, 0x3000)
    h = ctypes.c_void_p()
    assert L.nhp_planner_create(ctypes.byref(h), 9, 8, 80.0, ctypes.byref(w), None, ctypes.byref(bufs), None) == -3
    assert L.nhp_planner_create(ctypes.byref(h), 4, 8, 8.0, ctypes.byref(w), None, ctypes.byref(bufs), None) == -2
    assert L.nhp_planner_create(ctypes.byref(h), 6, 6, 0.5, ctypes.byref(w), None, ctypes.byref(bufs), None) == -1
    nob = b.Buffers(None, None, None, None)
    assert L.nhp_planner_create(ctypes.byref(h), 6, 6, 8.0, ctypes.byref(w), None, ctypes.byref(nob), None) == -6
    now = b.Buffers(0x1000, 0x2000, None, None)                          # the workspace is required (footprint tables)
    assert L.nhp_planner_create(ctypes.byref(h), 6, 6, 8.0, ctypes.byref(w), None, ctypes.byref(now), None) == -6
    bad = b.Limits(-1, 0)
    assert L.nhp_planner_create(ctypes.byref(h), 6, 6, 8.0, ctypes.byref(w), ctypes.byref(bad), ctypes.byref(bufs), None) == -1
    assert L.nhp_planner_create(None, 6, 6, 8.0, ctypes.byref(w), None, ctypes.byref(bufs), None) == -1


def test_default_cycles_is_the_papers():
    """PAPER.md:392 "our default is 8 cycles" (tests/golden/paper_constants.txt) is what n_cycles <= 0 selects."""
    gold = dict(ln.split("#")[0].split() for ln in open(os.path.join(ROOT, "tests", "golden", "paper_constants.txt"))
                if len(ln.split("#")[0].split()) == 2)
    hdr = open(os.path.join(ROOT, "include", "nhplan.h")).read()
    assert int(re.search(r"#define NHP_DEFAULT_CYCLES (\d+)", hdr).group(1)) == int(gold["default_cycles"])
    from paper_2306_01301_b200 import binding
    assert binding.DEFAULT_CYCLES == int(gold["default_cycles"])


def test_product_path_never_touches_the_oracle():
    """The CUDA package must not import, link or execute anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2306_01301_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, re.M), f
                assert "nhp_oracle" not in txt and "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2306_01301_b200\b", txt, re.M), f
            assert "nhplan.h" not in txt and "libnhplan" not in txt, f
    sc = open(os.path.join(ROOT, "scenes", "__init__.py")).read()
    assert not re.search(r"^\s*(import|from)\s+(oracle|paper_2306_01301_b200)\b", sc, re.M)
