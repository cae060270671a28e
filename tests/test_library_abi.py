"""The C-ABI library loads and exports every symbol include/gammanav.h declares (no compute without a GPU)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1209_5235_b200 import build, binding
    build.build()
    return binding.lib()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "gammanav.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gn_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert {"gn_geometry_create", "gn_nav_locate", "gn_nav_compute_step", "gn_transport_run"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    from paper_1209_5235_b200 import binding
    assert set(binding.EXPORTS) == set(names)


def test_struct_layouts_match_header():
    from paper_1209_5235_b200 import binding as B
    assert C.sizeof(B.Opts) == 4 * 8 + 8 * 4
    assert C.sizeof(B.CSource) == 8 + 6 * 8 + 4 * 8
    assert C.sizeof(B.RunStats) == 8 * 8 + 4 * 8 + 2 * 8 + 8 + 2 * 8


def test_no_cpu_fallback(lib):
    """Without a CUDA device the product path fails loudly instead of computing on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1209_5235_b200 import binding as B, workloads as W
    with pytest.raises(B.GammaNavError):
        B.Geometry(W.slab_geometry(1))
    with pytest.raises(B.GammaNavError):
        B.transport_run(None, W.slab_source(), 1, 10)


def test_argument_validation_needs_no_gpu(lib):
    h = C.c_void_p()
    assert lib.gn_geometry_create(None, 0, None, None, 0, None, 0, None, 0, None, C.byref(h)) == -1
    assert b"NULL" in lib.gn_last_error()
    assert lib.gn_nav_locate(None, 32, None, None, C.c_int64(0), None, None) == -1
    assert lib.gn_geometry_destroy(None) == 0
    assert lib.gn_version().startswith(b"gammanav")


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1209_5235_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert '#include "oracle' not in text and "liboracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1209_5235_b200" not in text.replace("paper_1209_5235_b200/csrc/", ""), f
            assert "gammanav.h\"" not in text.replace("include/gammanav.h", ""), f


def test_shard_ranges():
    from paper_1209_5235_b200.sharding import shard_range
    for n in (0, 1, 7, 10 ** 7 + 3):
        for w in (1, 2, 3, 8):
            spans = [shard_range(n, r, w) for r in range(w)]
            assert spans[0][0] == 0 and sum(c for _, c in spans) == n
            for (a, ca), (b, _) in zip(spans[:-1], spans[1:]):
                assert a + ca == b
            assert max(c for _, c in spans) - min(c for _, c in spans) <= 1
