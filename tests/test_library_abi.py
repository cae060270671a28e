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
    assert C.sizeof(B.Opts) == 4 * 8 + 10 * 4 + 8 + 2 * 4
    assert C.sizeof(B.CSource) == 8 + 6 * 8 + 4 * 8
    assert C.sizeof(B.RunStats) == 8 * 8 + 4 * 8 + 2 * 8 + 8 + 2 * 8 + 8


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


def test_setup_arithmetic_agrees_with_the_oracle_bit_for_bit(lib):
    """The library and the oracle derive the source frame and the composed transforms by their own code (hostmath.h's vector /
    matrix helpers vs the oracle's explicit loops); the definitions fix the order of
    the fp64 operations, so the rounded results must be equal bit for bit.  Host-only: needs no GPU."""
    import oracle
    from paper_1209_5235_b200 import binding as B, workloads as W
    rng = np.random.default_rng(12)
    axes = [(0, 0, 1.0), (1.0, 0, 0), (0, -2.0, 0), (1.0, 1.0, 1.0), (0.3, -0.3, 0.3), (1e-3, 5.0, -2.0)] + [tuple(rng.normal(size=3)) for _ in range(200)]
    for ax in axes:
        src = W.Source(W.SRC_CONE, (1.0, 2.0, 3.0), ax, W.E_MONO, 1.0, half_angle=0.1)
        for precision in (64, 32):
            a = B.host_source_frame(src, precision); b = oracle.source_frame(src, precision)
            assert np.array_equal(a, b), (ax, precision)
            if precision == 64:                      # and it is a right-handed orthonormal frame
                assert np.allclose(a @ a.T, np.eye(3), atol=1e-14) and np.allclose(np.cross(a[0], a[1]), a[2], atol=1e-14)
    for geom in (W.slab_geometry(1), W.detector_geometry(seed=4, n_phi=16, n_z=8, barrels=((200, 400), (450, 650))), W.lattice_geometry(4, seed=7),
                 W.cms_like_geometry()):
        M, T = B.host_compose_transforms(geom)
        Mo, To = oracle.OracleGeometry(geom).composed_transforms(64)
        assert np.array_equal(M, Mo) and np.array_equal(T, To), geom.name
    # the hook validates like gn_geometry_create
    g = W.slab_geometry(1)
    bad = W.Geometry(g.materials, g.solid_type, g.solid_params, g.placements[::-1].copy(), g.transforms)
    with pytest.raises(B.GammaNavError):
        B.host_compose_transforms(bad)
