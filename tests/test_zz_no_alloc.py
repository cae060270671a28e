"""gn_nav_compute_step_noalloc (scratch in a fixed device array, no allocation inside the library) against the existing
gn_nav_compute_step on the same seeded queries: step lengths and next-volume indices bit for bit (the tolerance of the
navigation tests in test_gpu_parity.py), on two calls in a row -- the second call finds the first one's counters, keys and
work order in the shared array.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_1209_5235_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_1209_5235_b200 import build, binding
    build.build()
    return binding


def _same_bits(a, b):
    return np.array_equal(a.cpu().numpy().view(np.uint8), b.cpu().numpy().view(np.uint8))


def _queries(B, geom, n, seed, dtype):
    import torch
    pos, dirs = W.nav_queries(geom, n, seed=seed, dtype=dtype)
    return torch.from_numpy(pos).cuda(), torch.from_numpy(dirs).cuda()


@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("name", ["detector", "cmslike", "phantom12"])
def test_noalloc_step_equals_the_existing_path_twice(B, name, precision):
    """General geometries (tubes, rotations: the query sort uses the scratch array) and a coherent one (no scratch)."""
    import torch
    geom = {"detector": lambda: W.detector_geometry(seed=4, n_phi=16, n_z=8, barrels=((200, 400), (450, 650))),
            "cmslike": lambda: W.cms_like_geometry(),
            "phantom12": lambda: W.phantom_geometry(12, 2.0, seed=3, world_half=20.0)}[name]()
    geo = B.Geometry(geom)
    dt = np.float32 if precision == 32 else np.float64
    tdt = torch.float32 if precision == 32 else torch.float64
    # two batches of different sizes and seeds: the second call must not see anything of the first
    for n, seed in ((200_000, 21), (70_001, 22)):
        pos, dirs = _queries(B, geom, n, seed, dt)
        vol = B.nav_locate(geo, pos, dirs)
        ref_step, ref_next = B.nav_compute_step(geo, pos, dirs, vol)
        out = (torch.full((n,), -7.0, dtype=tdt, device="cuda"), torch.full((n,), -7, dtype=torch.int32, device="cuda"))
        B.nav_compute_step_noalloc(geo, pos, dirs, vol, out)
        torch.cuda.synchronize()
        assert torch.equal(out[1], ref_next)
        assert _same_bits(out[0], ref_step)
        assert (ref_next >= -1).all() and int((ref_next >= 0).sum()) > n // 100        # the batch does real work


def test_noalloc_step_with_max_step_and_at_the_size_limit(B):
    import torch
    geom = W.detector_geometry(seed=4, n_phi=16, n_z=8, barrels=((200, 400), (450, 650)))
    geo = B.Geometry(geom)
    n = B.NOALLOC_MAX_QUERIES
    pos, dirs = _queries(B, geom, n, 23, np.float32)
    vol = B.nav_locate(geo, pos, dirs)
    ms = torch.full((n,), 150.0, dtype=torch.float32, device="cuda")
    for _ in range(2):                                                     # two calls in a row on the same inputs
        ref = B.nav_compute_step(geo, pos, dirs, vol, max_step=ms)
        out = (torch.empty(n, dtype=torch.float32, device="cuda"), torch.empty(n, dtype=torch.int32, device="cuda"))
        B.nav_compute_step_noalloc(geo, pos, dirs, vol, out, max_step=ms)
        assert torch.equal(out[1], ref[1]) and _same_bits(out[0], ref[0])
        assert bool(torch.isinf(ref[0]).any()) and bool((~torch.isinf(ref[0])).any())


def test_noalloc_step_rejects_sizes_beyond_the_limit(B):
    import torch
    geom = W.slab_geometry(1)
    geo = B.Geometry(geom)
    n = B.NOALLOC_MAX_QUERIES + 1
    pos = torch.zeros((n, 3), dtype=torch.float32, device="cuda")
    dirs = torch.zeros((n, 3), dtype=torch.float32, device="cuda"); dirs[:, 2] = 1
    vol = torch.zeros(n, dtype=torch.int32, device="cuda")
    out = (torch.full((n,), -7.0, dtype=torch.float32, device="cuda"), torch.full((n,), -7, dtype=torch.int32, device="cuda"))
    with pytest.raises(B.GammaNavError, match="GN_NOALLOC_MAX_QUERIES"):
        B.nav_compute_step_noalloc(geo, pos, dirs, vol, out)
    torch.cuda.synchronize()
    assert bool((out[0] == -7.0).all()) and bool((out[1] == -7).all())     # outputs untouched on failure


def test_noalloc_step_allocates_nothing(B):
    """Device memory in use (driver view, cudaMemGetInfo) does not move across calls once the library is loaded."""
    import torch
    geom = W.detector_geometry(seed=4, n_phi=16, n_z=8, barrels=((200, 400), (450, 650)))
    geo = B.Geometry(geom)
    n = 300_000
    pos, dirs = _queries(B, geom, n, 24, np.float32)
    vol = B.nav_locate(geo, pos, dirs)
    out = (torch.empty(n, dtype=torch.float32, device="cuda"), torch.empty(n, dtype=torch.int32, device="cuda"))
    B.nav_compute_step_noalloc(geo, pos, dirs, vol, out)                   # first use on this device: symbol address lookup
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        B.nav_compute_step_noalloc(geo, pos, dirs, vol, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
