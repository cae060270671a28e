"""N > 1 path on CPU: two gloo ranks each take a contiguous photon-id range, run the transport
(the oracle stands in for the kernels here -- the host-side sharding and the tally all-reduce are what is under
test), all-reduce the tally, and must reproduce the single-process result."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_1209_5235_b200 import workloads as W
from paper_1209_5235_b200.sharding import allreduce_tally, shard_range

N = 4001


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _case(secondaries):
    """config 1 as it stands, or -- secondaries -- its geometry under an 8 MeV beam with the annihilation photons followed
    (a photon's secondaries stay on the rank that owns its id)."""
    wl = W.config(1)
    if not secondaries:
        return wl.geometry, wl.source, {}
    return wl.geometry, W.Source(W.SRC_PENCIL, (0.0, 0.0, -500.0), (0.0, 0.0, 1.0), W.E_MONO, 8.0), dict(secondaries=1)


def _worker(rank, world, port, q, secondaries=False):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = W.config(1)
    geom, source, opts = _case(secondaries)
    og = oracle.OracleGeometry(geom, **opts)
    first, count = shard_range(N, rank, world)
    r = og.transport(source, wl.seed, count, 64, first_id=first)
    edep, stats = allreduce_tally(torch.from_numpy(r["edep"]), r["stats"])
    if rank == 0:
        q.put((edep.numpy().copy(), stats))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(180)
@pytest.mark.parametrize("secondaries", [False, True])
def test_two_rank_sharded_run_equals_single_run(secondaries):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q, secondaries)) for r in range(2)]
    for p in procs:
        p.start()
    edep, stats = q.get(timeout=150)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl = W.config(1)
    geom, source, opts = _case(secondaries)
    ref = oracle.OracleGeometry(geom, **opts).transport(source, wl.seed, N, 64)
    assert np.allclose(edep, ref["edep"], rtol=1e-12, atol=0)
    for k in ("n_steps", "n_compton", "n_pe", "n_pair", "n_cut", "n_escaped", "n_photons"):
        assert stats[k] == ref["stats"][k]
    if secondaries:
        assert stats["n_pair"] > 50
    assert abs(stats["e_source"] - ref["stats"]["e_source"]) < 1e-9
