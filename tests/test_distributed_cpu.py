"""N > 1 host logic of bench.py on CPU: gloo, world_size 2.

The path shards by curve with no exchange step, so what there is to test is that every
rank draws its own curves (weak scaling, disjoint seeds), that the max-over-ranks timing
reduction works, and that the reference arm runs on rank 0 only.
"""
import os
import socket
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import argparse
        import bench
        args = argparse.Namespace(config=2, curves=2, periods=16)
        w = bench.make_workload(args, rank)
        assert w.ncurves == 2 and w.nperiods == 16
        # every rank has its own curves: gather a fingerprint of the flux
        fp = torch.tensor([float(np.abs(w.flux.astype(np.float64)).sum())], dtype=torch.float64)
        got = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(got, fp)
        vals = [float(g.item()) for g in got]
        assert len(set(vals)) == world, vals
        # rank r's batch is curves [2r, 2r+2) of the config
        from paper_2312_02063_b200 import workloads
        ref = workloads.config2(ncurves=2, nperiods=16, first_curve=2 * rank)
        assert np.array_equal(ref.flux, w.flux) and np.array_equal(ref.times, w.times)
        # max-over-ranks timing
        ms = bench.max_over_ranks(10.0 + rank, world, "cpu")
        assert ms == 10.0 + (world - 1)
        dist.barrier()
        out.put((rank, "ok"))
    except Exception as e:          # pragma: no cover - reported to the parent
        out.put((rank, repr(e)))
    finally:
        dist.destroy_process_group()


def test_gloo_world2_sharding_and_timing():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(out.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
    assert res == {0: "ok", 1: "ok"}, res


def test_max_over_ranks_single_process():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
