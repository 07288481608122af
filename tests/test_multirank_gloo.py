"""-m "not gpu": the N > 1 host logic of bench.py under torch.distributed (gloo, world_size 2, CPU).  The path shards by
jets with no data-path collective ("replicas only"): the only communication is the MAX all-reduce
of the timed milliseconds, and ranks must draw disjoint batches."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import bench
import synth


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local_ms = 10.0 * (rank + 1)                       # rank 1 is the slow one
    value, t_max = bench.aggregate_throughput(local_ms, 1024 * 5, world, dist, "cpu")
    b = bench.make_batches(synth, rank, 8)[0]
    out.put((rank, value, t_max, float(b.feats.sum()), int(b.n_particles)))
    dist.barrier()
    dist.destroy_process_group()


def test_world2_max_over_ranks_and_disjoint_batches():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (r0, v0, t0, s0, n0), (r1, v1, t1, s1, n1) = res
    assert t0 == t1 == 20.0                            # the job takes as long as its slowest rank
    assert v0 == v1 == 2 * 1024 * 5 / 20e-3            # whole-job jets/s: all ranks' jets over the max time
    assert s0 != s1                                    # different seeds: the replicas do not repeat one batch


def test_single_rank_needs_no_process_group():
    v, t = bench.aggregate_throughput(4.0, 1024, 1)
    assert t == 4.0 and v == 1024 / 4e-3
    assert bench.batch_seed(0, 0) == 1002 and len({bench.batch_seed(r, k) for r in range(4) for k in range(8)}) == 32


def test_work_accounting_matches_the_survey_figures():
    """bench.work(): algorithmic MACs per particle: base arch F = 7, k_eff = 16: stated 4 118 976, minimal
    (layer 1 factorised) 2 876 736; head 66 048 MAC per jet; wide arch minimal 11 504 256; Tiny (k = 4): 9 344 / 8 576."""
    a = synth.ARCHS["particlenet"]
    w = bench.work(a, [17])                            # one jet of 17 particles: k_eff = 16 for every particle
    assert w["stated"] == 2 * (17 * 4118976 + 66048)
    assert w["min"] == 2 * (17 * 2876736 + 66048)
    assert w["blocks_min"] == [2 * 17 * 132416, 2 * 17 * 548864, 2 * 17 * 2195456]
    assert w["blocks_edge"][2] == 2 * 17 * 16 * (256 * 256 * 2)
    ww = bench.work(synth.ARCHS["wide"], [17])
    assert ww["min"] == 2 * (17 * 11504256 + 263168)
    t = bench.work(synth.ARCHS["tiny"], [16])
    assert t["stated"] == 2 * (16 * 9344 + 64) and t["min"] == 2 * (16 * 8576 + 64)
    # k_eff = min(k, n - 1): a jet of 5 particles has 4 neighbours per particle, a single particle none
    w5 = bench.work(a, [5, 1])
    assert w5["blocks_edge"][0] == 2 * (5 * 4) * (64 * 64 * 2)
