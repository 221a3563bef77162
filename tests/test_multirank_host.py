"""Host logic of the N > 1 bench path (replicas, no data-path collective) under gloo, world_size 2, on CPU:
every rank draws its own candidate set, per-step times are all-gathered, throughput = all units / slowest rank."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    from paper_2602_08266_b200 import synth
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = synth.make_workload(0)
    cams = bench.rank_candidates(0, wl, rank)
    step_ms = [10.0 + rank, 12.0 + 3 * rank, 11.0]          # rank 1 is the slower one
    t_all = bench.gather_over_ranks(step_ms, dist, "cpu")
    agg = bench.aggregate(t_all, len(cams))
    dist.barrier()
    q.put((rank, t_all.tolist(), agg, cams.tobytes(), len(cams)))
    dist.destroy_process_group()


def test_two_rank_gather_and_aggregate():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, t0, a0, c0, n0), (r1, t1, a1, c1, n1) = res
    assert t0 == t1 == [[10.0, 12.0, 11.0], [11.0, 15.0, 11.0]]         # every rank sees every rank's times, in rank order
    assert n0 == n1 == 4 and c0 != c1                                      # own candidate sets, same size
    expect = 2 * 4 * 3 / (37.0e-3)                                         # all units / slowest rank's total
    assert a0["value"] == pytest.approx(expect) and a1["value"] == pytest.approx(expect)
    assert a0["ms_per_step"] == pytest.approx(37.0 / 3)


def test_single_process_gather_is_identity():
    import bench
    t = bench.gather_over_ranks([1.0, 2.0], None, "cpu")
    assert t.shape == (1, 2) and bench.aggregate(t, 5)["value"] == pytest.approx(10 / 3e-3)


def test_rank_candidates_are_deterministic_and_valid():
    import bench
    from paper_2602_08266_b200 import synth
    wl = synth.make_workload(0)
    a, b = bench.rank_candidates(0, wl, 1), bench.rank_candidates(0, wl, 1)
    assert a.tobytes() == b.tobytes() and bench.rank_candidates(0, wl, 0) is wl.cand_cams
    R = np.asarray(a[0]["R"], dtype=np.float64).reshape(3, 3)
    assert np.allclose(R @ R.T, np.eye(3), atol=1e-6)
