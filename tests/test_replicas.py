"""N > 1 path on CPU: two processes over the gloo backend exercise the control plane bench.py uses under
torchrun -- rendezvous from the environment, barrier, max-over-ranks time, sum-over-ranks units.  The data path
has no collective (replicas only), so this is all there is to cover."""
import os
import socket

import pytest
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2606_17107_b200.replicas import Replicas, aggregate_throughput
    rep = Replicas(backend="gloo")
    assert rep.world == world and rep.rank == rank
    rep.barrier()
    # rank r processes (r + 1) * 1000 tokens in (r + 1) * 0.5 s: the job is as slow as its slowest rank
    agg = aggregate_throughput(rep, (rank + 1) * 1000, (rank + 1) * 0.5)
    out.put((rank, agg["units"], agg["seconds"], agg["per_second"], rep.max(float(rank)), rep.sum(rank + 10)))
    rep.barrier()
    rep.close()


def test_two_replicas_over_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, units, seconds, per_s, mx, sm in got:
        assert units == 3000 and seconds == pytest.approx(1.0) and per_s == pytest.approx(3000.0)
        assert mx == 1.0 and sm == 21


def test_single_process_is_a_noop():
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    from paper_2606_17107_b200.replicas import Replicas, aggregate_throughput
    rep = Replicas()
    assert rep.world == 1
    rep.barrier()
    assert aggregate_throughput(rep, 10, 2.0)["per_second"] == 5.0


def test_reference_arm_other_ranks_exit_without_work(monkeypatch):
    import bench
    monkeypatch.setenv("RANK", "1")
    args = type("A", (), dict(config=1, layout="NHD", steps=1, warmup=0, gpus=2))()
    assert bench.run_reference(args) == 0
