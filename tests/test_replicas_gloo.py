"""world_size-2 `gloo` test of the multi-GPU plumbing (replicas only: barrier + max-over-ranks, no data-path collective)."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from oracle import windows as ow
    from paper_2601_07154_b200 import replicas, synth
    assert replicas.init("gloo") == world
    assert replicas.env_world() == (rank, rank, world)
    replicas.barrier()
    # each rank "measures" a different step time: the job's time is the slowest rank's
    ms = replicas.max_over_ranks(10.0 + 5.0 * rank)
    value = replicas.whole_job_value(1800, ms, world)
    # every rank builds the same seeded clip (replicas): identical window partition and local poses on all ranks
    cfg = synth.CONFIGS[1]
    traj = synth.trajectory(cfg, synth.seed_for(1, 1), 24)
    loc = synth.local_windows(traj, cfg["W"], ow.window_starts(len(traj), cfg["W"], cfg["stride"]), seed=synth.seed_for(1, 2))
    checksum = replicas.max_over_ranks(float(abs(loc).sum())) - float(abs(loc).sum())
    replicas.barrier()
    out.put((rank, ms, value, checksum))
    replicas.finish()


def test_two_rank_replicas_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value, checksum in res:
        assert ms == 15.0                                   # max over ranks, seen by every rank
        assert value == 2 * 1800 / 15e-3                    # whole-job units / slowest rank's time
        assert checksum == 0.0                              # same seeded inputs on every rank


def test_single_process_defaults():
    from paper_2601_07154_b200 import replicas
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert replicas.env_world() == (0, 0, 1)
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.whole_job_value(100, 50.0, 1) == 2000.0
