"""The N > 1 path is replicas only: its host logic — rank -> launch power, barrier, sum of
units / max-over-ranks time — run with world_size 2 on the gloo backend (CPU)."""
import os
import socket

import pytest

from paper_1901_01895_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group(backend="gloo", rank=rank, world_size=world)
    try:
        assert replicas.env_rank_world() == (rank, rank, world)
        dist.barrier()
        # rank 1 is the slow one: the whole-job figure must use ITS time and BOTH ranks' units
        units, ms, value = replicas.whole_job(units_local=1000.0 * (rank + 1), ms_local=10.0 * (rank + 1), dist=dist)
        dist.barrier()
        out.put((rank, units, ms, value, replicas.launch_power_db(rank, world), replicas.amplitude_scale(rank, world)))
    finally:
        dist.destroy_process_group()


def test_whole_job_aggregate_world2_gloo():
    import torch.multiprocessing as mp
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
    for rank, units, ms, value, db, amp in res:
        assert units == 3000.0 and ms == 20.0                  # sum of units, max of times, on every rank
        assert value == pytest.approx(3000.0 / 20e-3)
    assert [r[4] for r in res] == [-1.0, 1.0]                   # launch-power sweep: -1 dB and +1 dB
    assert res[0][5] == pytest.approx(10 ** (-1 / 20)) and res[1][5] == pytest.approx(10 ** (1 / 20))


def test_single_process_defaults():
    assert replicas.launch_power_db(0, 1) == 0.0 and replicas.amplitude_scale(0, 1) == 1.0
    units, ms, value = replicas.whole_job(500.0, 5.0)
    assert (units, ms) == (500.0, 5.0) and value == pytest.approx(1e5)
    assert [replicas.launch_power_db(r, 8) for r in (0, 7)] == [-1.0, 1.0]
