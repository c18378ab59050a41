"""N > 1 path of bench.py (replicas only) on the gloo backend, world_size 2, CPU."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

from paper_1011_3318_b200 import inputs as I
from paper_1011_3318_b200 import replicas as R


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    assert R.env_rank() == (rank, world, rank)
    R.init("gloo")
    R.barrier(world, cuda=False)
    streams = R.source_streams(rank, world, 2)
    eta = I.spinor((4, 4, 4, 4), 7, stream=streams[0])
    local_ms = 10.0 + 5.0 * rank  # rank 1 is the slow replica
    job = R.job_summary(local_ms, 2, world)
    out[rank] = (streams, float(np.abs(eta).sum()), R.max_over_ranks(local_ms, world), job)
    R.barrier(world, cuda=False)
    R.shutdown(world)


def test_two_replicas_gloo():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert sorted(res) == [0, 1]
    s0, s1 = res[0][0], res[1][0]
    assert s0 == [0, 1] and s1 == [2, 3] and not set(s0) & set(s1)      # disjoint right-hand sides
    assert res[0][1] != res[1][1]                                        # the replicas really got different sources
    assert res[0][2] == res[1][2] == 15.0                                # max over ranks on every rank
    for r in (0, 1):
        job = res[r][3]
        assert job["ms_per_step"] == 15.0 and job["solves_per_step"] == 4
        assert job["solves_per_s"] == pytest.approx(4 / 15e-3)


def test_single_process_is_identity():
    assert R.max_over_ranks(3.5, 1) == 3.5
    assert R.source_streams(0, 1) == [0]
    with pytest.raises(ValueError):
        R.source_streams(2, 2)
