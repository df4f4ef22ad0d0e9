"""N>1 path of bench.py on CPU: world_size-2 gloo processes (replicas only, no data-path collective)."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_1206_0919_b200 import inputs, replicas
    r, w, _ = replicas.init(use_cuda=False)
    assert (r, w) == (rank, world)
    replicas.barrier(use_cuda=False)
    ms_local = 10.0 + 5.0 * rank                        # rank 1 is the slow one
    ms = replicas.max_over_ranks(ms_local, use_cuda=False)
    c = inputs.hotspots(8, steps=1, seed=replicas.event_seed(rank))
    out.put((rank, ms, float(c["e"].sum()), replicas.aggregate_rate(8 ** 3, 6, ms, w)))
    replicas.barrier(use_cuda=False)
    replicas.finalize()


def test_two_replicas_gloo():
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
    (r0, ms0, e0, v0), (r1, ms1, e1, v1) = res
    assert ms0 == ms1 == 15.0                            # MAX over ranks, the same on every rank
    assert e0 != e1                                      # a different event per replica
    assert v0 == v1 == 2 * 512 * 6 / 15e-3               # whole-job aggregate


def test_single_process_defaults():
    sys.path.insert(0, ROOT)
    from paper_1206_0919_b200 import replicas
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    assert replicas.env() == (0, 1, 0)
    assert replicas.max_over_ranks(3.5, use_cuda=False) == 3.5
    assert replicas.event_seed(0) == 12060919 and replicas.event_seed(3) == 12060922
    assert np.isclose(replicas.aggregate_rate(100, 2, 1.0, 1), 2e5)
