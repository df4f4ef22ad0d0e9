"""z-slab decomposition (paper_1206_0919_b200/zslab.py): host logic on CPU.

The slab drivers only orchestrate sweeps and carry planes, so here the solver of a slab is a stand-in that sweeps every
pencil with the oracle's oracle_sweep_pencil on host arrays; the reference is the oracle's own single-domain 3-D run.
The decomposition changes no cell's neighbourhood: the owned planes must come out BITWISE equal.  Two ways of carrying
the planes are covered: in-process copies (any number of slabs) and torch.distributed with gloo, world_size 2."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)

from paper_1206_0919_b200 import inputs, zslab   # noqa: E402

FIELDS = ("E", "Mx", "My", "Mz", "R")


class PencilSolver:
    """sweep / get_planes / set_planes of the binding, on a (5, nz, ny, nx) host array, pencil by pencil via the oracle"""

    def __init__(self, so, U, c, bc_z):
        self.so, self.U, self.c, self.bc_z = so, np.array(U, dtype=np.float64), c, bc_z
        self.sweeps = []

    def sweep(self, axis, emit=0):
        bc = self.bc_z if axis == 2 else self.c["boundary"]
        a = np.moveaxis(self.U, {0: 3, 1: 2, 2: 1}[axis], -1)          # view: (5, ., ., N)
        for i in range(a.shape[1]):
            for j in range(a.shape[2]):
                a[:, i, j, :] = self.so.sweep_pencil(a[:, i, j, :], axis, self.c["lam"], self.c["gamma"], self.c["mass"], bc)[0]
        self.sweeps.append((axis, emit))

    def get_planes(self, z0, n):
        return torch.from_numpy(self.U[:, z0:z0 + n].copy())

    def set_planes(self, z0, t):
        self.U[:, z0:z0 + t.shape[1]] = t.numpy()


def _initial(so, c):
    o = so.Oracle(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"])
    o.set_state(c["e"], c["n"], c["vx"], c["vy"], c["vz"])
    U0 = np.stack([o.get_conserved()[k] for k in FIELDS])
    return o, U0


def _make_slab(so, c, U0, world, rank):
    lay = zslab.layout(c["nz"], world, rank, bool(c["boundary"]))
    idx = np.asarray(zslab.local_planes(lay, c["nz"]))
    bc_z = inputs.OUTFLOW if world > 1 else c["boundary"]
    return zslab.ZSlab(PencilSolver(so, U0[:, idx], c, bc_z), lay)


# ---------------------------------------------------------------------------------------------- layout
def test_layout_covers_the_grid_once():
    for nz, world in ((19, 2), (29, 3), (32, 8), (4, 1), (17, 4)):
        for periodic in (False, True):
            lays = [zslab.layout(nz, world, r, periodic) for r in range(world)]
            assert [l.z0 for l in lays] == list(np.cumsum([0] + [l.nz for l in lays[:-1]]))
            assert sum(l.nz for l in lays) == nz and max(l.nz for l in lays) - min(l.nz for l in lays) <= 1
            for l in lays:
                if world == 1:
                    assert (l.lo, l.hi, l.lo_nb, l.hi_nb) == (0, 0, None, None)
                    continue
                assert l.lo == (zslab.G if (l.rank > 0 or periodic) else 0)
                assert l.hi == (zslab.G if (l.rank < world - 1 or periodic) else 0)
                assert l.lo_nb == ((l.rank - 1) % world if l.lo else None)
                assert l.hi_nb == ((l.rank + 1) % world if l.hi else None)
                planes = zslab.local_planes(l, nz)
                assert planes[l.lo:l.lo + l.nz] == list(range(l.z0, l.z0 + l.nz))
                assert planes[:l.lo] == [(l.z0 - l.lo + k) % nz for k in range(l.lo)]
    with pytest.raises(ValueError):
        zslab.layout(15, 4, 0, False)                 # slabs of 3 planes cannot feed a 4-plane halo
    assert zslab.sweeps_of_step(0) == (0, 1, 2) and zslab.sweeps_of_step(5) == (1, 0, 2) and zslab.sweeps_of_step(6) == (0, 1, 2)


# ---------------------------------------------------------------------------------------------- in-process
@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("world", [2, 3])
def test_slabs_in_one_process_equal_the_single_domain_run(oracle, bc, world):
    c = inputs.random_state(6, 5, 14, seed=3 + bc, kind="rough", boundary=bc)
    o, U0 = _initial(oracle, c)
    o.step(6)                                          # one whole cycle of the axis table
    ref = np.stack([o.get_conserved()[k] for k in FIELDS])
    slabs = [_make_slab(oracle, c, U0, world, r) for r in range(world)]
    zslab.step_in_process(slabs, 6)
    got = np.concatenate([sl.owned_conserved().numpy() for sl in slabs], axis=1)
    assert got.shape == ref.shape and np.array_equal(got, ref)
    assert slabs[0].step_index == 6
    assert slabs[0].s.sweeps[:3] == [(0, 0), (1, 0), (2, 1)]          # emit only in the last sweep of a step
    # the exchange is needed: without it the planes next to the interface differ
    lone = [_make_slab(oracle, c, U0, world, r) for r in range(world)]
    for sl in lone:
        zslab._advance([sl], 6, lambda: None)
    bad = np.concatenate([sl.owned_conserved().numpy() for sl in lone], axis=1)
    assert not np.array_equal(bad, ref)


# ---------------------------------------------------------------------------------------------- gloo, world_size 2
def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, bc, out):
    for p in (ROOT, os.path.join(ROOT, "tests")):
        if p not in sys.path:
            sys.path.insert(0, p)
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch.distributed as dist
    from oracle import shasta_oracle as so
    from paper_1206_0919_b200 import replicas
    replicas.init(use_cuda=False)
    c = inputs.random_state(6, 5, 19, seed=11 + bc, kind="rough", boundary=bc)     # 10 + 9 planes
    _, U0 = _initial(so, c)
    slab = _make_slab(so, c, U0, world, rank)
    zslab.step_distributed(slab, 6)
    own = slab.owned_conserved()
    tot = own.sum(dim=(1, 2, 3))                       # the all-reduce of the totals (sum order differs from the oracle's)
    dist.all_reduce(tot)
    out.put((rank, own.numpy(), tot.numpy() * c["dx"] ** 3))
    replicas.barrier(use_cuda=False)
    replicas.finalize()


@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
def test_two_slabs_over_gloo_equal_the_single_domain_run(oracle, bc):
    c = inputs.random_state(6, 5, 19, seed=11 + bc, kind="rough", boundary=bc)
    o, _ = _initial(oracle, c)
    o.step(6)
    ref = np.stack([o.get_conserved()[k] for k in FIELDS])
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, bc, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    got = np.concatenate([r[1] for r in res], axis=1)
    assert np.array_equal(got, ref)
    t_ref = o.conserved_totals()
    for r in res:
        assert np.max(np.abs(r[2] - t_ref)) <= 1e-12 * abs(t_ref[0])
