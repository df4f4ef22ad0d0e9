"""z-slab decomposition of ONE event over several ranks.

The step has exactly one exchange: a sweep reads 4 ghost cells per side, so only the z sweeps couple the
slabs.  Rank r owns nz_r consecutive planes; its solver's grid carries G = 4 halo planes per neighbour and runs its z
sweeps with the outflow rule (SHASTA_BOUNDARY_Z 0): the copy-edge ghosts then only feed the outer 4 planes, which are
halo and get overwritten.  Before EVERY z sweep each rank sends the 4 owned planes next to each interface and writes
what it receives into its halo planes (shasta_get_planes / shasta_set_planes + NCCL send/recv); x and y sweeps need
nothing.  A face without a neighbour (first/last rank of an outflow run) has no halo: the solver's own ghost rule is
the physical boundary there.  A periodic run wraps rank 0 <-> world-1.  Every owned cell therefore sees the same
9-point neighbourhood as in the single-domain run and is updated by the same kernel: the results are identical.

Orchestration and message passing only: every arithmetic step stays in the kernels behind the C ABI.  The solver is
any object with the binding's sweep / get_planes / set_planes (paper_1206_0919_b200.shasta.Shasta); the two drivers
below differ only in who carries the planes: torch.distributed (one process per GPU: nccl; gloo on CPU tensors, used by
tests/test_zslab.py with world_size 2) or plain copies between slabs living in one process (one GPU, tests).
Not overlapped with the interior yet (the exchange is 4 planes x 5 fields per face, 10.5 MB at 256^3).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

G = 4                                              # ghost radius of a sweep = halo planes per interface
BRANCH = (0, 1, 2, 0, 2, 1, 2, 0, 1, 2, 1, 0, 1, 2, 0, 1, 0, 2)


@dataclass(frozen=True)
class Layout:
    rank: int
    world: int
    z0: int                  # first owned plane (global index)
    nz: int                  # owned planes
    lo: int                  # halo planes below the owned ones (0 or G)
    hi: int                  # halo planes above
    lo_nb: Optional[int]     # rank owning the planes below (None: physical boundary)
    hi_nb: Optional[int]

    @property
    def nz_local(self):
        return self.lo + self.nz + self.hi


def layout(nz: int, world: int, rank: int, periodic: bool) -> Layout:
    """Planes of `rank`: nz // world each, the first nz % world ranks one more.  Every slab must hold >= G planes."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    base, rem = divmod(int(nz), int(world))
    if world > 1 and base < G:
        raise ValueError(f"z-slab: {nz} planes over {world} ranks leaves slabs thinner than the {G}-plane halo")
    n = base + (1 if rank < rem else 0)
    z0 = rank * base + min(rank, rem)
    if world == 1:
        return Layout(rank, world, z0, n, 0, 0, None, None)        # one rank: the solver's own boundary rule does it
    lo_nb = rank - 1 if rank > 0 else (world - 1 if periodic else None)
    hi_nb = rank + 1 if rank < world - 1 else (0 if periodic else None)
    return Layout(rank, world, z0, n, G if lo_nb is not None else 0, G if hi_nb is not None else 0, lo_nb, hi_nb)


def local_planes(lay: Layout, nz: int):
    """Global plane index of every local plane (halo included), wrapped for periodic neighbours: for slicing the
    initial state."""
    return [(lay.z0 - lay.lo + k) % nz for k in range(lay.nz_local)]


def sweeps_of_step(step_index: int, table=BRANCH):
    """The three axes of step s: table[3 (s mod n/3) ...]."""
    c = len(table) // 3
    i = 3 * (step_index % c)
    return tuple(table[i:i + 3])


class ZSlab:
    """One rank's slab: a solver over (nx, ny, lo + nz + hi) plus the plane bookkeeping."""

    def __init__(self, solver, lay: Layout, table=BRANCH):
        self.s, self.lay, self.table = solver, lay, tuple(table)
        self.step_index = 0

    # the owned planes next to each interface, as the neighbour's halo
    def planes_for_lo(self):
        return self.s.get_planes(self.lay.lo, G) if self.lay.lo_nb is not None else None

    def planes_for_hi(self):
        return self.s.get_planes(self.lay.lo + self.lay.nz - G, G) if self.lay.hi_nb is not None else None

    def put_halo(self, from_lo, from_hi):
        if from_lo is not None:
            self.s.set_planes(0, from_lo)
        if from_hi is not None:
            self.s.set_planes(self.lay.lo + self.lay.nz, from_hi)

    def owned(self, t):
        """owned planes of a local field tensor (..., nz_local, ny, nx)"""
        return t[..., self.lay.lo:self.lay.lo + self.lay.nz, :, :]

    def owned_conserved(self):
        return self.s.get_planes(self.lay.lo, self.lay.nz)


# ---------------------------------------------------------------------------------------------- exchange
def exchange_distributed(slab: ZSlab, group=None):
    """Halo refresh between ranks.  Message "up" (tag 0): my top planes -> hi neighbour's lo halo; "down" (tag 1): my
    bottom planes -> lo neighbour's hi halo.  Sends are posted up-then-down and receives lo-then-hi, so that with two
    periodic ranks (both neighbours the same peer) the in-order matching of nccl pairs them right; gloo uses the tags."""
    import torch
    import torch.distributed as dist
    lay = slab.lay
    if lay.lo_nb is None and lay.hi_nb is None:
        return
    to_lo, to_hi = slab.planes_for_lo(), slab.planes_for_hi()
    from_lo = torch.empty_like(to_lo) if to_lo is not None else None
    from_hi = torch.empty_like(to_hi) if to_hi is not None else None
    ops = []
    if to_hi is not None:
        ops.append(dist.P2POp(dist.isend, to_hi, lay.hi_nb, group, 0))
    if to_lo is not None:
        ops.append(dist.P2POp(dist.isend, to_lo, lay.lo_nb, group, 1))
    if from_lo is not None:
        ops.append(dist.P2POp(dist.irecv, from_lo, lay.lo_nb, group, 0))
    if from_hi is not None:
        ops.append(dist.P2POp(dist.irecv, from_hi, lay.hi_nb, group, 1))
    for w in dist.batch_isend_irecv(ops):
        w.wait()
    slab.put_halo(from_lo, from_hi)


def exchange_in_process(slabs):
    """The same refresh for slabs that live in one process (rank order): pack everything, then unpack."""
    msgs = [(sl.planes_for_lo(), sl.planes_for_hi()) for sl in slabs]
    for sl in slabs:
        lay = sl.lay
        sl.put_halo(msgs[lay.lo_nb][1] if lay.lo_nb is not None else None,
                    msgs[lay.hi_nb][0] if lay.hi_nb is not None else None)


# ---------------------------------------------------------------------------------------------- time steps
def _advance(slabs, nsteps, exchange):
    for _ in range(int(nsteps)):
        s = slabs[0].step_index
        axes = sweeps_of_step(s, slabs[0].table)
        for i, a in enumerate(axes):
            if a == 2:
                exchange()
            for sl in slabs:
                sl.s.sweep(a, 1 if i == 2 else 0)        # the last sweep of a step writes the primitive fields
        for sl in slabs:
            sl.step_index = s + 1


def step_distributed(slab: ZSlab, nsteps: int, group=None):
    """nsteps time steps of this rank's slab; collective: every rank of `group` calls it with the same nsteps."""
    _advance([slab], nsteps, lambda: exchange_distributed(slab, group))


def step_in_process(slabs, nsteps: int):
    """nsteps time steps of all slabs of one event held by this process (slabs in rank order)."""
    _advance(list(slabs), nsteps, lambda: exchange_in_process(slabs))


# ---------------------------------------------------------------------------------------------- the GPU solver of a slab
def make_gpu_slab(c, world: int, rank: int, table=BRANCH, **kw) -> ZSlab:
    """Slab `rank` of `world` of the event described by the config dict `c` (paper_1206_0919_b200.inputs), on the
    current CUDA device: a Shasta handle over the local planes, its state set from the global arrays."""
    import numpy as np
    import torch
    from .shasta import Shasta
    lay = layout(c["nz"], world, rank, bool(c["boundary"]))
    s = Shasta(c["nx"], c["ny"], lay.nz_local, c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"],
               boundary_z=(0 if world > 1 else None), **kw)
    idx = np.asarray(local_planes(lay, c["nz"]))
    s.set_state(*[torch.from_numpy(np.ascontiguousarray(c[k][idx])).cuda() for k in ("e", "n", "vx", "vy", "vz")])
    return ZSlab(s, lay, table)


def conserved_totals_distributed(slab: ZSlab, dx: float, group=None):
    """dx^3 * sums of E, Mx, My, Mz, R over the whole event: each rank sums its owned planes on the GPU
    (shasta_conserved_totals_static), then one all-reduce of 5 doubles.  Returns a CUDA tensor of 5."""
    import torch
    import torch.distributed as dist
    from . import shasta as sh
    U = slab.owned_conserved()
    out = torch.empty(5, dtype=torch.float64, device=U.device)
    sh.conserved_totals_static(U[0], U[1], U[2], U[3], U[4], float(dx) ** 3, out)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(out, group=group)
    return out


# ---------------------------------------------------------------------------------------------- command line
def main(argv=None):
    """`torchrun --nproc-per-node N -m paper_1206_0919_b200.zslab --size 256 --steps 20`: ONE hotspots event of size^3
    cells sharded over N GPUs (strong scaling; bench.py's --gpus N runs N independent events instead).  Device time of
    the K steps, MAX over ranks; rank 0 prints one JSON line."""
    import argparse
    import json
    import torch
    from . import inputs, replicas
    ap = argparse.ArgumentParser()
    ap.add_argument("--size", type=int, default=256)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=6)
    args = ap.parse_args(argv)
    rank, world, _ = replicas.init(use_cuda=True)
    c = inputs.hotspots(args.size, steps=0)
    slab = make_gpu_slab(c, world, rank)
    step_distributed(slab, args.warmup)
    replicas.barrier(True)
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    step_distributed(slab, args.steps)
    t1.record()
    replicas.barrier(True)
    ms = replicas.max_over_ranks(t0.elapsed_time(t1), True)
    tot = conserved_totals_distributed(slab, c["dx"]).cpu().tolist()
    if rank == 0:
        lay = slab.lay
        faces = (lay.lo_nb is not None) + (lay.hi_nb is not None)
        halo = faces * G * c["nx"] * c["ny"] * 5 * 8          # bytes this rank sends per step (one z sweep per step)
        print(json.dumps({
            "metric": "cell-updates/sec of ONE event sharded in z slabs", "value": c["nx"] * c["ny"] * c["nz"] * args.steps / (ms * 1e-3),
            "unit": "cell-updates/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "scaling": "strong", "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"hotspots {args.size}^3, z slabs of {lay.nz} (+{lay.lo}+{lay.hi} halo) planes",
                       "halo_bytes_sent_per_step_rank0": halo},
            "conserved_totals": tot}), flush=True)
    replicas.finalize()


if __name__ == "__main__":
    main()
