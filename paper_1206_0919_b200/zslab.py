"""z-slab decomposition of ONE event over several ranks.

The step has exactly one exchange: a sweep reads 4 ghost cells per side, so only the z sweeps couple the
slabs.  Rank r owns nz_r consecutive planes; its solver's grid carries G = 4 halo planes per neighbour and runs its z
sweeps with the outflow rule (SHASTA_BOUNDARY_Z 0): the copy-edge ghosts then only feed the outer 4 planes, which are
halo and get overwritten.  Before EVERY z sweep each rank sends the 4 owned planes next to each interface and writes
what it receives into its halo planes (NCCL send/recv straight from and into the planes of the handle's state buffer,
shasta_plane_ptr; or staged through shasta_get_planes / shasta_set_planes); x and y sweeps need nothing.  A face without a neighbour (first/last rank of an outflow run) has no halo: the solver's own ghost rule is
the physical boundary there.  A periodic run wraps rank 0 <-> world-1.  Every owned cell therefore sees the same
9-point neighbourhood as in the single-domain run and is updated by the same kernel: the results are identical.

Orchestration and message passing only: every arithmetic step stays in the kernels behind the C ABI.  The solver is
any object with the binding's sweep / get_planes / set_planes [/ plane_views] (paper_1206_0919_b200.shasta.Shasta); the two drivers
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

    # A message is a LIST of tensors.  With a solver that offers plane_views (shasta_plane_ptr) the five tensors alias
    # the field planes themselves: sent from and received into place, no staging copies.  Otherwise (get_planes /
    # set_planes only) it is one packed (5, G, ny, nx) tensor, received into a staging tensor and written by commit().
    def _take(self, z0):
        pv = getattr(self.s, "plane_views", None)
        return pv(z0, G) if pv is not None else [self.s.get_planes(z0, G)]

    def outgoing(self):
        """(to_lo, to_hi): the owned planes next to each interface (None: no neighbour there)"""
        lay = self.lay
        return (self._take(lay.lo) if lay.lo_nb is not None else None,
                self._take(lay.lo + lay.nz - G) if lay.hi_nb is not None else None)

    def incoming(self, to_lo, to_hi):
        """(from_lo, from_hi): where the neighbours' planes land: the halo planes themselves, or staging tensors shaped
        like the outgoing messages"""
        import torch
        lay = self.lay
        if hasattr(self.s, "plane_views"):
            return (self.s.plane_views(0, G) if lay.lo_nb is not None else None,
                    self.s.plane_views(lay.lo + lay.nz, G) if lay.hi_nb is not None else None)
        return ([torch.empty_like(t) for t in to_lo] if to_lo is not None else None,
                [torch.empty_like(t) for t in to_hi] if to_hi is not None else None)

    def commit(self, from_lo, from_hi):
        """staging tensors -> halo planes (nothing to do when the messages were received in place)"""
        if hasattr(self.s, "plane_views"):
            return
        if from_lo is not None:
            self.s.set_planes(0, from_lo[0])
        if from_hi is not None:
            self.s.set_planes(self.lay.lo + self.lay.nz, from_hi[0])

    def owned(self, t):
        """owned planes of a local field tensor (..., nz_local, ny, nx)"""
        return t[..., self.lay.lo:self.lay.lo + self.lay.nz, :, :]

    def owned_conserved(self):
        return self.s.get_planes(self.lay.lo, self.lay.nz)


# ---------------------------------------------------------------------------------------------- exchange
def exchange_distributed(slab: ZSlab, group=None):
    """Halo refresh between ranks.  Messages "up" (tags 0..): my top planes -> hi neighbour's lo halo; "down" (tags 8..):
    my bottom planes -> lo neighbour's hi halo.  Sends are posted up-then-down and receives lo-then-hi, field by field, so
    that with two periodic ranks (both neighbours the same peer) the in-order matching of nccl pairs them right; gloo
    matches by tag.  One batch = one NCCL group: no ordering deadlock."""
    import torch.distributed as dist
    lay = slab.lay
    if lay.lo_nb is None and lay.hi_nb is None:
        return
    to_lo, to_hi = slab.outgoing()
    from_lo, from_hi = slab.incoming(to_lo, to_hi)
    ops = []
    for i, t in enumerate(to_hi or ()):
        ops.append(dist.P2POp(dist.isend, t, lay.hi_nb, group, i))
    for i, t in enumerate(to_lo or ()):
        ops.append(dist.P2POp(dist.isend, t, lay.lo_nb, group, 8 + i))
    for i, t in enumerate(from_lo or ()):
        ops.append(dist.P2POp(dist.irecv, t, lay.lo_nb, group, i))
    for i, t in enumerate(from_hi or ()):
        ops.append(dist.P2POp(dist.irecv, t, lay.hi_nb, group, 8 + i))
    for w in dist.batch_isend_irecv(ops):
        w.wait()
    slab.commit(from_lo, from_hi)


def exchange_in_process(slabs):
    """The same refresh for slabs that live in one process (rank order): device-to-device copies in stream order."""
    msgs = [sl.outgoing() for sl in slabs]
    for sl, (to_lo, to_hi) in zip(slabs, msgs):
        lay = sl.lay
        from_lo, from_hi = sl.incoming(to_lo, to_hi)
        if from_lo is not None:
            for d, src in zip(from_lo, msgs[lay.lo_nb][1]):
                d.copy_(src)
        if from_hi is not None:
            for d, src in zip(from_hi, msgs[lay.hi_nb][0]):
                d.copy_(src)
        sl.commit(from_lo, from_hi)


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
    s.set_active_planes(lay.lo, lay.lo + lay.nz)           # x and y sweeps skip the halo planes (refreshed before each z sweep)
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
