"""GPU-vs-oracle parity through the C ABI (-m gpu).  Tolerances (north_star):
fp64 err_max <= 1e-10 per field (err_L1 reported, expected <= 1e-12); fp32 err_L1 <= 1e-4."""
import numpy as np
import pytest

from paper_1206_0919_b200 import inputs
import parity

pytestmark = pytest.mark.gpu

TOL64 = 1e-10
# Kernel-level (1-6 step) tests: every field to 1e-12 (n after its conditioning allowance, parity.n_allowance).
TOL_CONS, TOL_PRIM = 1e-12, 1e-12


def assert_kernel_parity(got, ref, label, tol_cons=TOL_CONS, tol_prim=TOL_PRIM):
    parity.assert_parity(got, ref, tol_cons, fields=parity.CONS, label=label + " [cons]")
    parity.assert_parity(got, ref, tol_prim, fields=parity.PRIM, label=label + " [prim]")


@pytest.fixture(scope="module", autouse=True)
def _built():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1206_0919_b200 import build
    build.build()


# ------------------------------------------------------------------ T1: kernel-level parity
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("kind", ["smooth", "rough"])
def test_single_axis_sweeps_ragged(oracle, axis, bc, kind):
    # 37x19x23: not a multiple of any tile, warp or chunk size; three sweeps along one axis
    c = inputs.random_state(37, 19, 23, seed=10 * axis + bc, kind=kind, boundary=bc)
    ref, o = parity.run_oracle(oracle, c, steps=1, table=[axis] * 3)
    got, s = parity.run_gpu(c, steps=1, table=[axis] * 3)
    assert_kernel_parity(got, ref, f"axis {axis} bc {bc} {kind}")
    # Pi fires in the same cells up to those sitting within rounding of the limit |M| = (1-1e-12) E
    # (cells within an ulp of the limit may fall on either side: at most 2, or 0.5 % of the firings)
    assert abs(s.diagnostics()[0] - o.diagnostics()[0]) <= max(2, o.diagnostics()[0] // 200)


@pytest.mark.parametrize("shape", [(1, 1, 50), (1, 40, 1), (64, 1, 1), (5, 1, 9), (2, 3, 4), (3, 3, 3), (130, 2, 1),
                                   (33, 65, 2)])
@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
def test_degenerate_shapes(oracle, shape, bc):
    nx, ny, nz = shape
    c = inputs.random_state(nx, ny, nz, seed=nx + ny + nz, kind="rough", boundary=bc)
    ref, _ = parity.run_oracle(oracle, c, steps=3)
    got, _ = parity.run_gpu(c, steps=3)
    assert_kernel_parity(got, ref, f"shape {shape} bc {bc}")


@pytest.mark.parametrize("segment", [8, 16, 40, 1000])
def test_segmentation_does_not_change_the_answer(oracle, segment):
    c = inputs.random_state(70, 45, 50, seed=77, kind="rough")
    ref, _ = parity.run_oracle(oracle, c, steps=2)
    got, _ = parity.run_gpu(c, steps=2, segment=segment)
    assert_kernel_parity(got, ref, f"segment {segment}")


@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("shape", [(38, 19, 23), (64, 5, 7), (130, 33, 2), (8, 40, 3)])
@pytest.mark.parametrize("segment", [0, 8, 12, 24])
def test_x_sweep_tma_and_cp_async_paths(oracle, bc, shape, segment):
    # even nx: interior 4-cell groups of the x sweep move by TMA (UTMALDG/UTMASTG), boundary groups and groups that
    # straddle a segment end by cp.async / stores; SHASTA_NO_TMA forces the latter everywhere.  Same bits either way.
    nx, ny, nz = shape
    c = inputs.random_state(nx, ny, nz, seed=nx + 3 * bc, kind="rough", boundary=bc)
    ref, _ = parity.run_oracle(oracle, c, steps=1, table=[0, 0, 0])
    got, s = parity.run_gpu(c, steps=1, table=[0, 0, 0], segment=segment)
    assert_kernel_parity(got, ref, f"x sweep tma shape {shape} bc {bc} segment {segment}")
    assert s.kernel_name(0) == "sweep_x2_kernel", "even nx: the x sweep must be on its TMA path"
    alt, sa = parity.run_gpu(c, steps=1, table=[0, 0, 0], segment=segment, no_tma=1)
    assert sa.kernel_name(0) == "sweep_x2_kernel(cp.async)"
    for k in parity.CONS + parity.PRIM:
        assert np.array_equal(got[k], alt[k]), k


@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("shape", [(38, 19, 23), (64, 9, 7), (130, 6, 5), (96, 40, 3), (32, 4, 4)])
@pytest.mark.parametrize("segment", [0, 8, 12])
def test_yz_sweeps_tma_and_cp_async_paths(oracle, bc, shape, segment):
    # nx >= 32 and even: the y/z sweeps are fed by 3-D TMA boxes {32, 4 cells} (ghost groups: four 1-cell boxes at the
    # ghost-mapped coordinate, partial x-blocks zero-filled and never stored); SHASTA_NO_TMA forces the cp.async fill.
    nx, ny, nz = shape
    c = inputs.random_state(nx, ny, nz, seed=nx + 5 * bc, kind="rough", boundary=bc)
    ref, _ = parity.run_oracle(oracle, c, steps=1, table=[1, 2, 1])
    got, s = parity.run_gpu(c, steps=1, table=[1, 2, 1], segment=segment)
    assert_kernel_parity(got, ref, f"y/z sweeps tma shape {shape} bc {bc} segment {segment}")
    alt, _ = parity.run_gpu(c, steps=1, table=[1, 2, 1], segment=segment, no_tma=1)
    for k in parity.CONS + parity.PRIM:
        assert np.array_equal(got[k], alt[k]), k


@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
def test_general_eos_mass(oracle, bc):
    c = inputs.random_state(24, 20, 28, seed=4, kind="rough", gamma=5.0 / 3.0, mass=1.0, boundary=bc)
    ref, _ = parity.run_oracle(oracle, c, steps=6)
    got, _ = parity.run_gpu(c, steps=6)
    assert_kernel_parity(got, ref, "general EOS", tol_cons=1e-11, tol_prim=1e-11)


def test_uniform_state_stays_uniform_bitwise():
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    sh = (12, 10, 40)
    s = Shasta(40, 10, 12, 0.1, 0.4, 4.0 / 3.0)
    mk = lambda v: torch.full(sh, v, dtype=torch.float64, device="cuda")
    s.set_state(mk(1.7), mk(0.9), mk(0.3), mk(-0.2), mk(0.5))
    before = {k: v.clone() for k, v in s.get_conserved().items()}
    s.step(6)
    after = s.get_conserved()
    for k in before:
        assert torch.equal(before[k], after[k]), k


@pytest.mark.parametrize("shape", [(96, 40, 24), (70, 45, 50)])
def test_run_to_run_bitwise_reproducible(shape):
    # the producer/consumer kernels reuse shared-memory ring and queue slots under barrier protocols: a race there
    # would show up as run-to-run differences (compute-sanitizer is closed on this pool).  Six steps = all axis orders.
    c = inputs.random_state(*shape, seed=99, kind="rough")
    first, _ = parity.run_gpu(c, steps=6)
    for _ in range(4):
        again, _ = parity.run_gpu(c, steps=6)
        for k in parity.CONS + parity.PRIM:
            assert np.array_equal(first[k], again[k]), k


@pytest.mark.parametrize("eos", ["mass", "table"])
def test_general_eos_bits_do_not_depend_on_idle_lanes_or_stale_memory(eos):
    # Newton kernels, ragged shapes (warps with idle lanes / rows whose shared-memory slots hold whatever was there): until a
    # converged cell was frozen in place, the warp-wide vote let such lanes decide how often the others iterated, and results
    # moved by an ulp from run to run (found with the scale-homogeneity test).  Other problems run in between to change
    # what stale memory holds.
    import hashlib
    tab = inputs.eos_table("soft") if eos == "table" else None
    kw = dict(gamma=5.0 / 3.0, mass=1.0 if eos == "mass" else 0.0, boundary=inputs.PERIODIC)

    def digest(r):
        return hashlib.md5(b"".join(np.ascontiguousarray(r[f]).tobytes() for f in sorted(r))).hexdigest()

    for shape in ((24, 20, 28), (40, 24, 13)):
        c = inputs.random_state(*shape, seed=93, kind="rough", **kw)
        seen = set()
        for rep in range(6):
            seen.add(digest(parity.run_gpu(c, steps=3, eos_table=tab)[0]))
            if rep % 2 == 0:
                parity.run_gpu(inputs.random_state(33, 17, 9, seed=rep, kind="rough", **kw), steps=1, eos_table=tab)
        assert len(seen) == 1, (shape, seen)


@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("shape", [(37, 19, 23), (64, 33, 6)])
def test_fp32_storage_kernel_level(oracle, bc, shape):
    # fp32 storage + transport, fp64 cons2prim (row a7): ragged shapes, every axis, 2 steps: one fp32 rounding per
    # operation, so a few 1e-7 relative; a wrong index or stride in the float instantiations would be O(1)
    c = inputs.random_state(*shape, seed=5 + bc, kind="smooth", boundary=bc)
    ref, _ = parity.run_oracle(oracle, c, steps=2)
    got, _ = parity.run_gpu(c, steps=2, precision=32)
    errs = parity.field_errors(got, ref)
    for k, (emax, el1) in errs.items():
        assert emax <= 2e-5 and el1 <= 2e-6, (k, emax, el1)


@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("shape", [(64, 9, 7), (132, 33, 2), (40, 40, 3), (38, 19, 5)])
@pytest.mark.parametrize("segment", [0, 8, 24])
def test_fp32_tma_and_cp_async_paths_same_bits(oracle, bc, shape, segment):
    # fp32 storage: nx % 4 == 0 gives 16 B row strides, so all three sweeps are TMA-fed (x: dense {4, 32} tiles);
    # SHASTA_NO_TMA forces the cp.async fill and the LSU drain.  Same bits either way, and close to the fp64 oracle.
    c = inputs.random_state(*shape, seed=shape[0] + 7 * bc, kind="smooth", boundary=bc)
    got, _ = parity.run_gpu(c, steps=2, precision=32, segment=segment)
    alt, _ = parity.run_gpu(c, steps=2, precision=32, segment=segment, no_tma=1)
    for k in parity.CONS + parity.PRIM:
        assert np.array_equal(got[k], alt[k]), k
    ref, _ = parity.run_oracle(oracle, c, steps=2)
    for k, (emax, el1) in parity.field_errors(got, ref).items():
        assert emax <= 2e-5 and el1 <= 2e-6, (k, emax, el1)


@pytest.mark.parametrize("eos", ["gamma", "mass", "table"])
def test_vacuum_and_superluminal_cells(oracle, eos):
    # E <= 0 cells and |M| > E cells fed through set_conserved: projection + vacuum rule (P13), all three EOS kinds
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    rng = np.random.default_rng(5)
    sh = (6, 7, 16)
    E = rng.uniform(0.5, 2.0, sh); E[2, 3, 4:7] = 0.0; E[4, 1, 9] = -0.1
    M = [rng.uniform(-0.4, 0.4, sh) for _ in range(3)]
    M[0][1, 2, 3] = 5.0
    R = rng.uniform(0.1, 1.0, sh) * (1.0 if eos == "gamma" else 0.3)
    gam = 4.0 / 3.0 if eos == "gamma" else 5.0 / 3.0
    kw = dict(eos_mass=1.0 if eos == "mass" else 0.0, eos_table=inputs.eos_table("soft") if eos == "table" else None)
    o = oracle.Oracle(16, 7, 6, 0.1, 0.4, gam, **kw)
    o.set_conserved(E, *M, R); o.step(2)
    s = Shasta(16, 7, 6, 0.1, 0.4, gam, **kw)
    s.set_conserved(*[torch.from_numpy(a).cuda() for a in (E, *M, R)]); s.step(2)
    ref = dict(o.get_conserved()); ref.update(o.get_primitives())
    got = {k: v.cpu().numpy() for k, v in s.get_conserved().items()}
    got.update({k: v.cpu().numpy() for k, v in s.get_primitives().items()})
    assert_kernel_parity(got, ref, "vacuum", tol_cons=1e-11, tol_prim=1e-11)
    assert all(np.all(np.isfinite(v)) for v in got.values())


def test_vacuum_front_general_eos_sweep_by_sweep(oracle):
    # p = (Gamma-1)(e - m n), a ball of matter in an EXACT-zero exterior.  Run freely, GPU and oracle drift apart here by 6e-4
    # within two steps (Gamma-law: 2e-8, next test; the oracle's own strict / FMA builds: 4e-6): just outside the front a
    # cell's new E is a rounding residue of either sign -- vacuum (v = 0) on one side, a light-like cell (v ~ 1) on the
    # other -- and that velocity enters Q+- (eq. (15)) of a front cell of size 5e-4.  That is the method's sensitivity at an
    # exact vacuum, not an arithmetic difference: started from the SAME state, every single sweep of the first two steps
    # agrees to rounding, which is what this test pins; the free run must stay finite.
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    nx, ny, nz = 40, 36, 44
    z, y, x = np.meshgrid(np.arange(nz) - nz / 2, np.arange(ny) - ny / 2, np.arange(nx) - nx / 2, indexing="ij")
    inside = (x * x + y * y + z * z) < 36.0
    cur = np.stack([np.where(inside, 1.0, 0.0)] + [np.where(inside, 0.2 * f, 0.0) for f in (1.0, -0.5, 0.25)] + [np.where(inside, 0.3, 0.0)])
    gam, mass, lam = 5.0 / 3.0, 1.0, 0.4
    free = Shasta(nx, ny, nz, 0.1, lam, gam, eos_mass=mass)
    free.set_conserved(*[torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in cur])
    free.step(12)
    assert all(bool(torch.isfinite(v).all()) for v in list(free.get_conserved().values()) + list(free.get_primitives().values()))
    for axis in (0, 1, 2, 0, 2, 1):                                     # the sweeps of steps 0 and 1
        s = Shasta(nx, ny, nz, 0.1, lam, gam, eos_mass=mass)
        s.set_conserved(*[torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in cur])
        s.sweep(axis, 0)
        G = np.stack([v.cpu().numpy() for v in s.get_conserved().values()])
        A = np.moveaxis(cur, {0: 3, 1: 2, 2: 1}[axis], -1).copy()
        for i in range(A.shape[1]):
            for j in range(A.shape[2]):
                A[:, i, j, :] = oracle.sweep_pencil(A[:, i, j, :], axis, lam, gam, mass, oracle.OUTFLOW)[0]
        O = np.moveaxis(A, -1, {0: 3, 1: 2, 2: 1}[axis])
        assert np.max(np.abs(G - O)) <= 1e-13, axis
        cur = np.ascontiguousarray(O)


@pytest.mark.parametrize("shape", [(600, 1, 1), (1, 600, 1), (40, 36, 44)])
def test_matter_marching_into_exact_vacuum_stays_finite(oracle, shape):
    # E = 0 exterior (accepted by shasta_set_conserved): the numerical diffusion front carries E down through 1e-150,
    # where E^2 underflows, and through the subnormals.  The Gamma-law kernels call E < 2^-498 vacuum (c2p_is_vacuum);
    # nothing may become NaN or inf, and everything of visible size must still agree with the oracle.
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    nx, ny, nz = shape
    z, y, x = np.meshgrid(np.arange(nz) - nz / 2, np.arange(ny) - ny / 2, np.arange(nx) - nx / 2, indexing="ij")
    inside = (x * x + y * y + z * z) < 36.0
    E = np.where(inside, 1.0, 0.0)
    M = [np.where(inside, 0.2 * s, 0.0) for s in (1.0, -0.5, 0.25)]
    R = np.where(inside, 0.7, 0.0)
    steps = 100 if max(shape) == 600 else 12
    o = oracle.Oracle(nx, ny, nz, 0.1, 0.4, 4.0 / 3.0)
    o.set_conserved(E, *M, R); o.step(steps)
    s = Shasta(nx, ny, nz, 0.1, 0.4, 4.0 / 3.0)
    s.set_conserved(*[torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (E, *M, R)]); s.step(steps)
    ref = dict(o.get_conserved()); ref.update(o.get_primitives())
    got = {k: v.cpu().numpy() for k, v in s.get_conserved().items()}
    got.update({k: v.cpu().numpy() for k, v in s.get_primitives().items()})
    assert all(np.all(np.isfinite(v)) for v in got.values())
    assert (got["E"] > 0).sum() > inside.sum()
    # Agreement with the oracle is loose BY NATURE here: next to an exact-zero exterior the new E of a front cell is a
    # rounding residue of either sign (flux form here, eq. (17) as printed in the oracle), i.e. vacuum on one side and a
    # light-like cell on the other, and its velocity enters Q+- of a neighbour of visible size.  Measured 2e-8 after 12
    # steps; the oracle's own strict/FMA builds happen to agree (2.5e-14) because both use the same form.
    scale = np.max(np.abs(ref["E"]))
    for k in ("E", "Mx", "My", "Mz", "R", "e", "p"):
        assert np.max(np.abs(got[k] - ref[k])) <= 1e-6 * scale, k
    # E and R are never modified by Pi or the vacuum rule: their totals are conserved until the front reaches the boundary
    if max(shape) == 600:
        assert abs(got["E"].sum() - E.sum()) <= 1e-12 * E.sum() and abs(got["R"].sum() - R.sum()) <= 1e-12 * R.sum()


def test_step_split_and_step_index(oracle):
    c = inputs.random_state(20, 18, 16, seed=3, kind="rough")
    a, sa = parity.run_gpu(c, steps=7)
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"])
    s.set_state(*[torch.from_numpy(c[k]).cuda() for k in ("e", "n", "vx", "vy", "vz")])
    s.step(3); s.step(4)
    assert s.step_index == 7 and sa.step_index == 7
    for k, v in s.get_conserved().items():
        assert np.array_equal(v.cpu().numpy(), a[k]), k
    assert s.launch_count >= 21


@pytest.mark.parametrize("shape", [(70, 45, 50), (64, 33, 6), (37, 19, 23)])
@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
def test_deferred_primitives_of_x_last_steps(oracle, shape, bc):
    # a step whose last sweep runs along x leaves its primitives to the first sweep of the next step (emit = 2, DESIGN.md
    # 7.2); SHASTA_NO_DEFER writes them at once.  Same bits either way, wherever the call is cut (steps 3 and 4 of the
    # paper's table end with x), and both equal the oracle.
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    c = inputs.random_state(*shape, seed=31 + bc, kind="rough", boundary=bc)
    dev = [torch.from_numpy(c[k]).cuda() for k in ("e", "n", "vx", "vy", "vz")]
    for cuts in [(4,), (5,), (3, 1, 1, 2), (6, 6)]:
        res = []
        for nd in (0, 1):
            s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"], no_defer=nd)
            s.set_state(*dev)
            for n in cuts:
                s.step(n)
            r = {k: v.cpu().numpy() for k, v in s.get_conserved().items()}
            r.update({k: v.cpu().numpy() for k, v in s.get_primitives().items()})
            res.append((r, s.launch_count))
        for k in parity.CONS + parity.PRIM:
            assert np.array_equal(res[0][0][k], res[1][0][k]), (cuts, k)
        assert res[0][1] <= res[1][1]
        if cuts in [(5,), (6, 6)]:          # an x-last step followed by another step inside one call
            assert res[0][1] < res[1][1], "the deferred path must launch fewer kernels"
    ref, _ = parity.run_oracle(oracle, c, steps=5)
    got, _ = parity.run_gpu(c, steps=5)
    assert_kernel_parity(got, ref, f"deferred primitives shape {shape} bc {bc}")
    # single sweeps through the ABI: emit_primitives = 2 writes the primitives of the state BEFORE the sweep; they are
    # read back as stored (SHASTA_PRIMS_RAW: no refresh) and must equal, bit for bit, what the x sweep + element-wise
    # pass writes for that state
    from paper_1206_0919_b200 import shasta as sh
    mk = lambda: Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"])
    for axis in (1, 2):
        s, want = mk(), mk()
        s.set_state(*dev); want.set_state(*dev)
        want.sweep(0, 1)
        pw = {k: v.cpu().numpy() for k, v in want.get_primitives().items()}
        want.sweep(axis, 0)
        s.sweep(0, 0)
        s.sweep(axis, 2)
        s.set_option(sh.PRIMS_RAW, 1)
        for k, v in s.get_primitives().items():
            assert np.array_equal(v.cpu().numpy(), pw[k]), (axis, k)
        for k, v in s.get_conserved().items():
            assert np.array_equal(v.cpu().numpy(), want.get_conserved()[k].cpu().numpy()), (axis, k)
    with pytest.raises(Exception):
        mk().sweep(0, 2)


@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("shape", [(37, 19, 23), (64, 12, 10), (8, 5, 3)])
def test_batch_of_independent_events(oracle, shape, bc):
    # SHASTA_BATCH (row f4): B different events advanced by the same launches must equal B separate
    # oracle runs -- no cell of one event may see another event across the stacked z axis (both boundary rules)
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    B = 3
    cs = [inputs.random_state(*shape, seed=50 + b, kind="rough" if b != 1 else "smooth", boundary=bc) for b in range(B)]
    c = cs[0]
    s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"], batch=B)
    s.set_state(*[torch.from_numpy(np.stack([cb[k] for cb in cs])).cuda() for k in ("e", "n", "vx", "vy", "vz")])
    s.step(6)
    got = {k: v.cpu().numpy() for k, v in s.get_conserved().items()}
    got.update({k: v.cpu().numpy() for k, v in s.get_primitives().items()})
    tot = s.conserved_totals()
    for b in range(B):
        ref, o = parity.run_oracle(oracle, cs[b], steps=6)
        assert_kernel_parity({k: v[b] for k, v in got.items()}, ref, f"batch event {b} shape {shape} bc {bc}")
        t_ref = o.conserved_totals()
        assert np.max(np.abs(np.array(tot[b]) - t_ref)) <= 1e-12 * abs(t_ref[0])
    # one event of the batch alone gives the same bits as inside the batch
    one, _ = parity.run_gpu(cs[1], steps=6)
    for k in parity.CONS + parity.PRIM:
        assert np.array_equal(one[k], got[k][1]), k


@pytest.mark.parametrize("shape", [(40, 24, 20), (64, 1, 32), (1, 1, 80)])
def test_cuda_graph_cycles_same_bits(shape):
    # SHASTA_GRAPH: whole cycles of the axis table replayed as one CUDA graph ("orchestration overhead");
    # same kernels, so the same bits as launch-by-launch, from any starting phase and with a remainder
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    c = inputs.random_state(*shape, seed=61, kind="rough")
    dev = [torch.from_numpy(c[k]).cuda() for k in ("e", "n", "vx", "vy", "vz")]
    res = []
    for graph in (0, 1):
        s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"], graph=graph)
        s.set_state(*dev)
        s.step(2); s.step(15); s.step(6); s.step(1)
        r = {k: v.cpu().numpy() for k, v in s.get_conserved().items()}
        r.update({k: v.cpu().numpy() for k, v in s.get_primitives().items()})
        res.append((r, s.launch_count, s.graph_launch_count, s.step_index, s.diagnostics()))
    for k in parity.CONS + parity.PRIM:
        assert np.array_equal(res[0][0][k], res[1][0][k]), k
    assert res[0][2] == 0 and res[1][2] == 3, (res[0][2], res[1][2])        # 15 = 2 cycles + 3, 6 = 1 cycle
    assert res[0][3] == res[1][3] == 24 and res[0][4] == res[1][4]
    assert res[0][1] == res[1][1], "launch_count counts the kernels inside the replayed graphs"
    # a table of period 1 with an odd number of sweeps per period: a replayed chunk is then two periods (the state has to
    # return to the buffer it started in), and [2, 1, 0] ends every step with x (deferred primitives inside the graph)
    if min(shape) > 1:
        out = []
        for graph in (0, 1):
            s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"], graph=graph)
            s.set_sweep_table([2, 1, 0])
            s.set_state(*dev)
            s.step(7)
            r = {k: v.cpu().numpy() for k, v in s.get_conserved().items()}
            r.update({k: v.cpu().numpy() for k, v in s.get_primitives().items()})
            out.append((r, s.graph_launch_count))
        for k in parity.CONS + parity.PRIM:
            assert np.array_equal(out[0][0][k], out[1][0][k]), k
        assert out[1][1] == 3 and out[0][1] == 0


# ------------------------------------------------------------------ f1: tabled EOS (oracle pins: test_oracle_eos_table.py)
@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("kind", ["soft", "ideal"])
@pytest.mark.parametrize("shape", [(37, 19, 23), (64, 12, 10)])
def test_tabled_eos_kernel_level(oracle, bc, kind, shape):
    # shasta_set_eos_table (reading T1): every cons2prim of the path and set_state read P from
    # the bilinear table.  "soft": a nonlinear synthetic EOS; "ideal": the m = 1 ideal gas as a table, which must ALSO
    # equal the analytic m = 1 run (bilinear interpolation is exact on it)
    tab = inputs.eos_table(kind)
    c = inputs.random_state(*shape, seed=70 + bc, kind="rough", gamma=5.0 / 3.0, mass=0.0, boundary=bc)
    ref, _ = parity.run_oracle(oracle, c, steps=6, eos_table=tab)
    got, _ = parity.run_gpu(c, steps=6, eos_table=tab)
    assert_kernel_parity(got, ref, f"tabled EOS {kind} shape {shape} bc {bc}", tol_cons=1e-11, tol_prim=1e-11)
    if kind == "ideal":
        ca = dict(c, mass=1.0)
        ana, _ = parity.run_gpu(ca, steps=6)
        parity.assert_parity(got, ana, 1e-10, label="table of the ideal gas vs the analytic kernels")


def test_tabled_eos_cell_path_and_fp32(oracle):
    tab = inputs.eos_table("soft")
    c = inputs.random_state(24, 20, 28, seed=9, kind="smooth", gamma=5.0 / 3.0)
    ref, _ = parity.run_oracle(oracle, c, steps=2, eos_table=tab)
    got, _ = parity.run_gpu(c, steps=2, eos_table=tab, cell_path=1)
    assert_kernel_parity(got, ref, "tabled EOS, per-cell kernels", tol_cons=1e-11, tol_prim=1e-11)
    got32, _ = parity.run_gpu(c, steps=2, eos_table=tab, precision=32)
    for k, (emax, el1) in parity.field_errors(got32, ref).items():
        assert emax <= 2e-5 and el1 <= 2e-6, (k, emax, el1)


def test_options_state_rules_and_combinations(oracle):
    # argument / state checks of the round-2 entry points, and one run with everything on at once:
    # tabled EOS + batch of 2 + CUDA-graph cycles + deferred primitives
    import torch
    from paper_1206_0919_b200 import shasta as sh
    from paper_1206_0919_b200.shasta import Shasta, ShastaError
    tab = inputs.eos_table("soft")
    cs = [inputs.random_state(40, 12, 10, seed=80 + b, kind="rough", gamma=5.0 / 3.0) for b in range(2)]
    c = cs[0]
    s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], 0.0, batch=2, graph=1, eos_table=tab)
    s.set_state(*[torch.from_numpy(np.stack([cb[k] for cb in cs])).cuda() for k in ("e", "n", "vx", "vy", "vz")])
    s.step(13)
    assert s.graph_launch_count == 2
    got = {k: v.cpu().numpy() for k, v in s.get_conserved().items()}
    got.update({k: v.cpu().numpy() for k, v in s.get_primitives().items()})
    for b in range(2):
        ref, _ = parity.run_oracle(oracle, cs[b], steps=13, eos_table=tab)
        assert_kernel_parity({k: v[b] for k, v in got.items()}, ref, f"table+batch+graph event {b}", tol_cons=1e-11, tol_prim=1e-11)
    for bad in [lambda: s.set_option(sh.BATCH, 3), lambda: s.set_option(sh.PRECISION, 32), lambda: s.set_option(sh.EOS_MASS, 0.5),
                lambda: s.set_option(sh.GRAPH, 7), lambda: s.set_option(sh.DIFF, -1.0), lambda: s.set_option(99, 0.0),
                lambda: s.set_eos_table(np.zeros((1, 5)), 1.0, 1.0), lambda: s.set_eos_table(np.zeros((4, 5)), -1.0, 1.0),
                lambda: s.sweep(1, 3), lambda: s.sweep(0, 2)]:
        with pytest.raises(ShastaError):
            bad()
    s.set_eos_table(None, 0, 0)                      # back to the analytic EOS: the next primitives are recomputed with it
    p_ana = s.get_primitives()["p"].cpu().numpy()
    e_now = s.get_primitives()["e"].cpu().numpy()
    assert np.allclose(p_ana, (c["gamma"] - 1.0) * e_now, rtol=1e-12, atol=0)


def test_fp64_issue_rate_probe():
    # the measured numbers DESIGN.md 7.1 and bench.py's alu_roofline use (FP64_RESULTS_PER_CLK_SM = 60): the probe is
    # tests/probes/fp64_issue_probe.cu, built here with nvcc for sm_100a; its line goes to the parity record
    import json, os, subprocess, tempfile
    src = os.path.join(os.path.dirname(os.path.abspath(__file__)), "probes", "fp64_issue_probe.cu")
    with tempfile.TemporaryDirectory() as d:
        exe = os.path.join(d, "probe")
        subprocess.run(["nvcc", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-o", exe, src], check=True)
        out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout
    r = json.loads(out.strip().splitlines()[-1])
    parity.record("probe fp64 issue rate", {}, **r)
    assert 6.0 <= r["dfma_dependent_latency_cycles"] <= 12.0, r
    assert 54.0 <= r["fp64_results_per_clk_per_sm"] <= 66.0, r        # nominal 64 (16 lanes per sub-partition)


@pytest.mark.parametrize("mass", [0.0, 1.0])
def test_fp32_with_batch_graph_and_general_eos(oracle, mass):
    # the fp32 storage path through the same option combinations as fp64: batch of 2, graph cycles, both analytic EOS
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    cs = [inputs.random_state(40, 12, 10, seed=90 + b, kind="smooth", gamma=5.0 / 3.0, mass=mass) for b in range(2)]
    c = cs[0]
    s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], mass, batch=2, graph=1, precision=32)
    s.set_state(*[torch.from_numpy(np.stack([cb[k] for cb in cs])).cuda() for k in ("e", "n", "vx", "vy", "vz")])
    s.step(7)
    got = {k: v.cpu().numpy() for k, v in s.get_conserved().items()}
    got.update({k: v.cpu().numpy() for k, v in s.get_primitives().items()})
    assert s.graph_launch_count == 1
    for b in range(2):
        ref, _ = parity.run_oracle(oracle, cs[b], steps=7)
        for k, (emax, el1) in parity.field_errors({k: v[b] for k, v in got.items()}, ref).items():
            assert emax <= 2e-4 and el1 <= 5e-6, (b, k, emax, el1)      # fp32 storage: a few 1e-7 per operation, 7 steps


def test_host_buffer_entry_points(oracle):
    c = inputs.random_state(21, 17, 13, seed=8, kind="smooth")
    ref, _ = parity.run_oracle(oracle, c, steps=2)
    got, _ = parity.run_gpu(c, steps=2, host_io=True)
    assert_kernel_parity(got, ref, "host io")


def test_conserved_totals_periodic(oracle):
    c = inputs.spherical_riemann(32, steps=12)
    ref, o = parity.run_oracle(oracle, c)
    got, s = parity.run_gpu(c)
    t_ref = o.conserved_totals()
    t = np.array(s.conserved_totals())
    assert np.max(np.abs(t - t_ref)) <= 1e-12 * abs(t_ref[0])
    # conservation on the GPU path itself: E and R to 1e-12 relative
    s0 = parity.run_gpu(c, steps=0)[1].conserved_totals()
    assert abs(t[0] - s0[0]) <= 1e-12 * abs(s0[0]) and abs(t[4] - s0[4]) <= 1e-12 * abs(s0[4])
    assert np.max(np.abs(t[1:4])) <= 1e-12 * abs(s0[0])


# ------------------------------------------------------------------ f2: scheme variants (oracle pins: test_oracle_variants.py)
@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("diff", [0.0, 0.5])
def test_variant_diff_fused_kernels(oracle, bc, diff):
    # `diff` and its diff = 0 case "n/af" run in the fused kernels: ragged shape
    c = inputs.random_state(37, 19, 23, seed=21 + bc, kind="rough", boundary=bc)
    ref, _ = parity.run_oracle(oracle, c, steps=2, diff=diff)
    got, _ = parity.run_gpu(c, steps=2, diff=diff)
    assert_kernel_parity(got, ref, f"diff {diff} bc {bc}")
    c = inputs.random_state(64, 33, 6, seed=22 + bc, kind="rough", boundary=bc)      # TMA-fed shapes
    ref, _ = parity.run_oracle(oracle, c, steps=2, diff=diff)
    got, _ = parity.run_gpu(c, steps=2, diff=diff)
    assert_kernel_parity(got, ref, f"diff {diff} bc {bc} (tma)")


@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("predictor,diff", [(1, 1.0), (1, 0.5), (0, 1.0)])
def test_variant_predictor_per_cell_kernels(oracle, bc, predictor, diff):
    # R2 predictor and, as a cross-check of the per-cell path itself, the default scheme through it
    c = inputs.random_state(37, 19, 23, seed=31 + bc, kind="rough", boundary=bc)
    ref, _ = parity.run_oracle(oracle, c, steps=2, predictor=predictor, diff=diff)
    got, s = parity.run_gpu(c, steps=2, predictor=predictor, diff=diff, cell_path=1)
    assert s.kernel_name(0) == "sweep_cell_kernel"
    assert_kernel_parity(got, ref, f"predictor {predictor} diff {diff} bc {bc}")
    for shape in ((5, 1, 9), (2, 3, 4), (64, 1, 1)):
        c = inputs.random_state(*shape, seed=7, kind="rough", boundary=bc)
        ref, _ = parity.run_oracle(oracle, c, steps=3, predictor=predictor, diff=diff)
        got, _ = parity.run_gpu(c, steps=3, predictor=predictor, diff=diff, cell_path=1)
        assert_kernel_parity(got, ref, f"predictor {predictor} shape {shape}")


@pytest.mark.parametrize("predictor,diff,cell", [(0, 0.0, 0), (0, 0.5, 0), (1, 1.0, 1), (0, 1.0, 1)])
def test_variants_config1(oracle, predictor, diff, cell):
    c = inputs.shock_tube(400, 0.01)
    ref, o = parity.run_oracle(oracle, c, predictor=predictor, diff=diff)
    got, s = parity.run_gpu(c, predictor=predictor, diff=diff, cell_path=cell)
    rep = parity.field_report(got, ref)
    parity.record(f"config1 eR=0.01 variant predictor={predictor} diff={diff} cell_path={cell}", rep, steps=c["steps"])
    parity.assert_parity(got, ref, TOL64, label=f"config1 predictor {predictor} diff {diff}")


def test_variant_general_eos_per_cell(oracle):
    c = inputs.random_state(24, 20, 28, seed=4, kind="rough", gamma=5.0 / 3.0, mass=1.0, boundary=inputs.PERIODIC)
    ref, _ = parity.run_oracle(oracle, c, steps=3, predictor=1)
    got, _ = parity.run_gpu(c, steps=3, predictor=1)
    assert_kernel_parity(got, ref, "general EOS R2", tol_cons=1e-11, tol_prim=1e-11)


# explicit antidiffusion (PAPER.md:123 footnote 1; oracle pin: test_explicit_antidiffusion_leaves_the_fourth_difference_at_rest)
@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("diff", [1.0, 0.5])
def test_variant_explicit_antidiffusion_fused_kernels(oracle, bc, diff):
    c = inputs.random_state(37, 19, 23, seed=41 + bc, kind="rough", boundary=bc)     # ragged: cp.async tiles
    ref, _ = parity.run_oracle(oracle, c, steps=2, diff=diff, antidiffusion=1)
    got, s = parity.run_gpu(c, steps=2, diff=diff, antidiffusion=1)
    assert s.kernel_name(0).startswith("sweep_x2_kernel")
    assert_kernel_parity(got, ref, f"explicit antidiffusion diff {diff} bc {bc}")
    # the variant is a different scheme, not a no-op: the default result is far from it at this tolerance
    dflt, _ = parity.run_gpu(c, steps=2, diff=diff)
    assert parity.field_errors(dflt, ref)["E"][0] > 1e-6
    c = inputs.random_state(64, 33, 6, seed=42 + bc, kind="rough", boundary=bc)      # TMA-fed shapes
    ref, _ = parity.run_oracle(oracle, c, steps=2, diff=diff, antidiffusion=1)
    got, _ = parity.run_gpu(c, steps=2, diff=diff, antidiffusion=1)
    assert_kernel_parity(got, ref, f"explicit antidiffusion diff {diff} bc {bc} (tma)")


@pytest.mark.parametrize("predictor", [0, 1])
def test_variant_explicit_antidiffusion_per_cell_kernels(oracle, predictor):
    # with the R2 predictor the half step runs eqs. (18)-(22) too: the variant applies there as well
    for bc in (inputs.OUTFLOW, inputs.PERIODIC):
        c = inputs.random_state(37, 19, 23, seed=43 + bc, kind="rough", boundary=bc)
        ref, _ = parity.run_oracle(oracle, c, steps=2, predictor=predictor, antidiffusion=1)
        got, s = parity.run_gpu(c, steps=2, predictor=predictor, antidiffusion=1, cell_path=1)
        assert s.kernel_name(0) == "sweep_cell_kernel"
        assert_kernel_parity(got, ref, f"explicit antidiffusion per-cell predictor {predictor} bc {bc}")


def test_variant_explicit_antidiffusion_general_eos_batch_and_graph(oracle):
    # general-EOS kernels (S3 in the consumer), two events per launch, graph replay of whole table cycles
    cs = [inputs.random_state(24, 20, 28, seed=44 + b, kind="rough", gamma=5.0 / 3.0, mass=1.0, boundary=inputs.PERIODIC)
          for b in range(2)]
    refs = [parity.run_oracle(oracle, c, steps=6, antidiffusion=1)[0] for c in cs]
    c2 = dict(cs[0])
    for k in ("e", "n", "vx", "vy", "vz"):
        c2[k] = np.stack([c[k] for c in cs])
    got, s = parity.run_gpu(c2, steps=6, antidiffusion=1, batch=2, graph=1)
    assert s.graph_launch_count >= 1
    for b in range(2):
        assert_kernel_parity({k: v[b] for k, v in got.items()}, refs[b], f"explicit antidiffusion general EOS event {b}",
                             tol_cons=1e-11, tol_prim=1e-11)


def test_variant_explicit_antidiffusion_config1(oracle):
    c = inputs.shock_tube(400, 0.01)
    ref, _ = parity.run_oracle(oracle, c, antidiffusion=1)
    got, _ = parity.run_gpu(c, antidiffusion=1)
    rep = parity.field_report(got, ref)
    parity.record("config1 eR=0.01 variant antidiffusion=explicit", rep, steps=c["steps"])
    parity.assert_parity(got, ref, TOL64, label="config1 explicit antidiffusion")


# ------------------------------------------------------------------ the step / graph / deferral state machine
def test_random_call_sequences_equal_plain_stepping():
    # seeded random sequences of step(k), option changes (launch mode, deferral of the x-last primitives) and reads in between
    # must land on the bits of one step at a time with no graph and no deferral: shasta_step's bookkeeping (cached graph
    # cycles per phase, pending primitive output, buffer parity) may not leak into the results
    import torch
    from paper_1206_0919_b200 import shasta as sh
    from paper_1206_0919_b200.shasta import Shasta
    rng = np.random.default_rng(1234)
    for trial in range(12):
        shape = [(24, 20, 28), (64, 32, 16), (37, 19, 23)][trial % 3]
        kw = dict(gamma=5.0 / 3.0, mass=1.0) if trial % 2 else {}
        bc = [inputs.OUTFLOW, inputs.PERIODIC][(trial // 2) % 2]
        c = inputs.random_state(*shape, seed=trial, kind="rough", boundary=bc, **kw)
        st = [torch.from_numpy(c[k]).cuda() for k in ("e", "n", "vx", "vy", "vz")]
        total = int(rng.integers(5, 20))
        ref = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"], graph=0, no_defer=1)
        ref.set_state(*st)
        for _ in range(total):
            ref.step(1)
        want = {**ref.get_conserved(), **ref.get_primitives()}
        a = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"])
        a.set_state(*st)
        done, log = 0, []
        while done < total:
            op = int(rng.integers(0, 6))
            if op == 0:
                g = int(rng.integers(0, 3)); a.set_option(sh.GRAPH, g); log.append(f"graph={g}")
            elif op == 1:
                nd = int(rng.integers(0, 2)); a.set_option(sh.NO_DEFER, nd); log.append(f"no_defer={nd}")
            elif op == 2:
                a.get_primitives(); log.append("prims")
            elif op == 3:
                a.get_conserved(); a.conserved_totals(); log.append("cons")
            else:
                k = int(min(rng.integers(1, 9), total - done)); a.step(k); done += k; log.append(f"step{k}")
        got = {**a.get_conserved(), **a.get_primitives()}
        assert a.step_index == total
        for k in want:
            assert torch.equal(got[k], want[k]), (trial, k, log)


# ------------------------------------------------------------------ parameter range of shasta_create
@pytest.mark.parametrize("lam", [0.5, 0.25, 0.05])
@pytest.mark.parametrize("gamma", [1.2, 5.0 / 3.0, 1.8])
def test_lambda_and_gamma_range(oracle, lam, gamma):
    # lambda up to the stability limit 0.5 (eq. (15)'s denominators stay > 0) and down to slow flows; Gamma = 1.2 and 5/3
    # run the closed-form kernels (5/3 is their limit), Gamma = 1.8 the Newton kernels with m = 0 (shasta_create wants
    # 1 < Gamma < 2: c_s^2 = Gamma - 1 < 1)
    # Not beyond 1.8: in a cell at the causality clamp the contraction factor of the paper's fixed-point map is
    # Gamma - 1, and the ORACLE's 200 iterations (reading G9) then stop short of the root -- 0.9^200 = 7e-10 at Gamma = 1.9,
    # measured 7e-11 in v against bisection, 6e-6 in n = R sqrt(1 - v^2) -- while the kernels' bracketed Newton reaches it.
    c = inputs.random_state(37, 19, 23, seed=int(100 * lam + 10 * gamma), kind="rough", gamma=gamma, boundary=inputs.PERIODIC)
    c["lam"] = lam
    ref, _ = parity.run_oracle(oracle, c, steps=2)
    got, s = parity.run_gpu(c, steps=2)
    tol = 1e-12 if gamma < 1.7 else 1e-11
    assert_kernel_parity(got, ref, f"lambda {lam} gamma {gamma}", tol_cons=tol, tol_prim=tol)


# ------------------------------------------------------------------ symmetries of the scheme on the GPU path itself (no oracle)
def test_energy_scale_homogeneity_is_bitwise():
    # p = (Gamma-1) e, m = 0: eqs. (9)-(22) are homogeneous of degree one in (E, M) and leave R alone, and v depends on M/E
    # only.  Scaling e by a power of two must therefore scale E, M, e, p by it EXACTLY and leave R, n, v untouched -- through
    # the closed-form cons2prim (E^2, |M|^2 up to 2^+-400), the limiter and the causality clamp.  Absolute thresholds
    # (vacuum 2^-498) are far away.
    c = inputs.random_state(40, 24, 13, seed=91, kind="rough", boundary=inputs.PERIODIC)
    base, _ = parity.run_gpu(c, steps=3)
    for k in (200, -200):
        sc = 2.0 ** k
        cs = dict(c)
        cs["e"] = c["e"] * sc
        got, _ = parity.run_gpu(cs, steps=3)
        for f in ("E", "Mx", "My", "Mz", "e", "p"):
            assert np.array_equal(got[f], base[f] * sc), (k, f)
        for f in ("R", "n", "vx", "vy", "vz"):
            assert np.array_equal(got[f], base[f]), (k, f)
    # p = (Gamma-1)(e - m n): homogeneous in (e, n) together -- the Newton kernels (MUFU seeds, bracket, warp votes) too
    c = inputs.random_state(24, 20, 28, seed=93, kind="rough", gamma=5.0 / 3.0, mass=1.0, boundary=inputs.PERIODIC)
    base, _ = parity.run_gpu(c, steps=3)
    for k in (200, -200):
        sc = 2.0 ** k
        cs = dict(c)
        cs["e"], cs["n"] = c["e"] * sc, c["n"] * sc
        got, _ = parity.run_gpu(cs, steps=3)
        for f in ("E", "Mx", "My", "Mz", "R", "e", "p", "n"):
            assert np.array_equal(got[f], base[f] * sc), (k, f)
        for f in ("vx", "vy", "vz"):
            assert np.array_equal(got[f], base[f]), (k, f)


@pytest.mark.parametrize("eos", ["gamma", "mass", "table"])
@pytest.mark.parametrize("shape,shift", [((37, 19, 23), (5, 3, 7)), ((64, 32, 16), (33, 1, 9)), ((130, 6, 5), (64, 2, 1))])
def test_translation_invariance_is_bitwise(eos, shape, shift):
    # periodic box: the state rolled by (sx, sy, sz) cells gives the result rolled by the same shift, bit for bit -- whichever
    # tile, group phase, segment or lane a cell lands in, and whether its neighbours arrive through the ghost wrap or not
    nx, ny, nz = shape
    tab = inputs.eos_table("soft") if eos == "table" else None
    c = inputs.random_state(nx, ny, nz, seed=95, kind="rough", gamma=5.0 / 3.0, mass=1.0 if eos == "mass" else 0.0,
                            boundary=inputs.PERIODIC)
    base, _ = parity.run_gpu(c, steps=6, eos_table=tab)
    sx, sy, sz = shift
    cr = dict(c)
    for k in ("e", "n", "vx", "vy", "vz"):
        cr[k] = np.ascontiguousarray(np.roll(c[k], (sz, sy, sx), axis=(0, 1, 2)))
    got, _ = parity.run_gpu(cr, steps=6, eos_table=tab)
    for k in parity.CONS + parity.PRIM:
        assert np.array_equal(got[k], np.roll(base[k], (sz, sy, sx), axis=(0, 1, 2))), k


@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_state_uniform_along_an_axis_stays_uniform_bitwise(axis, bc):
    # a state that does not depend on one coordinate (and has no velocity along it) keeps that property exactly: the sweep
    # along that axis must be the identity in every cell, edge cells and ghost cells included, and the other sweeps must treat
    # every copy alike (P11 of the oracle, here on the kernels: 2-D flow in a 3-D grid)
    shape = [29, 21, 18]                                   # (nz, ny, nx)
    c2 = inputs.random_state(*[1 if a == axis else n for a, n in ((0, shape[2]), (1, shape[1]), (2, shape[0]))], seed=96,
                             kind="rough", boundary=bc)
    c = dict(c2)
    reps = [1, 1, 1]
    reps[2 - axis] = shape[2 - axis]
    for k in ("e", "n", "vx", "vy", "vz"):
        c[k] = np.ascontiguousarray(np.tile(c2[k], reps))
    c["v" + "xyz"[axis]] = np.zeros_like(c["e"])
    c["nz"], c["ny"], c["nx"] = c["e"].shape
    got, _ = parity.run_gpu(c, steps=6)
    for k in parity.CONS + parity.PRIM:
        a = np.moveaxis(got[k], 2 - axis, 0)
        assert np.array_equal(a, np.broadcast_to(a[0], a.shape)), k
    assert float(np.abs(got["v" + "xyz"[axis]]).max()) == 0.0


@pytest.mark.parametrize("shape", [(37, 19, 23), (64, 32, 8)])
def test_axis_permutation_covariance_is_bitwise(shape):
    # the x kernel (rows in swizzled 4-cell tiles) and the y/z kernel (x across the lanes) are different code around the same
    # per-pencil arithmetic: three x sweeps of a conserved state = three y (z) sweeps of the state with the axes rotated
    # CYCLICALLY (so that the two transverse momenta keep their order in |M|^2 = M_par^2 + (M_perp1^2 + M_perp2^2), which is
    # not associative).  Starts from conserved fields: prim2cons sums v^2 in natural order, which a rotation changes by an ulp.
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    nx, ny, nz = shape
    c = inputs.random_state(nx, ny, nz, seed=92, kind="rough", boundary=inputs.PERIODIC)
    U0 = parity.run_gpu(c, steps=0)[0]

    def sweeps(U, dims, axis):
        s = Shasta(dims[2], dims[1], dims[0], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"])
        s.set_conserved(*[torch.from_numpy(np.ascontiguousarray(U[k])).cuda() for k in parity.CONS])
        s.set_sweep_table([axis] * 3)
        s.step(1)
        return {k: v.cpu().numpy() for k, v in s.get_conserved().items()}

    ref = sweeps(U0, (nz, ny, nx), 0)
    # arrays are (z, y, x).  axis 1: (z', y', x') = (y, x, z);  axis 2: (z', y', x') = (x, z, y);  old component -> new name
    for axis, perm, new_of in ((1, (1, 2, 0), {"x": "y", "y": "z", "z": "x"}), (2, (2, 0, 1), {"x": "z", "y": "x", "z": "y"})):
        Ut = {k: np.transpose(U0[k], perm) for k in ("E", "R")}
        for old, new_ in new_of.items():
            Ut["M" + new_] = np.transpose(U0["M" + old], perm)
        got = sweeps(Ut, Ut["E"].shape, axis)
        back = tuple(np.argsort(perm))
        names = {"E": "E", "R": "R", **{"M" + old: "M" + new_ for old, new_ in new_of.items()}}
        for k, kt in names.items():
            assert np.array_equal(np.transpose(got[kt], back), ref[k]), (axis, k)


# ------------------------------------------------------------------ long runs (no oracle: properties that hold at any length)
@pytest.mark.parametrize("precision", [64, 32])
def test_long_runs_stay_finite_causal_and_conservative(precision):
    # (a) periodic box, rough state, 1500 steps: E and R are conserved by the flux form (eqs. (17), (22)) -- to rounding in
    # fp64, to the fp32 storage rounding otherwise -- and every primitive stays finite with |v| < 1;  (b) hotspots
    # expanding into a near-vacuum exterior through outflow faces, 600 steps: the front runs at the causality clamp
    # (|M| <= (1 - 1e-12) E, readings G6-G8), nothing becomes NaN, e >= 0
    import torch
    from paper_1206_0919_b200.shasta import Shasta

    def run(c, steps, chunk):
        s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"], precision=precision)
        s.set_state(*[torch.from_numpy(c[k]).cuda() for k in ("e", "n", "vx", "vy", "vz")])
        t0 = np.array(s.conserved_totals())
        for _ in range(0, steps, chunk):
            s.step(chunk)
            p = s.get_primitives()
            assert all(bool(torch.isfinite(v).all()) for v in p.values())
            assert float((p["vx"] ** 2 + p["vy"] ** 2 + p["vz"] ** 2).max()) < 1.0
            assert float(p["e"].min()) >= 0.0 and float(p["p"].min()) >= 0.0 and float(p["n"].min()) >= 0.0
        return t0, np.array(s.conserved_totals()), s

    t0, t1, _ = run(inputs.random_state(48, 48, 48, seed=3, kind="rough", boundary=inputs.PERIODIC), 1500, 500)
    tol = 1e-12 if precision == 64 else 1e-6
    assert abs(t1[0] - t0[0]) <= tol * abs(t0[0]) and abs(t1[4] - t0[4]) <= tol * abs(t0[4])
    t0, t1, s = run(inputs.hotspots(64, steps=0), 600, 200)
    assert t1[0] < t0[0] and s.diagnostics()[0] > 0          # matter left through the faces; the clamp did fire at the front


# ------------------------------------------------------------------ z-slab decomposition (host logic: test_zslab.py)
@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
@pytest.mark.parametrize("world,zero_copy", [(2, True), (3, True), (3, False), (7, True)])     # 7: slabs of 4-5 planes, the minimum
def test_zslab_in_process_equals_the_single_domain_run(oracle, bc, world, zero_copy):
    # the slabs of one event as `world` handles on this GPU, planes carried by shasta_get_planes / shasta_set_planes:
    # same kernels, same neighbourhood for every owned cell -> the same bits as one handle over the whole grid
    import torch
    from paper_1206_0919_b200 import zslab
    c = inputs.random_state(40, 24, 29, seed=51 + bc, kind="rough", boundary=bc)
    one, s1 = parity.run_gpu(c, steps=6)
    slabs = [zslab.make_gpu_slab(c, world, r) for r in range(world)]
    assert [sl.s.nz for sl in slabs] == [sl.lay.nz_local for sl in slabs]
    if not zero_copy:                                  # the staged exchange: a solver without plane_views
        class Staged:
            def __init__(self, s):
                self.sweep, self.get_planes, self.set_planes, self.get_primitives = s.sweep, s.get_planes, s.set_planes, s.get_primitives
        for sl in slabs:
            sl.s = Staged(sl.s)
    zslab.step_in_process(slabs, 6)
    U = torch.cat([sl.owned_conserved() for sl in slabs], dim=1).cpu().numpy()
    for f, k in enumerate(parity.CONS):
        assert np.array_equal(U[f], one[k]), k
    prims = [sl.s.get_primitives() for sl in slabs]
    for k in parity.PRIM:
        assert np.array_equal(torch.cat([sl.owned(p[k]) for sl, p in zip(slabs, prims)], dim=0).cpu().numpy(), one[k]), k
    ref, _ = parity.run_oracle(oracle, c, steps=6)
    assert_kernel_parity(dict(zip(parity.CONS, U), **{k: one[k] for k in parity.PRIM}), ref, f"zslab world {world} bc {bc}")
    # totals: every slab sums its owned planes (no process group here: no all-reduce), the sum is the event's
    tot = sum(zslab.conserved_totals_distributed(sl, c["dx"]).cpu().numpy() for sl in slabs)
    t1 = np.array(s1.conserved_totals())
    assert np.max(np.abs(tot - t1)) <= 1e-12 * abs(t1[0])


def test_zslab_fp32_storage_and_general_eos():
    # the slab machinery is storage- and EOS-agnostic: fp32 fields travel as fp32 plane views; config-3-like EOS with a table cycle
    import torch
    from paper_1206_0919_b200 import zslab
    c = inputs.random_state(40, 24, 21, seed=61, kind="rough", boundary=inputs.PERIODIC)
    one, _ = parity.run_gpu(c, steps=6, precision=32)
    slabs = [zslab.make_gpu_slab(c, 2, r, precision=32) for r in range(2)]
    assert slabs[0].s.plane_views(0, 1)[0].dtype == torch.float32
    zslab.step_in_process(slabs, 6)
    U = torch.cat([sl.owned_conserved() for sl in slabs], dim=1).cpu().numpy()
    for f, k in enumerate(parity.CONS):
        assert np.array_equal(U[f], one[k]), k
    c = inputs.random_state(24, 20, 17, seed=62, kind="rough", gamma=5.0 / 3.0, mass=1.0, boundary=inputs.OUTFLOW)
    one, _ = parity.run_gpu(c, steps=6)
    slabs = [zslab.make_gpu_slab(c, 2, r) for r in range(2)]
    zslab.step_in_process(slabs, 6)
    U = torch.cat([sl.owned_conserved() for sl in slabs], dim=1).cpu().numpy()
    # bitwise here too: a cell of the Newton loop stops moving with its own first converged step, whatever the cells it
    # shares the loop (and the warp vote) with -- which depends on where the march started
    for f, k in enumerate(parity.CONS):
        assert np.array_equal(U[f], one[k]), k


@pytest.mark.parametrize("shape", [(40, 24, 13), (64, 33, 12)])
def test_active_planes_restrict_the_x_and_y_sweeps(shape):
    # shasta_set_active_planes: x and y sweeps update planes [3, 9) only -- the same bits there as the full sweep -- and the
    # z sweep still covers every plane (ragged cp.async shapes and TMA-fed ones)
    import torch
    from paper_1206_0919_b200.shasta import Shasta, ShastaError
    nx, ny, nz = shape
    c = inputs.random_state(nx, ny, nz, seed=71, kind="rough", boundary=inputs.PERIODIC)
    st = [torch.from_numpy(c[k]).cuda() for k in ("e", "n", "vx", "vy", "vz")]
    for axis in (0, 1, 2):
        full = Shasta(nx, ny, nz, c["dx"], c["lam"], c["gamma"], c["boundary"])
        part = Shasta(nx, ny, nz, c["dx"], c["lam"], c["gamma"], c["boundary"])
        part.set_active_planes(3, 9)
        for s in (full, part):
            s.set_state(*st)
            s.sweep(axis, 1)
        a, b = full.get_planes(0, nz), part.get_planes(0, nz)
        lo, hi = (0, nz) if axis == 2 else (3, 9)
        assert torch.equal(a[:, lo:hi], b[:, lo:hi]), axis
        pa, pb = full.get_primitives(), part.get_primitives()
        assert all(torch.equal(pa[k][lo:hi], pb[k][lo:hi]) for k in pa), axis
    with pytest.raises(ShastaError):
        part.set_active_planes(5, 5)
    with pytest.raises(ShastaError):
        part.set_active_planes(0, nz + 1)
    part.set_active_planes(0, nz)


def test_planes_round_trip_and_errors():
    import torch
    from paper_1206_0919_b200.shasta import Shasta, ShastaError
    c = inputs.random_state(12, 10, 9, seed=5, kind="rough")
    for precision in (64, 32):
        s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], precision=precision)
        with pytest.raises(ShastaError):
            s.get_planes(0, 1)                                   # no state yet
        s.set_state(*[torch.from_numpy(c[k]).cuda() for k in ("e", "n", "vx", "vy", "vz")])
        U = torch.stack(list(s.get_conserved().values()))
        assert torch.equal(s.get_planes(2, 4), U[:, 2:6])
        views = s.plane_views(2, 4)                              # aliases of the state buffer, storage dtype
        assert views[0].dtype == (torch.float64 if precision == 64 else torch.float32)
        assert all(torch.equal(v.double(), U[f, 2:6]) for f, v in enumerate(views))
        views[4].mul_(2.0)
        assert torch.equal(s.get_planes(2, 4)[4], 2.0 * U[4, 2:6])
        views[4].mul_(0.5)
        s.set_planes(5, U[:, 0:3].contiguous())
        V = torch.stack(list(s.get_conserved().values()))
        assert torch.equal(V[:, 5:8], U[:, 0:3]) and torch.equal(V[:, :5], U[:, :5]) and torch.equal(V[:, 8:], U[:, 8:])
        for z0, n in ((-1, 2), (7, 3), (0, 10)):
            with pytest.raises(ShastaError):
                s.get_planes(z0, n)
        assert s.get_planes(9, 0).shape[1] == 0
    b = Shasta(8, 8, 8, 0.1, 0.4, 4.0 / 3.0, batch=2)
    b.set_state(*[torch.full((2, 8, 8, 8), v, dtype=torch.float64, device="cuda") for v in (1.0, 1.0, 0.0, 0.0, 0.0)])
    with pytest.raises(ShastaError):
        b.get_planes(0, 1)


# ------------------------------------------------------------------ T2: the configs
# Bars (north_star): fp64 err_max <= 1e-10 per field, err_L1 reported (expected <= 1e-12).  Configs 3 and 4
# amplify rounding noise: two equally valid fp64 evaluations of the ORACLE (strict vs FMA-contracted build) already
# differ by more than 1e-10 in some fields there (R and the primitives of config 4, p of config 3), so the bar is
# max(1e-10, 2 x that floor): the GPU path is one more valid evaluation and must sit at the floor, not above it.
# E and the momenta are held to 1e-10 outright.  Every achieved number goes to gpurun_out/parity_r2.json.
OUTRIGHT = ("E", "Mx", "My", "Mz")
FLOOR_FACTOR = 2.0


def _check_config(oracle, name, c, got, ref, s=None, o=None, floor=True, l1=True, outright=OUTRIGHT, factor=FLOOR_FACTOR,
                  **meta):
    fl = parity.noise_floor(oracle, c, ref, steps=meta.get("steps")) if floor else None
    errs = parity.field_errors(got, ref)
    bar = {k: (max(TOL64, factor * fl[k][0]) if fl else TOL64) for k in errs}
    for k in outright:
        bar[k] = TOL64
    rep = parity.field_report(got, ref, fl, bar)
    if s is not None and o is not None:
        meta["pi_fired_gpu_oracle"] = [s.diagnostics()[0], o.diagnostics()[0]]
    meta["north_star_1e-10_met"] = bool(all(v[0] <= TOL64 for v in errs.values()))
    parity.record(name, rep, **meta)
    bad = {k: (v, bar[k]) for k, v in errs.items() if not v[0] <= bar[k]}
    assert not bad, f"{name}: (err_max, err_L1), bar: {bad}; all: {rep}"
    if l1:
        badl = {k: v for k, v in errs.items() if not v[1] <= max(1e-12, FLOOR_FACTOR * (fl[k][1] if fl else 0.0))}
        assert not badl, f"{name}: err_L1 above max(1e-12, 2 x floor): {badl}; all: {rep}"
    return rep


def test_config1_shock_tube(oracle):
    for e_right in (0.01, 1e-8):
        c = inputs.shock_tube(400, e_right)
        ref, o = parity.run_oracle(oracle, c)
        got, s = parity.run_gpu(c)
        _check_config(oracle, f"config1 eR={e_right}", c, got, ref, s, o, floor=False, steps=c["steps"], grid=[400, 1, 1])
        assert s.diagnostics()[0] == o.diagnostics()[0]


def test_config1_along_y_and_z(oracle):
    for axis in (1, 2):
        c = inputs.shock_tube(400, 0.01, axis=axis, transverse=3)
        ref, _ = parity.run_oracle(oracle, c)
        got, _ = parity.run_gpu(c)
        parity.assert_parity(got, ref, TOL64, label=f"config1 axis {axis}")


def test_config2_fireball(oracle):
    c = inputs.fireball(64, steps=100)
    ref, o = parity.run_oracle(oracle, c)
    got, s = parity.run_gpu(c)
    _check_config(oracle, "config2 fireball 64^3", c, got, ref, s, o, floor=False, steps=100, grid=[64, 64, 64])


def test_config3_spherical_riemann(oracle):
    c = inputs.spherical_riemann(128, steps=100)
    ref, o = parity.run_oracle(oracle, c)
    got, s = parity.run_gpu(c)
    # strong spherical shock: the rounding-noise floor of the step map itself reaches ~1e-10 in p
    # (p = (Gamma-1)(e - n) cancels)
    _check_config(oracle, "config3 spherical riemann 128^3", c, got, ref, s, o, steps=100, grid=[128, 128, 128])
    t = np.array(s.conserved_totals())
    t0 = np.array(parity.run_gpu(c, steps=0)[1].conserved_totals())
    assert abs(t[0] - t0[0]) <= 1e-12 * t0[0] and abs(t[4] - t0[4]) <= 1e-12 * t0[4]
    assert np.max(np.abs(t[1:4])) <= 1e-12 * t0[0]


def test_config4_hotspots_reduced(oracle):
    # same box, flow and hotspots on 96^3 for the full 200 steps (the 256^3 runs are below)
    c = inputs.hotspots(96, steps=200)
    ref, o = parity.run_oracle(oracle, c)
    got, s = parity.run_gpu(c)
    _check_config(oracle, "config4 hotspots 96^3 (dx=0.267)", c, got, ref, s, o, steps=200, grid=[96, 96, 96])


def test_config4_hotspots_crop_at_full_resolution(oracle):
    # the 256^3 state at its own dx = 0.1 fm on the 96^3 sub-box touching the +z face (gamma up to 12 at
    # the outflow boundary), 100 steps
    c = inputs.hotspots_crop(96, steps=100)
    ref, o = parity.run_oracle(oracle, c)
    got, s = parity.run_gpu(c)
    _check_config(oracle, "config4 crop 96^3 of 256^3 at +z face", c, got, ref, s, o, steps=100, grid=[96, 96, 96])


FP32_STEPS = (12, 24, 48, 96, 200)


def _fp32_study(oracle, name, c):
    """f3: err_L1 of the fp32-storage path (fp32 transport, fp64 cons2prim) vs the fp64 oracle as the run proceeds."""
    out = {}
    for st in FP32_STEPS:
        if st > c["steps"]:
            break
        ref, _ = parity.run_oracle(oracle, c, steps=st)
        got, _ = parity.run_gpu(c, steps=st, precision=32)
        rep = parity.field_report(got, ref)
        parity.record(f"{name} fp32 {st} steps", rep, steps=st, precision=32, grid=[c["nx"], c["ny"], c["nz"]])
        out[st] = {k: v["err_L1"] for k, v in rep.items()}
    return out


def test_config4_hotspots_fp32_48_steps(oracle):
    # fp32 storage + transport, fp64 cons2prim.  north_star: err_L1 <= 1e-4 vs the fp64 oracle: holds through 48 steps
    # (and through 96: recorded); the error grows with the step count exactly as the fp64 rounding noise does
    l1 = _fp32_study(oracle, "config4 hotspots 96^3", inputs.hotspots(96, steps=48))
    for st, d in l1.items():
        for k, v in d.items():
            assert v <= 1e-4, (st, k, v)


@pytest.mark.xfail(strict=True, reason="north_star's fp32 bar (err_L1 <= 1e-4) at config 4's own 200 steps is NOT met: "
                   "measured 2.8e-4 in E; the scheme amplifies one fp32 rounding (2^29 coarser than fp64) exactly as it "
                   "amplifies fp64 rounding (floor64 x 2^29 ~ 5e-4 at 200 steps).  DESIGN.md 4, row a7: bar not met.")
def test_config4_hotspots_fp32_200_steps_north_star_bar(oracle):
    c = inputs.hotspots(96, steps=200)
    ref, _ = parity.run_oracle(oracle, c)
    got, _ = parity.run_gpu(c, precision=32)
    rep = parity.field_report(got, ref)
    parity.record("config4 hotspots 96^3 fp32 200 steps", rep, steps=200, precision=32, grid=[96, 96, 96])
    for k, v in rep.items():
        assert v["err_L1"] <= 1e-4, (k, v)


def test_config4_hotspots_fp32_200_steps_stays_at_the_noise_scaled_level(oracle):
    # what CAN be asserted at 200 steps: the fp32 path is no worse than fp64 rounding noise scaled by 2^29
    c = inputs.hotspots(96, steps=200)
    ref, _ = parity.run_oracle(oracle, c)
    got, _ = parity.run_gpu(c, precision=32)
    errs = parity.field_errors(got, ref)
    floor = parity.noise_floor(oracle, c, ref)
    for k, (emax, el1) in errs.items():
        assert el1 <= max(1e-4, floor[k][1] * 2.0 ** 29), (k, emax, el1, floor[k])


def test_config5_slabs_fp32_study(oracle):
    # f3 at high gamma: the slab column (1x1x512 = config 5 by pin P11), fp32 transport vs the fp64 oracle
    _fp32_study(oracle, "config5 slabs 1x1x512", inputs.slabs(512, steps=100, nxy=1))


def test_config4_full_size_every_cell_24_steps(oracle):
    # the metric's own configuration: 256^3, dx = 0.1 fm, in the launch configuration bench.py times, EVERY cell compared
    # after 24 steps (four cycles of the six axis orders); the oracle runs on all host cores (~1 min on 16); fp32 too
    c = inputs.hotspots(256, steps=24)
    ref, o = parity.run_oracle(oracle, c)
    got, s = parity.run_gpu(c)
    _check_config(oracle, "config4 hotspots 256^3 (full size), 24 steps", c, got, ref, s, o, steps=24, grid=[256] * 3)
    del got
    got32, _ = parity.run_gpu(c, precision=32)
    rep = parity.field_report(got32, ref)
    parity.record("config4 hotspots 256^3 (full size) fp32 24 steps", rep, steps=24, precision=32, grid=[256] * 3)
    for k, v in rep.items():
        assert v["err_L1"] <= 1e-4, (k, v)


@pytest.mark.slow
def test_config4_full_size_every_cell_200_steps(oracle):
    # config 4 exactly as BASELINE.json states it: 256^3 x 200 steps, every cell (oracle: ~7 min on 16 cores, twice
    # for the noise floor).  Opt-in: SHASTA_SLOW=1 or -m "gpu and slow".
    # Result of the round-2 run (profiles/parity_r2.json): at the config's own size and step count the rounding-noise floor
    # of the scheme (strict vs FMA build of the ORACLE) is 8e-9 in E and the momenta, 5e-8 in e, p: north_star's 1e-10 is out
    # of reach of any two fp64 evaluations.  The GPU path sits at that floor (err_L1 within 1 % of floor_L1 in E, M, R;
    # err_max 1.2x .. 2.3x floor_max; Pi fires in exactly the same 20 583 497 cells).  Asserted here: max-norm within 4x
    # the floor's (a tail statistic), L1 within 1.25x the floor's (a bulk statistic); then the test reports the literal
    # bar as NOT met (xfail) instead of passing on the relaxed one.
    c = inputs.hotspots(256, steps=200)
    ref, o = parity.run_oracle(oracle, c)
    got, s = parity.run_gpu(c)
    rep = _check_config(oracle, "config4 hotspots 256^3 (full size), 200 steps", c, got, ref, s, o, l1=False, outright=(),
                        factor=4.0, steps=200, grid=[256] * 3)
    for k, v in rep.items():
        assert v["err_L1"] <= max(1e-12, 1.25 * v["floor_L1"]), (k, v)
    assert s.diagnostics()[0] == o.diagnostics()[0]
    if not all(v["err_max"] <= TOL64 for v in rep.values()):
        pytest.xfail("north_star's literal err_max <= 1e-10 is NOT met at 256^3 x 200 steps: the oracle's own strict-vs-FMA "
                     "noise floor is 8e-9 (E) .. 4e-7 (n) there; the GPU result sits at that floor (DESIGN.md 4)")


def test_config4_full_size_sampled(oracle):
    # 256^3 in the launch configuration bench.py times; the oracle recomputes sampled sub-boxes:
    # after s steps a cell depends on +-4 s cells per axis (one sweep per axis per step)
    steps, w = 6, 16
    halo = 4 * steps
    c = inputs.hotspots(256, steps=steps)
    got, _ = parity.run_gpu(c)
    rng = np.random.default_rng(1)
    for _ in range(3):
        lo = rng.integers(0, 256 - (w + 2 * halo), 3)
        sl = tuple(slice(l, l + w + 2 * halo) for l in lo)
        sub = dict(c)
        for k in ("e", "n", "vx", "vy", "vz"):
            sub[k] = np.ascontiguousarray(c[k][sl])
        sub["nx"] = sub["ny"] = sub["nz"] = w + 2 * halo
        ref, _ = parity.run_oracle(oracle, sub, steps=steps)
        inner = tuple(slice(halo, halo + w) for _ in range(3))
        g = {k: v[sl][inner] for k, v in got.items()}
        r = {k: v[inner] for k, v in ref.items()}
        # normalise by the global field scale, not the sub-box's
        for k in r:
            d = np.abs(g[k] - r[k]).max()
            scale = np.abs(got[k]).max() if k not in parity.GROUPS else max(np.abs(got[q]).max() for q in parity.GROUPS[k])
            assert d <= TOL64 * scale, (k, d, scale)


def test_config5_slabs_full_size(oracle):
    # 512^3; uniform in x,y => the oracle is the 1x1x512 column broadcast (pin P11)
    c1 = inputs.slabs(512, steps=100, nxy=1)
    ref, _ = parity.run_oracle(oracle, c1)
    c = inputs.slabs(512, steps=100)
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    s = Shasta(512, 512, 512, c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"])
    s.set_state(*[torch.from_numpy(c[k]).cuda() for k in ("e", "n", "vx", "vy", "vz")])
    del c
    s.step(100)
    cons = s.get_conserved()
    prim = s.get_primitives()
    for k, v in list(cons.items()) + list(prim.items()):
        r = torch.from_numpy(ref[k]).cuda()                       # (512,1,1)
        if k in parity.GROUPS:
            scale = max(np.abs(ref[q]).max() for q in parity.GROUPS[k])
        else:
            scale = np.abs(ref[k]).max()
        d = (v - r).abs().max().item()
        assert d <= TOL64 * max(scale, 1e-300), (k, d, scale)
