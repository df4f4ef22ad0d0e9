"""Pins of the oracle's scheme variants, each before any kernel work:

diff      PAPER.md:159, 279 (`const float diff = 1.0f`, "fine controlled application of numerical viscosity"): factor on
          the antidiffusive flux A^ph.  Pin: P4 generalised -- at rest (v = 0, uniform pressure) the limiter-free
          update is U^{n+1} - U^n = (1 - diff) * 1/8 * second difference of U, exactly (eqs. (17)-(22) with Q+- = 1/2).
n/af      PAPER.md:201-205 (Fig. 7 "n/af": no anti-flux) = diff 0.  Pin: equals P3's closed form for uniform eps
          (Lax-Wendroff + 1/8 diffusion, the textbook SHASTA transport stage).
explicit  PAPER.md:123, footnote 1 ("Different anti-diffusion terms are possible"): the explicit term of the original SHASTA,
          A^ex_j = 1/8 Dhat_j (Boris & Book).  Pin (textbook property): at rest, limiter inactive, the explicit scheme leaves
          the residual damping U^{n+1} - U^n = -1/64 delta^4 U, where the phoenical one gives exactly 0 (P4).
R2        PAPER.md:302-313 (Listing 2 runs the ordinary prop kernels after half_cfl): the half step is the whole
          kernel with lambda/2, eq. (17) AND eqs. (18)-(22).  Pins: P14 (acoustic wave) must still give order >= 1.8;
          the Riemann problem converges to the exact solution (P8 gates); R2 differs from R1 (the option is live).
"""
import numpy as np
import pytest

import exact_riemann as ex
from paper_1206_0919_b200 import inputs

CS = 1.0 / np.sqrt(3.0)
GAM = 4.0 / 3.0


def _rest_pencil(oracle, N=40, seed=0):
    """e = 1 (uniform pressure), v = 0, n = monotone smooth ramp: only R moves, and only by diffusion"""
    x = np.arange(N, dtype=np.float64)
    n = 1.0 + 0.02 * x + 0.0004 * x * x                      # monotone, curvature != 0
    U = np.array([oracle.prim2cons(1.0, n[j], 0.0, 0.0, 0.0, GAM) for j in range(N)]).T.copy()
    return U


@pytest.mark.parametrize("diff", [0.0, 0.25, 0.5, 1.0])
@pytest.mark.parametrize("predictor", [0, 1])
def test_diff_at_rest_is_scaled_eighth_diffusion(oracle, diff, predictor):
    U = _rest_pencil(oracle)
    V, _ = oracle.sweep_pencil(U, 0, 0.4, GAM, bc=oracle.OUTFLOW, diff=diff, predictor=predictor)
    R0, R1 = U[4], V[4]
    d2 = np.zeros_like(R0)
    d2[1:-1] = (R0[2:] - R0[1:-1]) - (R0[1:-1] - R0[:-2])
    inner = slice(4, -4)                                      # away from the ghost copies, where the limiter clips
    want = (1.0 - diff) * 0.125 * d2
    assert np.max(np.abs((R1 - R0)[inner] - want[inner])) <= 4e-16 * np.abs(R0).max()
    # E and M untouched at rest
    assert np.array_equal(V[0], U[0]) and np.all(V[1:4] == 0.0)
    if diff != 1.0:
        assert np.max(np.abs((R1 - R0)[inner])) > 1e-5       # not vacuous


def test_noaf_equals_diff_zero_and_P3_closed_form(oracle):
    # n/af: the antidiffusion stage with diff = 0 leaves U-hat; with uniform eps that is Lax-Wendroff + 1/8 diffusion
    rng = np.random.default_rng(2)
    N = 32
    U = np.exp(rng.normal(size=N))
    vel = np.full(N, 0.37)
    lam = 0.4
    eps = lam * 0.37
    got, uh = oracle.advect_pencil(U, vel, lam, oracle.PERIODIC, 1)
    Up, Um = np.roll(U, -1), np.roll(U, 1)
    closed = U - 0.5 * eps * (Up - Um) + (0.125 + 0.5 * eps * eps) * (Up - 2 * U + Um)
    assert np.max(np.abs(uh - closed)) <= 4e-16 * np.abs(U).max()
    # the oracle's antidiffusion routine with diff = 0 returns U-hat bitwise
    ext = np.concatenate([U[-4:], U, U[:4]])
    uhe = np.concatenate([uh[-4:], uh, uh[:4]])
    out = oracle.antidiffuse(ext, uhe, 4, 4 + N, diff=0.0)
    assert np.array_equal(out[4:4 + N], uh)


def _acoustic_error(oracle, N, predictor, diff=1.0, A=1e-6, lam=0.4):
    dx = 1.0 / N
    x = (np.arange(N) + 0.5) * dx
    de = A * np.cos(2 * np.pi * x)
    e = 1.0 + de
    v = CS * de / (4.0 / 3.0)
    sh = (1, 1, N)
    o = oracle.Oracle(N, 1, 1, dx, lam, GAM, boundary=oracle.PERIODIC, predictor=predictor, diff=diff)
    z = np.zeros(sh)
    o.set_state(e.reshape(sh), (e ** 0.75).reshape(sh), v.reshape(sh), z, z)
    steps = 5 * N // 4
    o.step(steps)
    got = o.get_primitives()["e"].ravel()
    exact = 1.0 + A * np.cos(2 * np.pi * (x - CS * steps * lam * dx))
    return np.abs(got - exact).mean() / A


def test_R2_acoustic_wave_second_order(oracle):
    Ns = (48, 96, 192, 384)
    errs = [_acoustic_error(oracle, N, predictor=1) for N in Ns]
    orders = [np.log2(errs[i] / errs[i + 1]) for i in range(len(Ns) - 1)]
    assert errs[0] < 1e-2 and all(o >= 1.8 for o in orders), (errs, orders)


def _tube(oracle, ncell, predictor, diff=1.0):
    c = inputs.shock_tube(ncell, 0.01)
    o = oracle.Oracle(c["nx"], 1, 1, c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"],
                      predictor=predictor, diff=diff)
    o.set_state(c["e"], c["n"], c["vx"], c["vy"], c["vz"])
    o.step(c["steps"])
    t = c["steps"] * c["lam"] * c["dx"]
    xi = (-1.0 + (np.arange(ncell) + 0.5) * c["dx"]) / t
    p = {k: v.ravel() for k, v in o.get_primitives().items()}
    e, v, nd = ex.solution(xi, 1.0, 0.01)
    return np.abs(p["e"] - e).sum() / e.sum(), p


def test_R2_riemann_converges_and_differs_from_R1(oracle):
    l1 = {n: _tube(oracle, n, 1)[0] for n in (200, 400, 800)}
    assert l1[400] < 1e-2
    assert np.log(l1[200] / l1[800]) / np.log(4.0) > 0.8, l1
    r1, p1 = _tube(oracle, 400, 0)
    r2, p2 = _tube(oracle, 400, 1)
    assert not np.array_equal(p1["e"], p2["e"])
    assert abs(r1 - r2) < 3e-3                                # both first order at the shock; neither is "wrong" (G4)


def test_diff_below_one_adds_viscosity_monotonically(oracle):
    # smaller diff = more residual diffusion: the shock-tube overshoot of v shrinks and the L1 error grows
    over, l1 = [], []
    for diff in (1.0, 0.75, 0.5, 0.0):
        err, p = _tube(oracle, 400, 0, diff)
        over.append(p["vx"].max()); l1.append(err)
    assert over[0] >= over[1] >= over[2] >= over[3]
    assert l1[3] > l1[0]


def test_explicit_antidiffusion_leaves_the_fourth_difference_at_rest(oracle):
    # v = 0, uniform pressure: U^ = U + 1/8 d2 U; explicit antidiffusion removes 1/8 d2 U^  ->  U^{n+1} = U - 1/64 d4 U
    N = 48
    x = np.arange(N, dtype=np.float64)
    n = 1.0 + 0.02 * x + 0.0004 * x * x + 2e-7 * x ** 4             # monotone and smooth: the limiter does not bind
    U = np.array([oracle.prim2cons(1.0, n[j], 0.0, 0.0, 0.0, GAM) for j in range(N)]).T.copy()
    V, _ = oracle.sweep_pencil(U, 0, 0.4, GAM, bc=oracle.OUTFLOW, antidiffusion=oracle.EXPLICIT)
    W, _ = oracle.sweep_pencil(U, 0, 0.4, GAM, bc=oracle.OUTFLOW)
    R0 = U[4]
    d4 = np.zeros_like(R0)
    d4[2:-2] = R0[4:] - 4 * R0[3:-1] + 6 * R0[2:-2] - 4 * R0[1:-3] + R0[:-4]
    inner = slice(6, -6)
    assert np.max(np.abs(d4[inner])) > 1e-6                          # the pin has something to see
    assert np.max(np.abs((V[4] - R0)[inner] + d4[inner] / 64.0)) <= 1e-15 * np.abs(R0).max()
    assert np.max(np.abs((W[4] - R0)[inner])) <= 4e-16 * np.abs(R0).max()        # phoenical: nothing left (P4)
    # the building block alone, against the formula retyped: A = 1/8 (U^_{j+1} - U^_j) where the limiter is inactive
    Uh = R0 + 0.0
    Uh[1:-1] = R0[1:-1] + 0.125 * ((R0[2:] - R0[1:-1]) - (R0[1:-1] - R0[:-2]))
    out = oracle.antidiffuse(R0, Uh, 4, N - 4, kind=oracle.EXPLICIT)
    want = Uh[4:N - 4] - 0.125 * ((Uh[5:N - 3] - Uh[4:N - 4]) - (Uh[4:N - 4] - Uh[3:N - 5]))
    assert np.max(np.abs(out[4:N - 4] - want)) <= 4e-16 * np.abs(R0).max()


def test_explicit_antidiffusion_keeps_the_limiter_properties(oracle):
    # eqs. (20)-(22) do not care which raw antidiffusive flux they limit: with A = 1/8 D^ the update still creates no new
    # extrema of U^ (Boris-Book) and stays in flux form (telescoping sum); repeated on a square wave at rest
    n = 120
    U = np.where((np.arange(n) > 40) & (np.arange(n) < 80), 2.0, 0.5).astype(np.float64)
    total0 = float(np.sum(U))
    for _ in range(30):
        uh = U.copy()
        uh[1:-1] = U[1:-1] + 0.125 * ((U[2:] - U[1:-1]) - (U[1:-1] - U[:-2]))         # transport at rest = pure diffusion (P4)
        un = oracle.antidiffuse(U, uh, 4, n - 4, kind=oracle.EXPLICIT)
        lo = np.minimum(np.minimum(uh[3:n - 5], uh[4:n - 4]), uh[5:n - 3])
        hi = np.maximum(np.maximum(uh[3:n - 5], uh[4:n - 4]), uh[5:n - 3])
        assert np.all(un[4:n - 4] >= lo - 1e-14) and np.all(un[4:n - 4] <= hi + 1e-14)
        U = U.copy()
        U[4:n - 4] = un[4:n - 4]
    assert abs(float(np.sum(U)) - total0) < 1e-11                                      # flat ends: no flux through them
    assert U.min() >= 0.5 - 1e-12 and U.max() <= 2.0 + 1e-12
    # the explicit term steepens less than the phoenical one would undo: the wave is smeared over a few cells, not 30 steps' worth
    assert np.sum((U > 0.65) & (U < 1.85)) <= 12
