"""Pins P14, P15: the oracle's half-step predictor (steps 3-5 of oracle_sweep_pencil) and its outflow
ghost rule -- the two parts the pins P1-P13 leave free (a predictor source scaled by lambda
instead of lambda/2, no half step at all, corrector sources taken at time n, or reflected ghosts all passed).

P14  Linear acoustic wave (textbook, not from the paper): for p = e/3 the sound speed is c_s = 1/sqrt(3) and a
     right-going simple wave of small amplitude has dv = c_s de/(e+p).  A scheme whose velocity and source terms
     are centred at n+1/2 ("staggered grid in time direction"; "implemented based on a
     half-step method") transports it with second-order accuracy; any error in the time centring (no half step,
     wrong lambda factor in the predictor, sources at time n) degrades the observed order to ~1 or worse.
     The limiter does not act on a resolved cosine away from its extrema enough to matter at A = 1e-6.
P15  Ghost extension, reading G11 (PAPER.md:161, 276-277 halo): sweeping a pencil with OUTFLOW must equal, bitwise,
     the interior of the same sweep on the pencil extended BY HAND with 4 copies of each edge cell, whatever
     boundary rule the extended pencil is swept with (the interior's dependency radius is 4).
"""
import numpy as np
import pytest

CS = 1.0 / np.sqrt(3.0)


def _acoustic_error(oracle, N, A=1e-6, lam=0.4):
    dx = 1.0 / N
    x = (np.arange(N) + 0.5) * dx
    de = A * np.cos(2 * np.pi * x)
    e = 1.0 + de
    v = CS * de / (4.0 / 3.0)                                 # dv = c_s de / (e + p), e + p = 4/3
    sh = (1, 1, N)
    o = oracle.Oracle(N, 1, 1, dx, lam, 4.0 / 3.0, boundary=oracle.PERIODIC)
    z = np.zeros(sh)
    o.set_state(e.reshape(sh), (e ** 0.75).reshape(sh), v.reshape(sh), z, z)
    steps = 5 * N // 4                                        # t = steps * lam * dx = 0.5
    o.step(steps)
    t = steps * lam * dx
    got = o.get_primitives()["e"].ravel()
    exact = 1.0 + A * np.cos(2 * np.pi * (x - CS * t))
    return np.abs(got - exact).mean() / A


def test_P14_acoustic_wave_second_order(oracle):
    Ns = (48, 96, 192, 384)
    errs = [_acoustic_error(oracle, N) for N in Ns]
    orders = [np.log2(errs[i] / errs[i + 1]) for i in range(len(Ns) - 1)]
    assert errs[0] < 1e-2, errs                               # the wave arrives where c_s says it should
    assert all(o >= 1.8 for o in orders), (errs, orders)


def test_P14_left_going_wave(oracle):
    # mirror image: dv = -c_s de/(e+p) travels to the left at c_s (a sign error in the source term or in Q+-
    # would not be mirror symmetric)
    N, A, lam = 96, 1e-6, 0.4
    dx = 1.0 / N
    x = (np.arange(N) + 0.5) * dx
    de = A * np.cos(2 * np.pi * x)
    sh = (1, 1, N)
    z = np.zeros(sh)
    o = oracle.Oracle(N, 1, 1, dx, lam, 4.0 / 3.0, boundary=oracle.PERIODIC)
    o.set_state((1 + de).reshape(sh), ((1 + de) ** 0.75).reshape(sh), (-CS * de * 0.75).reshape(sh), z, z)
    o.step(120)
    got = o.get_primitives()["e"].ravel()
    exact = 1.0 + A * np.cos(2 * np.pi * (x + CS * 120 * lam * dx))
    assert np.abs(got - exact).mean() / A < 3e-3


def _rough_pencil(seed, N=24):
    rng = np.random.default_rng(seed)
    e = np.exp(rng.normal(size=N))
    e[N // 3: N // 2] *= 50.0
    v = np.clip(0.5 * rng.normal(size=(3, N)), -0.55, 0.55)
    n = e ** 0.75
    return e, n, v


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_P15_outflow_equals_hand_extended_pencil(oracle, axis, seed):
    e, n, v = _rough_pencil(seed)
    N = e.size
    U = np.array([oracle.prim2cons(e[j], n[j], v[0, j], v[1, j], v[2, j], 4.0 / 3.0) for j in range(N)]).T.copy()
    assert U[1 + axis, 0] != U[1 + axis, 1] and U[0, -1] != U[0, -2]      # edges are NOT uniform
    swept, _ = oracle.sweep_pencil(U, axis, 0.4, 4.0 / 3.0, bc=oracle.OUTFLOW)
    ext = np.concatenate([np.repeat(U[:, :1], 4, axis=1), U, np.repeat(U[:, -1:], 4, axis=1)], axis=1)
    for bc in (oracle.OUTFLOW, oracle.PERIODIC):
        swept_ext, _ = oracle.sweep_pencil(ext, axis, 0.4, 4.0 / 3.0, bc=bc)
        assert np.array_equal(swept_ext[:, 4:4 + N], swept), bc
    # and the edge cells really changed (the test is not vacuous)
    assert not np.array_equal(swept[:, :2], U[:, :2])


def test_P15_periodic_equals_hand_wrapped_pencil(oracle):
    e, n, v = _rough_pencil(7)
    N = e.size
    U = np.array([oracle.prim2cons(e[j], n[j], v[0, j], v[1, j], v[2, j], 4.0 / 3.0) for j in range(N)]).T.copy()
    swept, _ = oracle.sweep_pencil(U, 0, 0.4, 4.0 / 3.0, bc=oracle.PERIODIC)
    ext = np.concatenate([U[:, -4:], U, U[:, :4]], axis=1)
    swept_ext, _ = oracle.sweep_pencil(ext, 0, 0.4, 4.0 / 3.0, bc=oracle.OUTFLOW)
    assert np.array_equal(swept_ext[:, 4:4 + N], swept)
