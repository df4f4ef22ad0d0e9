"""Pins P1-P5 and G12: algebraic identities of eqs. (15)-(22) that a dropped
term, wrong sign or wrong index in oracle/shasta_oracle.c would break.  CPU only."""
import numpy as np
import pytest


def test_P1_qplus_qminus_partition(oracle):
    # eq. (15), reading G1: Q+_j + Q-_{j+1} = 1 for ANY velocity field
    rng = np.random.default_rng(1)
    eps = rng.uniform(-0.49, 0.49, 1000)
    for j in range(999):
        qp, qm = oracle.qplus(eps[j], eps[j + 1]), oracle.qminus(eps[j + 1], eps[j])
        den = 1.0 + (eps[j + 1] - eps[j])                    # common denominator, rounded once
        assert abs(qp + qm - 1.0) < 4e-16 * (1.0 + 1.0 / den)
    # v = 0: both are exactly 1/2
    assert oracle.qplus(0.0, 0.0) == 0.5 and oracle.qminus(0.0, 0.0) == 0.5


def test_P2_flux_form_and_conservation(oracle):
    # eq. (17) equals U_j - F_{j+1/2} + F_{j-1/2} with F = (1/2 - q) U_j - 1/2 q^2 Delta_j, q = Q+_j
    rng = np.random.default_rng(2)
    n = 64
    U = rng.normal(size=n) + 3.0
    eps = rng.uniform(-0.45, 0.45, n)
    f = rng.normal(size=n)
    lam = 0.4
    # periodic extension by 1
    Ue = np.concatenate([U[-1:], U, U[:1]]); ee = np.concatenate([eps[-1:], eps, eps[:1]])
    fe = np.concatenate([f[-1:], f, f[:1]])
    uh = oracle.transport(Ue, ee, fe, lam, 1, n + 1)[1:n + 1]
    q = (0.5 - ee[:-1]) / (1.0 + (ee[1:] - ee[:-1]))         # interface j+1/2, j = -1..n-1
    F = (0.5 - q) * Ue[:-1] - 0.5 * q * q * (Ue[1:] - Ue[:-1])
    ref = Ue[1:n + 1] - F[1:] + F[:-1] - 0.5 * lam * (fe[2:] - fe[:-2])
    assert np.max(np.abs(uh - ref)) < 1e-14
    import math
    assert abs(math.fsum(uh) - math.fsum(U)) < 1e-13 * n


def test_P3_uniform_velocity_is_lax_wendroff_plus_eighth(oracle):
    rng = np.random.default_rng(3)
    n = 50
    U = rng.normal(size=n)
    for e in (0.0, 0.2, -0.37):
        eps = np.full(n, e)
        uh = oracle.transport(U, eps, None, 0.4, 1, n - 1)[1:-1]
        ref = U[1:-1] - 0.5 * e * (U[2:] - U[:-2]) + (0.125 + 0.5 * e * e) * (U[2:] - 2 * U[1:-1] + U[:-2])
        assert np.max(np.abs(uh - ref)) < 1e-15 * 10


def test_P4_phoenical_cancels_diffusion_at_rest(oracle):
    # v = 0, no source: Uhat_j = U_j + 1/8 (U_{j+1} - 2U_j + U_{j-1}); with a monotone profile the limiter
    # is inactive and A = A^ph = 1/8 Delta_j exactly => U^{n+1} = U^n  (the inner 1/8 of eq. (19))
    n = 40
    x = np.arange(n, dtype=np.float64)
    U = np.tanh((x - 20) / 6.0) + 2.0                       # smooth monotone: limiter never clips
    eps = np.zeros(n)
    uh = oracle.transport(U, eps, None, 0.4, 1, n - 1)
    ref = U.copy(); ref[1:-1] += 0.125 * (U[2:] - 2 * U[1:-1] + U[:-2])
    assert np.max(np.abs(uh[1:-1] - ref[1:-1])) < 1e-15
    un = oracle.antidiffuse(U, uh, 4, n - 4)
    assert np.max(np.abs(un[4:n - 4] - U[4:n - 4])) < 5e-16


def test_P5_no_new_extrema_square_wave(oracle):
    # eqs. (21)-(22), Boris-Book: prescribed constant velocity, source free
    n = 200
    U0 = np.where((np.arange(n) > 60) & (np.arange(n) < 120), 2.0, 0.5)
    vel = np.full(n, 0.5)                                    # eps = 0.4*0.5 = 0.2
    U = U0.copy()
    for _ in range(100):
        U, uh = oracle.advect_pencil(U, vel, 0.4, 1, 1)      # periodic
        lo = np.minimum(np.minimum(np.roll(uh, 1), uh), np.roll(uh, -1))
        hi = np.maximum(np.maximum(np.roll(uh, 1), uh), np.roll(uh, -1))
        assert np.all(U >= lo - 1e-14) and np.all(U <= hi + 1e-14)
    assert U.min() >= 0.5 - 1e-12 and U.max() <= 2.0 + 1e-12
    import math
    assert abs(math.fsum(U) - math.fsum(U0)) < 1e-11
    # the wave moved by eps*100 = 20 cells: centre of mass of (U - 0.5)
    com0 = np.sum((U0 - 0.5) * np.arange(n)) / np.sum(U0 - 0.5)
    com1 = np.sum((U - 0.5) * np.arange(n)) / np.sum(U - 0.5)
    assert abs((com1 - com0) - 20.0) < 0.05
    # and it stays sharp (FCT): the 10-90% rise takes only a few cells
    rise = np.sum((U > 0.5 + 0.15) & (U < 2.0 - 0.15))
    assert rise <= 10


def test_P5_direction_of_transport(oracle):
    # a wrong sign in eq. (15) moves the pulse the wrong way
    n = 100
    U0 = np.exp(-0.5 * ((np.arange(n) - 50) / 4.0) ** 2)
    for v, shift in ((0.75, 12.0), (-0.75, -12.0)):
        U, _ = oracle.advect_pencil(U0, np.full(n, v), 0.4, 1, 40)
        com = np.sum(U * np.arange(n)) / np.sum(U)
        assert abs(com - 50 - shift) < 0.05


def test_G12_limiter_zero_and_sign(oracle):
    # local extremum of Uhat: the antidiffusive flux towards it is cut to zero (eq. (21))
    n = 16
    U = np.zeros(n); U[8] = 1.0
    uh = oracle.transport(U, np.zeros(n), None, 0.4, 1, n - 1)
    un = oracle.antidiffuse(U, uh, 4, n - 4)
    assert un[8] <= uh[8] + 1e-16 or un[8] <= 1.0
    assert un.min() >= -1e-16                                 # no undershoot next to the peak
    assert abs(un[4:n - 4].sum() - U[4:n - 4].sum()) < 1e-15
