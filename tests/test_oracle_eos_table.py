"""Pins of the oracle's tabled equation of state (row f1; "a fixed point root finding algorithm to
allow for an easy implementation of a tabled equation of state").  The paper gives no table and no interpolation rule;
reading T1: P at nodes (i de, j dn), bilinear between nodes, linear continuation outside, floored at 0.

What the mathematics fixes, independent of the oracle:
  * bilinear interpolation reproduces a function that is linear in e and in n EXACTLY, on any grid: a table sampled from the
    ideal gas p = (Gamma-1)(e - m n) must give the analytic EOS back (cons2prim, prim2cons and whole runs);
  * scipy's RegularGridInterpolator(method="linear", fill_value=None) is the same rule written by someone else;
  * the velocity is the root of g(v) = v (E + P(E - M v, R sqrt(1 - v^2))) - M: brute-force bisection with the scipy rule.
"""
import numpy as np
import pytest

from paper_1206_0919_b200 import inputs

NE, NN, EMAX, NMAX = 41, 17, 8.0, 3.0          # ne != nn: a transposed table cannot pass


def _grid():
    return np.linspace(0.0, EMAX, NE), np.linspace(0.0, NMAX, NN)


def soft_eos(e, n):
    """synthetic, smooth, causal (dp/de <= 0.4) and NOT linear: a softened crossover plus a density term"""
    return e / 3.0 * (1.0 - 0.25 * np.exp(-0.5 * (e - 2.0) ** 2)) + 0.05 * n * n / (1.0 + n)


def _table(fn):
    eg, ng = _grid()
    return fn(eg[None, :], ng[:, None]) + 0.0 * eg[None, :] * ng[:, None]        # shape (NN, NE)


def test_T1_linear_table_is_the_ideal_gas(oracle):
    G, m = 5.0 / 3.0, 1.0
    tab = oracle.make_table(_table(lambda e, n: (G - 1.0) * (e - m * n)), EMAX, NMAX)
    assert oracle.eos_table_P(tab, 0.5, 2.0) == 0.0 and oracle.eos_table_P(tab, 0.0, 0.1) == 0.0      # floored at 0 (e < m n)
    rng = np.random.default_rng(1)
    for _ in range(2000):
        e = 10.0 ** rng.uniform(-3, 1.2); n = e * rng.uniform(0.0, 0.95); v = rng.uniform(-0.99, 0.99, 3) / np.sqrt(3)
        assert abs(oracle.eos_table_P(tab, e, n) - max((G - 1) * (e - m * n), 0.0)) <= 4e-15 * (e + n)
        c_t = oracle.prim2cons_table(e, n, *v, tab)
        c_a = oracle.prim2cons(e, n, *v, G, m)
        assert np.max(np.abs(c_t - c_a)) <= 1e-13 * abs(c_a[0])
        o_t, _, _ = oracle.cons2prim_table(*c_a, tab)
        o_a, _, _ = oracle.cons2prim(*c_a, G, m)
        assert np.max(np.abs(o_t - o_a)) <= 1e-12 * max(1.0, abs(o_a[0]))


def test_T2_bilinear_rule_against_scipy(oracle):
    from scipy.interpolate import RegularGridInterpolator
    p2d = _table(soft_eos)
    tab = oracle.make_table(p2d, EMAX, NMAX)
    eg, ng = _grid()
    ref = RegularGridInterpolator((ng, eg), p2d, method="linear", bounds_error=False, fill_value=None)
    rng = np.random.default_rng(2)
    e = np.concatenate([rng.uniform(0, EMAX, 3000), rng.uniform(EMAX, 1.5 * EMAX, 300), eg[:10], [0.0, EMAX]])
    n = np.concatenate([rng.uniform(0, NMAX, 3000), rng.uniform(NMAX, 1.3 * NMAX, 300), ng[:10], [0.0, NMAX]])
    want = np.maximum(ref(np.stack([n, e], axis=1)), 0.0)
    got = np.array([oracle.eos_table_P(tab, a, b) for a, b in zip(e, n)])
    assert np.max(np.abs(got - want)) <= 1e-12 * np.max(np.abs(want))      # rounding only (extrapolation weights > 1)
    # the nodes themselves are returned exactly
    for j in (0, 5, NN - 1):
        for i in (0, 7, NE - 1):
            assert oracle.eos_table_P(tab, eg[i], ng[j]) == pytest.approx(max(p2d[j, i], 0.0), abs=1e-15)


def test_T3_velocity_root_by_bisection(oracle):
    from scipy.interpolate import RegularGridInterpolator
    p2d = _table(soft_eos)
    tab = oracle.make_table(p2d, EMAX, NMAX)
    eg, ng = _grid()
    ref = RegularGridInterpolator((ng, eg), p2d, method="linear", bounds_error=False, fill_value=None)
    P = lambda e, n: max(float(ref([[n, e]])[0]), 0.0)
    rng = np.random.default_rng(3)
    for _ in range(300):
        e = rng.uniform(0.05, 6.0); n = rng.uniform(0.0, 2.5); v0 = rng.uniform(0.0, 0.97)
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        c = oracle.prim2cons_table(e, n, *(v0 * d), tab)
        E, R = c[0], c[4]
        M = np.linalg.norm(c[1:4])
        g = lambda v: v * (E + P(E - M * v, R * np.sqrt(1.0 - v * v))) - M
        lo, hi = 0.0, min(M / E, 1.0 - 1e-12)
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if g(mid) < 0.0 else (lo, mid)
        out, it, _ = oracle.cons2prim_table(*c, tab)
        assert it < 200
        assert abs(out[6] - 0.5 * (lo + hi)) <= 5e-13
        # and the round trip gives the primitives back
        assert abs(out[6] - v0) <= 1e-11 and abs(out[0] - e) <= 1e-11 * (1.0 + e) / (1.0 - v0 * v0)
        assert abs(out[1] - P(out[0], out[2])) <= 1e-13 * (1.0 + out[1])


@pytest.mark.parametrize("bc", [inputs.OUTFLOW, inputs.PERIODIC])
def test_T4_whole_run_with_a_linear_table_equals_the_analytic_run(oracle, bc):
    # plumbing of the table through set_state, every cons2prim of the sweep and get_primitives: 3 steps of a rough 3-D
    # state with the m = 1 ideal gas as a table against the analytic m = 1 run (differences: rounding of the lookup only)
    G, m = 5.0 / 3.0, 1.0
    c = inputs.random_state(14, 11, 9, seed=12, kind="rough", gamma=G, mass=m, boundary=bc)
    emax = 4.0 * max(c["e"].max(), 1.0) * 50.0
    nmax = 4.0 * max(c["n"].max(), 1.0) * 10.0
    eg, ng = np.linspace(0, emax, 33), np.linspace(0, nmax, 21)
    p2d = (G - 1.0) * (eg[None, :] - m * ng[:, None])
    a = oracle.Oracle(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], G, bc, m)
    t = oracle.Oracle(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], G, bc, 0.0, eos_table=(p2d, emax, nmax))
    for o in (a, t):
        o.set_state(c["e"], c["n"], c["vx"], c["vy"], c["vz"])
        o.step(3)
    ra, rt = dict(a.get_conserved()), dict(t.get_conserved())
    ra.update(a.get_primitives()); rt.update(t.get_primitives())
    for k in ra:
        assert np.max(np.abs(ra[k] - rt[k])) <= 1e-10 * max(np.max(np.abs(ra[k])), 1e-30), k
