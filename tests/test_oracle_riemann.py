"""Pins P8/P9: the assembled 1D scheme against the exact relativistic Riemann solution (config 1)."""
import os

import numpy as np
import pytest

import exact_riemann as ex
from paper_1206_0919_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden", "riemann_plateau.txt")


def _run(oracle, ncell, e_right):
    c = inputs.shock_tube(ncell, e_right)
    o = oracle.Oracle(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"])
    o.set_state(c["e"], c["n"], c["vx"], c["vy"], c["vz"])
    o.step(c["steps"])
    t = c["steps"] * c["lam"] * c["dx"]
    x = -1.0 + (np.arange(ncell) + 0.5) * c["dx"]
    p = {k: v.ravel() for k, v in o.get_primitives().items()}
    return x / t, p, o


def test_exact_solution_matches_golden_values():
    # the closed form in tests/exact_riemann.py reproduces the printed plateau values (tests/golden)
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        eL, eR, es, vs, vsh, xit = map(float, line.split())
        got = ex.plateau(eL, eR)
        for g, w in zip(got, (es, vs, vsh, xit)):
            assert abs(g - w) < 6e-5 * abs(w) if eR < 1e-6 else abs(g - w) < 1e-7


def test_P8_shock_tube_converges_to_exact(oracle):
    errs = {}
    for n in (200, 400, 800):
        xi, p, o = _run(oracle, n, 0.01)
        e, v, nd = ex.solution(xi, 1.0, 0.01)
        errs[n] = np.abs(p["e"] - e).sum() / e.sum()
        if n == 400:
            assert errs[n] < 1e-2
            assert np.abs(p["vx"] - v).mean() < 6e-3
            assert np.abs(p["n"] - nd).sum() / nd.sum() < 1e-2
            plat = (xi >= 0.55) & (xi <= 0.8)                # right of the start-up dip that rides at xi~0.43
            es = ex.plateau(1.0, 0.01)[0]
            assert np.max(np.abs(p["e"][plat] - es)) < 0.01 * es
            assert abs(np.median(p["e"][plat]) - es) < 0.01 * es
            assert np.all(p["vy"] == 0.0) and np.all(p["vz"] == 0.0)
            assert p["vx"].max() < 0.83                       # bounded overshoot at the shock (exact 0.768)
    order = np.log(errs[200] / errs[800]) / np.log(4.0)
    assert order > 0.8, (errs, order)


def test_P8_near_vacuum_variant_fan(oracle):
    # e_R = 1e-8 ("0 plus floor"): the shell is unresolvable, compare the rarefaction fan only
    xi, p, o = _run(oracle, 400, 1e-8)
    e, v, nd = ex.solution(xi, 1.0, 1e-8)
    m = xi < 0.8
    assert np.abs(p["e"][m] - e[m]).sum() / e[m].sum() < 1e-2
    assert np.all(np.isfinite(p["e"])) and np.all(p["e"] >= 0.0)
    assert np.all(np.abs(p["vx"]) < 1.0)
