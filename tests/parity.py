"""Shared helpers of the GPU parity tests: error metrics of DESIGN.md 4 (reading G18) and drivers
that run the same seeded config through the oracle (CPU) and through the C ABI (GPU)."""
import numpy as np

CONS = ("E", "Mx", "My", "Mz", "R")
PRIM = ("e", "p", "n", "vx", "vy", "vz")
GROUPS = {"Mx": ("Mx", "My", "Mz"), "My": ("Mx", "My", "Mz"), "Mz": ("Mx", "My", "Mz"),
          "vx": ("vx", "vy", "vz"), "vy": ("vx", "vy", "vz"), "vz": ("vx", "vy", "vz")}


EPS = 2.0 ** -52


V2_NEAR_LIGHT = 1e-6


def n_allowance(ref):
    """Conditioning of n = R sqrt(1-v^2): one ulp of v moves n by n v dv/(1-v^2).  Where the
    causality projection holds v at 1-1e-12 this is ~1e-4 of the cell's n, on BOTH sides (the oracle's own n
    carries it).  |dn| up to 32 eps n/(1-v^2) is therefore not an error of either implementation.  Applied ONLY in
    cells with 1 - v^2 < 1e-6 (gamma > 1000): everywhere else n is compared raw."""
    v2 = sum(np.asarray(ref[c], dtype=np.float64) ** 2 for c in ("vx", "vy", "vz"))
    a = 32.0 * EPS * np.abs(ref["n"]) / np.maximum(1.0 - v2, EPS)
    return np.where(1.0 - v2 < V2_NEAR_LIGHT, a, 0.0)


def _scales(ref, k):
    if k in GROUPS:
        mag = np.sqrt(sum(np.asarray(ref[c], dtype=np.float64) ** 2 for c in GROUPS[k]))
    else:
        mag = np.abs(np.asarray(ref[k], dtype=np.float64))
    return mag.max(), mag.sum()


def field_errors(got, ref):
    """per field: (err_max, err_L1) = (max|X-X*| / max|X*|, sum|X-X*| / sum|X*|); the three momentum
    (velocity) components share one denominator built from |M*| (|v*|).  For n the conditioning allowance
    n_allowance() is subtracted from |X-X*| first (near-light cells only)."""
    out = {}
    for k in ref:
        g = np.asarray(got[k], dtype=np.float64)
        r = np.asarray(ref[k], dtype=np.float64)
        dmax, dsum = _scales(ref, k)
        d = np.abs(g - r)
        if k == "n" and all(c in ref for c in ("vx", "vy", "vz")):
            d = np.maximum(d - n_allowance(ref), 0.0)
        out[k] = (d.max() / dmax if dmax > 0 else d.max(), d.sum() / dsum if dsum > 0 else d.sum())
    return out


def field_report(got, ref, floor=None, bar=None):
    """What profiles/parity_r2.json records per field: achieved err_max / err_L1 (with the n allowance), the noise
    floor and the bar applied (when given), and for n the RAW numbers without allowance plus the number of cells in
    which the allowance exceeds 1e-12 max|n|."""
    errs = field_errors(got, ref)
    rep = {}
    for k, (emax, el1) in errs.items():
        rep[k] = {"err_max": float(emax), "err_L1": float(el1)}
        if floor is not None and k in floor:
            rep[k]["floor_max"], rep[k]["floor_L1"] = float(floor[k][0]), float(floor[k][1])
        if bar is not None:
            rep[k]["bar_max"] = float(bar[k] if isinstance(bar, dict) else bar)
    if "n" in ref and all(c in ref for c in ("vx", "vy", "vz")):
        d = np.abs(np.asarray(got["n"], dtype=np.float64) - np.asarray(ref["n"], dtype=np.float64))
        dmax, dsum = _scales(ref, "n")
        al = n_allowance(ref)
        rep["n"].update({"err_max_raw": float(d.max() / dmax), "err_L1_raw": float(d.sum() / dsum),
                         "allowance_cells": int((al > 1e-12 * dmax).sum()), "cells": int(d.size)})
    return rep


_RECORD = {}


def record(name, rep, **meta):
    """Collected by tests/conftest.py and written to gpurun_out/parity_r2.json at the end of the session."""
    _RECORD[name] = dict(meta, fields=rep)


def run_oracle(oracle, c, steps=None, table=None, variant="strict", predictor=0, diff=1.0, eos_table=None,
               antidiffusion=0):
    o = oracle.Oracle(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"],
                      variant=variant, predictor=predictor, diff=diff, eos_table=eos_table, antidiffusion=antidiffusion)
    if table is not None:
        o.set_sweep_table(table)
    o.set_state(c["e"], c["n"], c["vx"], c["vy"], c["vz"])
    o.step(c["steps"] if steps is None else steps)
    res = dict(o.get_conserved())
    res.update(o.get_primitives())
    return res, o


def run_gpu(c, steps=None, table=None, precision=64, segment=0, host_io=False, no_tma=0, predictor=0, diff=1.0,
            cell_path=0, eos_table=None, antidiffusion=0, batch=1, graph=None):
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"],
               precision=precision, segment=segment, no_tma=no_tma, predictor=predictor, diff=diff, cell_path=cell_path,
               eos_table=eos_table, antidiffusion=antidiffusion, batch=batch, graph=graph)
    if table is not None:
        s.set_sweep_table(table)
    if host_io:
        s.set_state_host(*[torch.from_numpy(c[k]) for k in ("e", "n", "vx", "vy", "vz")])
    else:
        s.set_state(*[torch.from_numpy(c[k]).cuda() for k in ("e", "n", "vx", "vy", "vz")])
    s.step(c["steps"] if steps is None else steps)
    res = {k: v.cpu().numpy() for k, v in s.get_conserved().items()}
    if host_io:
        outs = [torch.empty(s.shape, dtype=torch.float64) for _ in range(6)]
        s.get_primitives_host(outs)
        torch.cuda.synchronize()
        res.update(dict(zip(PRIM, [o.numpy() for o in outs])))
    else:
        res.update({k: v.cpu().numpy() for k, v in s.get_primitives().items()})
    return res, s


def assert_parity(got, ref, tol_max, tol_l1=None, fields=None, label=""):
    errs = field_errors({k: got[k] for k in (fields or ref)}, {k: ref[k] for k in (fields or ref)})
    bad = {k: v for k, v in errs.items() if not (v[0] <= tol_max) or (tol_l1 is not None and not (v[1] <= tol_l1))}
    assert not bad, f"{label} parity failed (err_max, err_L1): {bad}; all: {errs}"
    return errs


def noise_floor(oracle, c, ref, steps=None):
    """Rounding-noise floor of the step map for this config: the oracle source compiled with FMA contraction
    (an equally valid fp64 evaluation of the same formulas) against the strict oracle `ref`.  Returns the
    field_errors dict.  DESIGN.md 4."""
    alt, _ = run_oracle(oracle, c, steps=steps, variant="fma")
    return field_errors(alt, ref)


def assert_parity_noise(got, ref, floor, tol=1e-10, factor=4.0, label=""):
    """fp64 bar: err_max <= max(tol, factor * noise floor of that field)."""
    errs = field_errors(got, ref)
    bad = {k: (v[0], floor[k][0]) for k, v in errs.items() if not v[0] <= max(tol, factor * floor[k][0])}
    assert not bad, f"{label} parity failed (err_max, noise floor): {bad}; all: {errs}; floor: {floor}"
    return errs
