"""Shared helpers of the GPU parity tests: error metrics of DESIGN.md 4 (reading G18) and drivers
that run the same seeded config through the oracle (CPU) and through the C ABI (GPU)."""
import numpy as np

CONS = ("E", "Mx", "My", "Mz", "R")
PRIM = ("e", "p", "n", "vx", "vy", "vz")
GROUPS = {"Mx": ("Mx", "My", "Mz"), "My": ("Mx", "My", "Mz"), "Mz": ("Mx", "My", "Mz"),
          "vx": ("vx", "vy", "vz"), "vy": ("vx", "vy", "vz"), "vz": ("vx", "vy", "vz")}


EPS = 2.0 ** -52


def n_allowance(ref):
    """Conditioning of n = R sqrt(1-v^2): one ulp of v moves n by n v dv/(1-v^2).  Where the
    causality projection holds v at 1-1e-12 this is ~1e-4 of the cell's n, on BOTH sides (the oracle's own n
    carries it).  |dn| up to 32 eps n/(1-v^2) is therefore not an error of either implementation."""
    v2 = sum(np.asarray(ref[c], dtype=np.float64) ** 2 for c in ("vx", "vy", "vz"))
    return 32.0 * EPS * np.abs(ref["n"]) / np.maximum(1.0 - v2, EPS)


def field_errors(got, ref):
    """per field: (err_max, err_L1) = (max|X-X*| / max|X*|, sum|X-X*| / sum|X*|); the three momentum
    (velocity) components share one denominator built from |M*| (|v*|).  For n the conditioning allowance
    n_allowance() is subtracted from |X-X*| first."""
    out = {}
    for k in ref:
        g = np.asarray(got[k], dtype=np.float64)
        r = np.asarray(ref[k], dtype=np.float64)
        if k in GROUPS:
            mag = np.sqrt(sum(np.asarray(ref[c], dtype=np.float64) ** 2 for c in GROUPS[k]))
        else:
            mag = np.abs(r)
        dmax, dsum = mag.max(), mag.sum()
        d = np.abs(g - r)
        if k == "n" and all(c in ref for c in ("vx", "vy", "vz")):
            d = np.maximum(d - n_allowance(ref), 0.0)
        out[k] = (d.max() / dmax if dmax > 0 else d.max(), d.sum() / dsum if dsum > 0 else d.sum())
    return out


def run_oracle(oracle, c, steps=None, table=None, variant="strict"):
    o = oracle.Oracle(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"],
                      variant=variant)
    if table is not None:
        o.set_sweep_table(table)
    o.set_state(c["e"], c["n"], c["vx"], c["vy"], c["vz"])
    o.step(c["steps"] if steps is None else steps)
    res = dict(o.get_conserved())
    res.update(o.get_primitives())
    return res, o


def run_gpu(c, steps=None, table=None, precision=64, segment=0, host_io=False, variant=0, no_tma=0):
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"],
               precision=precision, segment=segment, variant=variant, no_tma=no_tma)
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
