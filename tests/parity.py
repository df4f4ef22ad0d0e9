"""Shared helpers of the GPU parity tests: error metrics of DESIGN.md 4 (reading G18) and drivers
that run the same seeded config through the oracle (CPU) and through the C ABI (GPU)."""
import numpy as np

CONS = ("E", "Mx", "My", "Mz", "R")
PRIM = ("e", "p", "n", "vx", "vy", "vz")
GROUPS = {"Mx": ("Mx", "My", "Mz"), "My": ("Mx", "My", "Mz"), "Mz": ("Mx", "My", "Mz"),
          "vx": ("vx", "vy", "vz"), "vy": ("vx", "vy", "vz"), "vz": ("vx", "vy", "vz")}


def field_errors(got, ref):
    """per field: (err_max, err_L1) = (max|X-X*| / max|X*|, sum|X-X*| / sum|X*|); the three momentum
    (velocity) components share one denominator built from |M*| (|v*|)."""
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
        out[k] = (d.max() / dmax if dmax > 0 else d.max(), d.sum() / dsum if dsum > 0 else d.sum())
    return out


def run_oracle(oracle, c, steps=None, table=None):
    o = oracle.Oracle(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"])
    if table is not None:
        o.set_sweep_table(table)
    o.set_state(c["e"], c["n"], c["vx"], c["vy"], c["vz"])
    o.step(c["steps"] if steps is None else steps)
    res = dict(o.get_conserved())
    res.update(o.get_primitives())
    return res, o


def run_gpu(c, steps=None, table=None, precision=64, segment=0, host_io=False):
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"],
               precision=precision, segment=segment)
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
