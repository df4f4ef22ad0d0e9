"""Seeded, synthetic initial states for the five BASELINE.json configs.

This module serves BOTH the oracle tests and the CUDA path and therefore holds none of the
method's arithmetic: it only builds primitive fields (e, n, vx, vy, vz) as numpy float64
arrays of shape (nz, ny, nx) (x fastest) plus the run parameters.  It imports neither
`oracle/` nor the CUDA binding.  Nothing here is taken from a dataset: the paper's own
workloads (expanding ball, UrQMD Au+Au initial state) are not in the
container; configs 2-4 stand in for them with the same grid scale, dx and lambda.
"""
from __future__ import annotations

import numpy as np

OUTFLOW, PERIODIC = 0, 1
SEED = 12060919


def _centres(n, dx):
    """symmetric cell centres c_i = (i - (n-1)/2) dx"""
    return (np.arange(n, dtype=np.float64) - 0.5 * (n - 1)) * dx


def _cfg(name, nx, ny, nz, dx, steps, bc, gamma, mass, e, n, vx, vy, vz, lam=0.4):
    shape = (nz, ny, nx)
    f = lambda a: np.array(np.broadcast_to(a, shape), dtype=np.float64, order="C")     # writable copy
    return dict(name=name, nx=nx, ny=ny, nz=nz, dx=float(dx), lam=float(lam), steps=int(steps),
                boundary=bc, gamma=float(gamma), mass=float(mass),
                e=f(e), n=f(n), vx=f(vx), vy=f(vy), vz=f(vz))


def shock_tube(ncell=400, e_right=0.01, axis=0, transverse=1, steps=None):
    """Config 1: 1D relativistic Riemann problem on [-1,1], e_L=1, v=0, n=e^(3/4), p=e/3.
    `axis` lays the tube along x/y/z; `transverse` is the extent of the two other axes."""
    dx = 2.0 / ncell
    x = -1.0 + (np.arange(ncell) + 0.5) * dx
    e1 = np.where(x < 0.0, 1.0, e_right)
    dims = [transverse] * 3
    dims[axis] = ncell
    nx, ny, nz = dims
    sh = [1, 1, 1]
    sh[2 - axis] = ncell
    e = e1.reshape(sh)
    steps = ncell // 2 if steps is None else steps          # t = steps*0.4*dx = 0.4 at 400 cells
    return _cfg("shock_tube", nx, ny, nz, dx, steps, OUTFLOW, 4.0 / 3.0, 0.0,
                e, e ** 0.75, 0.0, 0.0, 0.0)


def fireball(n=64, steps=100):
    """Config 2: Gaussian fireball, box fixed at 64*0.2 fm, e = 10 exp(-r^2/(2*1.5^2)) + 1e-6."""
    dx = 0.2 * 64 / n
    c = _centres(n, dx)
    r2 = c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2
    e = 10.0 * np.exp(-r2 / (2.0 * 1.5 ** 2)) + 1e-6
    return _cfg("fireball", n, n, n, dx, steps, OUTFLOW, 4.0 / 3.0, 0.0, e, e ** 0.75, 0.0, 0.0, 0.0)


def spherical_riemann(n=128, steps=100, p_in=1.0, p_out=0.01):
    """Config 3: sphere of radius 2.0 (20 cells at 128^3) at pressure ratio 100:1, n=1,
    p=(Gamma-1)(e-n), Gamma=5/3, periodic."""
    dx = 0.1 * 128 / n
    c = _centres(n, dx)
    r2 = c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2
    gamma = 5.0 / 3.0
    p = np.where(r2 < 2.0 ** 2, p_in, p_out)
    nn = np.ones_like(p)
    e = nn + p / (gamma - 1.0)
    return _cfg("spherical_riemann", n, n, n, dx, steps, PERIODIC, gamma, 1.0, e, nn, 0.0, 0.0, 0.0)


def hotspots(n=256, steps=200, seed=SEED):
    """Config 4: 50 Gaussian hotspots + longitudinal flow vz = tanh(z/4); box +-12.8 fm."""
    dx = 0.1 * 256 / n
    rng = np.random.default_rng(seed)
    centres = rng.uniform(-7.68, 7.68, (50, 3))
    w = rng.uniform(0.4, 1.0, 50)
    amp = 20.0 * rng.lognormal(0.0, 0.5, 50)
    c = _centres(n, dx)
    e = np.full((n, n, n), 1e-6)
    for k in range(50):
        gx = np.exp(-(c - centres[k, 0]) ** 2 / (2.0 * w[k] ** 2))
        gy = np.exp(-(c - centres[k, 1]) ** 2 / (2.0 * w[k] ** 2))
        gz = np.exp(-(c - centres[k, 2]) ** 2 / (2.0 * w[k] ** 2))
        e += amp[k] * gz[:, None, None] * gy[None, :, None] * gx[None, None, :]
    vz = np.tanh(c / 4.0)[:, None, None]
    return _cfg("hotspots", n, n, n, dx, steps, OUTFLOW, 4.0 / 3.0, 0.0, e, e ** 0.75, 0.0, 0.0, vz)


def hotspots_crop(n=96, steps=200, lo=(80, 80, 160), seed=SEED):
    """Config 4 at its own resolution on a sub-box: the n^3 cells starting at lo=(ix,iy,iz) of the 256^3
    hotspots state (dx = 0.1 fm).  The default box touches the +z face, where vz = tanh(z/4) reaches
    gamma = 12, so the outflow boundary is exercised at high Lorentz factor."""
    c = hotspots(256, steps=steps, seed=seed)
    sl = (slice(lo[2], lo[2] + n), slice(lo[1], lo[1] + n), slice(lo[0], lo[0] + n))
    f = {k: np.ascontiguousarray(c[k][sl]) for k in ("e", "n", "vx", "vy", "vz")}
    return _cfg("hotspots_crop", n, n, n, c["dx"], steps, OUTFLOW, c["gamma"], c["mass"],
                f["e"], f["n"], f["vx"], f["vy"], f["vz"])


def slabs(n=512, steps=100, nxy=None):
    """Config 5: two Woods-Saxon slabs at z=+-6 moving with vz=-+0.9; uniform in x,y
    (nxy=1 gives the 1x1xn column whose broadcast is the full 3D answer, pin P11)."""
    dx = 0.05 * 512 / n
    nxy = n if nxy is None else nxy
    z = _centres(n, dx)
    e1 = 1e-6 + 5.0 / (1.0 + np.exp((np.abs(z - 6.0) - 1.5) / 0.5)) \
              + 5.0 / (1.0 + np.exp((np.abs(z + 6.0) - 1.5) / 0.5))
    vz1 = -0.9 * np.sign(z)
    e = e1[:, None, None]
    return _cfg("slabs", nxy, nxy, n, dx, steps, OUTFLOW, 4.0 / 3.0, 0.0,
                e, e ** 0.75, 0.0, 0.0, vz1[:, None, None])


def random_state(nx, ny, nz, seed=0, kind="smooth", vmax=0.6, gamma=4.0 / 3.0, mass=0.0,
                 boundary=OUTFLOW):
    """Kernel-level parity inputs: 'smooth' = a few random Fourier modes; 'rough' = smooth plus
    random blocks with jumps in e and v (limiter and projection active)."""
    rng = np.random.default_rng(seed)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")

    def modes(nm):
        f = np.zeros((nz, ny, nx))
        for _ in range(nm):
            k = rng.integers(0, 3, 3)
            ph = rng.uniform(0, 2 * np.pi)
            f += rng.normal() * np.cos(2 * np.pi * (k[0] * x / max(nx, 1) + k[1] * y / max(ny, 1)
                                                    + k[2] * z / max(nz, 1)) + ph)
        return f / np.sqrt(nm)

    e = np.exp(modes(4))
    v = [np.tanh(0.5 * modes(3)) for _ in range(3)]
    if kind == "rough":
        for _ in range(6):
            lo = [rng.integers(0, s) for s in (nz, ny, nx)]
            hi = [min(s, l + 1 + rng.integers(0, max(s // 2, 1))) for s, l in zip((nz, ny, nx), lo)]
            sl = tuple(slice(l, h) for l, h in zip(lo, hi))
            e[sl] *= 10.0 ** rng.uniform(-3, 2)
            for c in range(3):
                v[c][sl] = rng.uniform(-1, 1)
    norm = np.sqrt(v[0] ** 2 + v[1] ** 2 + v[2] ** 2)
    scale = np.where(norm > vmax, vmax / np.maximum(norm, 1e-300), 1.0)
    v = [c * scale for c in v]
    n = e ** 0.75 if mass == 0.0 else 0.3 * e ** 0.75
    return _cfg(f"random_{kind}", nx, ny, nz, 1.0, 1, boundary, gamma, mass, e, n, v[2], v[1], v[0])


CONFIGS = {
    "shock_tube": shock_tube, "fireball": fireball, "spherical_riemann": spherical_riemann,
    "hotspots": hotspots, "hotspots_crop": hotspots_crop, "slabs": slabs,
}


# ------------------------------------------------------------------ synthetic tabled equations of state (row f1)
def eos_table(kind="soft", ne=193, nn=49, e_max=12.0, n_max=4.0, gamma=5.0 / 3.0, mass=1.0):
    """A pressure table P(e_i, n_j), e_i = i e_max/(ne-1), n_j = j n_max/(nn-1), as (p2d (nn, ne), e_max, n_max): the
    argument of shasta_set_eos_table and of the oracle's eos_table option.  No physical table is in the container
    (PAPER.md:36 only names "non analytic equations of state"); two synthetic ones stand in:
      "ideal"  the ideal gas (gamma-1)(e - m n) sampled on the grid (bilinear interpolation returns it exactly),
      "soft"   a smooth causal crossover, p = e/3 (1 - 0.25 exp(-(e-2)^2/2)) + 0.05 n^2/(1+n)  (0 < dp/de < 0.45)."""
    e = np.linspace(0.0, e_max, ne)[None, :]
    n = np.linspace(0.0, n_max, nn)[:, None]
    if kind == "ideal":
        p = (gamma - 1.0) * (e - mass * n)
    elif kind == "soft":
        p = e / 3.0 * (1.0 - 0.25 * np.exp(-0.5 * (e - 2.0) ** 2)) + 0.05 * n * n / (1.0 + n) + 0.0 * e
    else:
        raise ValueError(kind)
    return np.ascontiguousarray(p, dtype=np.float64), float(e_max), float(n_max)
