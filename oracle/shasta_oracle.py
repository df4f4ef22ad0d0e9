"""ctypes wrapper around oracle/shasta_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It shares nothing with paper_1206_0919_b200 (the CUDA path).
All pointers are HOST pointers (numpy float64, C-contiguous, shape (nz, ny, nx), x fastest).
See shasta_oracle.c for the citations into PAPER.md.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "shasta_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_shasta.so")

BOUNDARY, EOS_MASS, STEP_INDEX, PREDICTOR, DIFF, ANTIDIFFUSION = 0, 1, 3, 4, 5, 6
PHOENICAL, EXPLICIT = 0, 1
R1, R2 = 0, 1
OUTFLOW, PERIODIC = 0, 1
BRANCH = (0, 1, 2, 0, 2, 1, 2, 0, 1, 2, 1, 0, 1, 2, 0, 1, 0, 2)


_LIB_FMA = os.path.join(_HERE, "liboracle_shasta_fma.so")


def build(force: bool = False, variant: str = "strict") -> str:
    """gcc -O2 -ffp-contract=off -fopenmp: plain C, no FMA contraction.
    variant="fma": the SAME source compiled with -ffp-contract=fast -mfma, i.e. an equally valid but
    differently rounded evaluation of the same formulas.  The distance between the two after s steps is the
    rounding-noise floor of the step map ("noise floor"); parity tests use it to scale the
    tolerance where 1e-10 is below what ANY two fp64 evaluations can agree to."""
    out, flags = (_LIB, ["-ffp-contract=off"]) if variant == "strict" else (_LIB_FMA, ["-ffp-contract=fast", "-mfma"])
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2"] + flags + ["-fopenmp", "-fPIC", "-shared", "-std=c11",
               "-Wall", "-Wextra", "-o", out, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return out


_libs = {}
_dp = C.POINTER(C.c_double)


class EosTable(C.Structure):
    """eos_table_t of shasta_oracle.c: p[i + ne*j] at (i de, j dn) (reading T1)."""
    _fields_ = [("ne", C.c_int), ("nn", C.c_int), ("de", C.c_double), ("dn", C.c_double), ("p", _dp)]


def make_table(p2d, e_max, n_max):
    """p2d: array (nn, ne), p2d[j, i] = P(i e_max/(ne-1), j n_max/(nn-1)).  Returns (EosTable, keep-alive array)."""
    a = np.ascontiguousarray(p2d, dtype=np.float64)
    nn, ne = a.shape
    return EosTable(ne, nn, e_max / (ne - 1), n_max / (nn - 1), a.ctypes.data_as(_dp)), a


def lib(variant: str = "strict"):
    if variant not in _libs:
        L = C.CDLL(build(variant=variant))
        L.oracle_create.restype = C.c_void_p
        L.oracle_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_set_option.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.oracle_set_sweep_table.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.c_int]
        L.oracle_set_state.argtypes = [C.c_void_p] + [_dp] * 5
        L.oracle_set_conserved.argtypes = [C.c_void_p] + [_dp] * 5
        L.oracle_get_conserved.argtypes = [C.c_void_p] + [_dp] * 5
        L.oracle_get_primitives.argtypes = [C.c_void_p] + [_dp] * 6
        L.oracle_step.argtypes = [C.c_void_p, C.c_int]
        L.oracle_conserved_totals.argtypes = [C.c_void_p, _dp]
        L.oracle_diagnostics.argtypes = [C.c_void_p, C.POINTER(C.c_ulonglong)]
        L.oracle_step_index.restype = C.c_longlong
        L.oracle_step_index.argtypes = [C.c_void_p]
        L.oracle_set_threads.argtypes = [C.c_int]
        L.oracle_get_threads.restype = C.c_int
        L.oracle_qplus.restype = C.c_double
        L.oracle_qplus.argtypes = [C.c_double, C.c_double]
        L.oracle_qminus.restype = C.c_double
        L.oracle_qminus.argtypes = [C.c_double, C.c_double]
        L.oracle_transport.argtypes = [C.c_int, _dp, _dp, _dp, C.c_double, _dp, C.c_int, C.c_int]
        L.oracle_antidiffuse.argtypes = [C.c_int, _dp, _dp, C.c_double, _dp, C.c_int, C.c_int]
        L.oracle_antidiffuse_kind.argtypes = [C.c_int, _dp, _dp, C.c_double, C.c_int, _dp, C.c_int, C.c_int]
        L.oracle_prim2cons.argtypes = [C.c_double] * 7 + [_dp]
        L.oracle_cons2prim.restype = C.c_int
        L.oracle_cons2prim.argtypes = [C.c_double] * 7 + [_dp, C.POINTER(C.c_int)]
        L.oracle_project.restype = C.c_int
        L.oracle_project.argtypes = [C.c_double, _dp]
        L.oracle_sweep_pencil.argtypes = [C.c_int, C.POINTER(_dp), C.c_int, C.c_double, C.c_double,
                                          C.c_double, C.c_int, C.POINTER(C.c_ulonglong)]
        L.oracle_sweep_pencil_ex.argtypes = [C.c_int, C.POINTER(_dp), C.c_int, C.c_double, C.c_double,
                                             C.c_double, C.c_int, C.POINTER(C.c_ulonglong), C.c_double, C.c_int]
        L.oracle_sweep_pencil_full.argtypes = [C.c_int, C.POINTER(_dp), C.c_int, C.c_double, C.c_double,
                                               C.c_double, C.c_int, C.POINTER(C.c_ulonglong), C.c_double, C.c_int,
                                               C.POINTER(EosTable), C.c_int]
        L.oracle_set_eos_table.argtypes = [C.c_void_p, _dp, C.c_int, C.c_int, C.c_double, C.c_double]
        L.oracle_eos_table_P.restype = C.c_double
        L.oracle_eos_table_P.argtypes = [C.POINTER(EosTable), C.c_double, C.c_double]
        L.oracle_prim2cons_eos.argtypes = [C.c_double] * 7 + [C.POINTER(EosTable), _dp]
        L.oracle_cons2prim_eos.restype = C.c_int
        L.oracle_cons2prim_eos.argtypes = [C.c_double] * 7 + [C.POINTER(EosTable), _dp, C.POINTER(C.c_int)]
        L.oracle_advect_pencil.argtypes = [C.c_int, _dp, _dp, C.c_double, C.c_int, C.c_int, _dp]
        L.oracle_set_threads(_threads[0])
        _libs[variant] = L
    return _libs[variant]


_threads = [1]


def _p(a):
    return a.ctypes.data_as(_dp)


def _arr(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def set_threads(n: int) -> None:
    _threads[0] = int(n)
    lib()
    for L in _libs.values():
        L.oracle_set_threads(int(n))


def get_threads() -> int:
    return lib().oracle_get_threads()


# ----------------------------------------------------------- building blocks (pins)
def qplus(eps_j, eps_jp1):
    return lib().oracle_qplus(eps_j, eps_jp1)


def qminus(eps_j, eps_jm1):
    return lib().oracle_qminus(eps_j, eps_jm1)


def transport(U, eps, f, lam, lo, hi):
    """eq. (17) on one extended pencil; returns Uhat (only [lo,hi) is meaningful)."""
    U, eps = _arr(U), _arr(eps)
    out = np.zeros_like(U)
    fp = None
    if f is not None:
        f = _arr(f)
        fp = _p(f)
    lib().oracle_transport(len(U), _p(U), _p(eps), fp, lam, _p(out), lo, hi)
    return out


def antidiffuse(U, Uhat, lo, hi, diff=1.0, kind=PHOENICAL):
    U, Uhat = _arr(U), _arr(Uhat)
    out = np.zeros_like(U)
    if kind == PHOENICAL:
        lib().oracle_antidiffuse(len(U), _p(U), _p(Uhat), diff, _p(out), lo, hi)
    else:
        lib().oracle_antidiffuse_kind(len(U), _p(U), _p(Uhat), diff, kind, _p(out), lo, hi)
    return out


def prim2cons(e, n, vx, vy, vz, gamma, mass=0.0):
    out = np.zeros(5)
    lib().oracle_prim2cons(e, n, vx, vy, vz, gamma, mass, _p(out))
    return out


def cons2prim(E, Mx, My, Mz, R, gamma, mass=0.0):
    """returns (array [e,p,n,vx,vy,vz,|v|], iterations, flags[2])."""
    out = np.zeros(7)
    fl = (C.c_int * 2)(0, 0)
    it = lib().oracle_cons2prim(E, Mx, My, Mz, R, gamma, mass, _p(out), fl)
    return out, it, (fl[0], fl[1])


def eos_table_P(tab, e, n):
    return lib().oracle_eos_table_P(C.byref(tab[0]), e, n)


def prim2cons_table(e, n, vx, vy, vz, tab):
    out = np.zeros(5)
    lib().oracle_prim2cons_eos(e, n, vx, vy, vz, 4.0 / 3.0, 0.0, C.byref(tab[0]), _p(out))
    return out


def cons2prim_table(E, Mx, My, Mz, R, tab):
    out = np.zeros(7)
    fl = (C.c_int * 2)(0, 0)
    it = lib().oracle_cons2prim_eos(E, Mx, My, Mz, R, 4.0 / 3.0, 0.0, C.byref(tab[0]), _p(out), fl)
    return out, it, (fl[0], fl[1])


def project(E, M):
    m = np.array(M, dtype=np.float64)
    r = lib().oracle_project(E, _p(m))
    return m, r


def sweep_pencil(U5, axis, lam, gamma, mass=0.0, bc=OUTFLOW, diff=1.0, predictor=R1, antidiffusion=PHOENICAL):
    """U5: (5, N) array; returns the swept copy and the counts [Pi fired, vacuum]."""
    U5 = np.array(U5, dtype=np.float64, order="C")
    N = U5.shape[1]
    ptrs = (_dp * 5)(*[_p(U5[f]) for f in range(5)])
    cnt = (C.c_ulonglong * 2)(0, 0)
    if antidiffusion != PHOENICAL:
        lib().oracle_sweep_pencil_full(N, ptrs, axis, lam, gamma, mass, bc, cnt, diff, predictor, None, antidiffusion)
    elif diff == 1.0 and predictor == R1:
        lib().oracle_sweep_pencil(N, ptrs, axis, lam, gamma, mass, bc, cnt)
    else:
        lib().oracle_sweep_pencil_ex(N, ptrs, axis, lam, gamma, mass, bc, cnt, diff, predictor)
    return U5, (cnt[0], cnt[1])


def advect_pencil(U, vel, lam, bc, nsteps):
    """P5 helper: prescribed-velocity source-free advection; returns (U_new, Uhat of last step)."""
    U = np.array(U, dtype=np.float64)
    vel = _arr(vel)
    uh = np.zeros_like(U)
    lib().oracle_advect_pencil(len(U), _p(U), _p(vel), lam, bc, nsteps, _p(uh))
    return U, uh


# ----------------------------------------------------------------------- the grid
class Oracle:
    """Same call sequence as the product's C ABI (include/shasta.h) with host arrays."""

    def __init__(self, nx, ny, nz, dx, lam, eos_gamma, boundary=OUTFLOW, eos_mass=0.0, variant="strict",
                 predictor=R1, diff=1.0, eos_table=None, antidiffusion=PHOENICAL):
        self._L = lib(variant)
        self.shape = (nz, ny, nx)
        self._h = self._L.oracle_create(nx, ny, nz, dx, lam, eos_gamma)
        if not self._h:
            raise ValueError("oracle_create: bad argument")
        self.set_option(BOUNDARY, boundary)
        self.set_option(EOS_MASS, eos_mass)
        if predictor != R1:
            self.set_option(PREDICTOR, predictor)
        if diff != 1.0:
            self.set_option(DIFF, diff)
        if antidiffusion != PHOENICAL:
            self.set_option(ANTIDIFFUSION, antidiffusion)
        if eos_table is not None:           # (p2d (nn, ne), e_max, n_max)
            a = np.ascontiguousarray(eos_table[0], dtype=np.float64)
            self._chk(self._L.oracle_set_eos_table(self._h, _p(a), a.shape[1], a.shape[0], float(eos_table[1]),
                                                   float(eos_table[2])), "oracle_set_eos_table")

    def __del__(self):
        if getattr(self, "_h", None):
            self._L.oracle_destroy(self._h)
            self._h = None

    def _chk(self, rc, what):
        if rc != 0:
            raise RuntimeError(f"{what} failed: {rc}")

    def set_option(self, key, value):
        self._chk(self._L.oracle_set_option(self._h, key, float(value)), "oracle_set_option")

    def set_sweep_table(self, axes):
        a = (C.c_int * len(axes))(*axes)
        self._chk(self._L.oracle_set_sweep_table(self._h, a, len(axes)), "oracle_set_sweep_table")

    def set_state(self, e, n, vx, vy, vz):
        arrs = [_arr(x).reshape(self.shape) for x in (e, n, vx, vy, vz)]
        self._chk(self._L.oracle_set_state(self._h, *[_p(a) for a in arrs]), "oracle_set_state")

    def set_conserved(self, E, Mx, My, Mz, R):
        arrs = [_arr(x).reshape(self.shape) for x in (E, Mx, My, Mz, R)]
        self._chk(self._L.oracle_set_conserved(self._h, *[_p(a) for a in arrs]), "oracle_set_conserved")

    def step(self, nsteps=1):
        self._chk(self._L.oracle_step(self._h, int(nsteps)), "oracle_step")

    def get_conserved(self):
        out = [np.empty(self.shape) for _ in range(5)]
        self._chk(self._L.oracle_get_conserved(self._h, *[_p(a) for a in out]), "oracle_get_conserved")
        return dict(zip(("E", "Mx", "My", "Mz", "R"), out))

    def get_primitives(self):
        out = [np.empty(self.shape) for _ in range(6)]
        self._chk(self._L.oracle_get_primitives(self._h, *[_p(a) for a in out]), "oracle_get_primitives")
        return dict(zip(("e", "p", "n", "vx", "vy", "vz"), out))

    def conserved_totals(self):
        t = np.zeros(5)
        self._chk(self._L.oracle_conserved_totals(self._h, _p(t)), "oracle_conserved_totals")
        return t

    def diagnostics(self):
        c = (C.c_ulonglong * 4)()
        self._chk(self._L.oracle_diagnostics(self._h, c), "oracle_diagnostics")
        return [int(x) for x in c]

    @property
    def step_index(self):
        return int(self._L.oracle_step_index(self._h))
