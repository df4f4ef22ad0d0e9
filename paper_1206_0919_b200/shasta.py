"""Thin Python binding over the C ABI of csrc/libshasta.so (include/shasta.h).

Argument marshalling only: every step of the path runs in the CUDA kernels.  PyTorch is used for
device memory and streams (torch tensors of shape (nz, ny, nx), float64, on cuda).  There is no
CPU fallback: if the library is missing or cannot be loaded this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libshasta.so")

BOUNDARY, EOS_MASS, PRECISION, STEP_INDEX, SEGMENT, VARIANT, NO_TMA, PREDICTOR, DIFF, CELL_PATH, NO_DEFER, PRIMS_RAW, BATCH, GRAPH, ANTIDIFFUSION, BOUNDARY_Z = range(16)
R1, R2 = 0, 1
PHOENICAL, EXPLICIT = 0, 1
OUTFLOW, PERIODIC = 0, 1
BRANCH = (0, 1, 2, 0, 2, 1, 2, 0, 1, 2, 1, 0, 1, 2, 0, 1, 0, 2)

# every symbol include/shasta.h declares
SYMBOLS = (
    "shasta_create", "shasta_destroy", "shasta_set_option", "shasta_set_eos_table", "shasta_set_sweep_table", "shasta_set_state",
    "shasta_set_state_host", "shasta_set_conserved", "shasta_get_conserved", "shasta_get_planes", "shasta_set_planes", "shasta_plane_ptr", "shasta_set_active_planes", "shasta_step", "shasta_sweep",
    "shasta_get_primitives", "shasta_get_primitives_host", "shasta_conserved_totals", "shasta_diagnostics",
    "shasta_launch_count", "shasta_graph_launch_count", "shasta_step_index", "shasta_kernel_name", "shasta_last_error",
    "shasta_conserved_totals_static", "shasta_conserved_totals_static_max_cells",
)

_lib = None
_vp, _dp = C.c_void_p, C.c_void_p     # device/host pointers are passed as integers


def load():
    """dlopen libshasta.so; raises (no fallback) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(
            f"{LIB_PATH} not found: build it with `python -m paper_1206_0919_b200.build` "
            "(or __graft_entry__.build()).  There is no CPU fallback.")
    L = C.CDLL(LIB_PATH)
    L.shasta_create.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double]
    L.shasta_destroy.argtypes = [_vp]
    L.shasta_destroy.restype = None
    L.shasta_set_option.argtypes = [_vp, C.c_int, C.c_double]
    L.shasta_set_eos_table.argtypes = [_vp, _dp, C.c_int, C.c_int, C.c_double, C.c_double]
    L.shasta_set_sweep_table.argtypes = [_vp, C.POINTER(C.c_int), C.c_int]
    L.shasta_set_state.argtypes = [_vp] + [_dp] * 5 + [_vp]
    L.shasta_set_state_host.argtypes = [_vp] + [_dp] * 5 + [_vp]
    L.shasta_set_conserved.argtypes = [_vp] + [_dp] * 5 + [_vp]
    L.shasta_get_conserved.argtypes = [_vp] + [_dp] * 5 + [_vp]
    L.shasta_get_planes.argtypes = [_vp, C.c_int, C.c_int] + [_dp] * 5 + [_vp]
    L.shasta_set_planes.argtypes = [_vp, C.c_int, C.c_int] + [_dp] * 5 + [_vp]
    L.shasta_plane_ptr.argtypes = [_vp, C.c_int, C.c_int, C.POINTER(_vp)]
    L.shasta_set_active_planes.argtypes = [_vp, C.c_int, C.c_int]
    L.shasta_step.argtypes = [_vp, C.c_int, _vp]
    L.shasta_sweep.argtypes = [_vp, C.c_int, C.c_int, _vp]
    L.shasta_get_primitives.argtypes = [_vp] + [_dp] * 6 + [_vp]
    L.shasta_get_primitives_host.argtypes = [_vp] + [_dp] * 6 + [_vp]
    L.shasta_conserved_totals.argtypes = [_vp, C.POINTER(C.c_double), _vp]
    L.shasta_diagnostics.argtypes = [_vp, C.POINTER(C.c_ulonglong)]
    L.shasta_launch_count.argtypes = [_vp]
    L.shasta_launch_count.restype = C.c_longlong
    L.shasta_graph_launch_count.argtypes = [_vp]
    L.shasta_graph_launch_count.restype = C.c_longlong
    L.shasta_step_index.argtypes = [_vp]
    L.shasta_step_index.restype = C.c_longlong
    L.shasta_kernel_name.argtypes = [_vp, C.c_int]
    L.shasta_kernel_name.restype = C.c_char_p
    L.shasta_last_error.argtypes = [_vp]
    L.shasta_last_error.restype = C.c_char_p
    L.shasta_conserved_totals_static.argtypes = [C.c_longlong] + [_dp] * 5 + [C.c_double, _dp, _vp]
    L.shasta_conserved_totals_static_max_cells.argtypes = []
    L.shasta_conserved_totals_static_max_cells.restype = C.c_longlong
    _lib = L
    return L


class ShastaError(RuntimeError):
    pass


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dev(t):
    import torch
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise ValueError("expected a contiguous float64 CUDA tensor")
    return C.c_void_p(t.data_ptr())


def _host(t):
    import torch
    if t is None:
        return None
    if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise ValueError("expected a contiguous float64 CPU tensor")
    return C.c_void_p(t.data_ptr())


def conserved_totals_static_max_cells():
    return int(load().shasta_conserved_totals_static_max_cells())


def conserved_totals_static(E, Mx, My, Mz, R, dv, out, stream=None):
    """shasta_conserved_totals_static: dv * sums of five float64 CUDA tensors into `out` (5 doubles, CUDA), no allocation,
    asynchronous on `stream`.  Marshalling only; sizes beyond the static scratch array raise ShastaError."""
    L = load()
    n = E.numel()
    if any(t.numel() != n for t in (Mx, My, Mz, R)) or out.numel() != 5:
        raise ValueError("five fields of equal size and an output of 5 doubles expected")
    rc = L.shasta_conserved_totals_static(n, _dev(E), _dev(Mx), _dev(My), _dev(Mz), _dev(R), float(dv), _dev(out),
                                          _stream_ptr(stream))
    if rc != 0:
        raise ShastaError(f"shasta_conserved_totals_static failed ({rc}): {L.shasta_last_error(None).decode()}")
    return out


class _DeviceMemory:
    """memory owned by a handle, seen through __cuda_array_interface__ (torch.as_tensor makes a view, not a copy)"""

    def __init__(self, ptr, shape, typestr):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 2, "strides": None}


class Shasta:
    """One solver handle = shasta_create ... shasta_destroy.  Method names follow the C ABI."""

    def __init__(self, nx, ny, nz, dx, lam, eos_gamma, boundary=OUTFLOW, eos_mass=0.0, precision=64,
                 segment=0, no_tma=0, predictor=0, diff=1.0, cell_path=0, no_defer=0, batch=1, graph=None, eos_table=None,
                 antidiffusion=PHOENICAL, boundary_z=None):
        L = load()
        self._L = L
        self._h = _vp()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.batch = int(batch)
        self.shape = (self.nz, self.ny, self.nx) if self.batch == 1 else (self.batch, self.nz, self.ny, self.nx)
        rc = L.shasta_create(C.byref(self._h), nx, ny, nz, dx, lam, eos_gamma)
        if rc != 0:
            msg = L.shasta_last_error(None).decode()
            self._h = _vp()
            raise ShastaError(f"shasta_create failed ({rc}): {msg}")
        self.set_option(BOUNDARY, boundary)
        self.set_option(EOS_MASS, eos_mass)
        self.set_option(PRECISION, precision)
        self._typestr = "<f8" if int(precision) == 64 else "<f4"
        self._views = {}
        if segment:
            self.set_option(SEGMENT, segment)
        if no_tma:
            self.set_option(NO_TMA, 1)
        if predictor:
            self.set_option(PREDICTOR, predictor)
        if diff != 1.0:
            self.set_option(DIFF, diff)
        if cell_path:
            self.set_option(CELL_PATH, 1)
        if no_defer:
            self.set_option(NO_DEFER, 1)
        if self.batch != 1:
            self.set_option(BATCH, self.batch)
        if graph is not None:
            self.set_option(GRAPH, graph)
        if eos_table is not None:
            self.set_eos_table(*eos_table)
        if antidiffusion:
            self.set_option(ANTIDIFFUSION, antidiffusion)
        if boundary_z is not None:
            self.set_option(BOUNDARY_Z, boundary_z)

    def close(self, _null=C.c_void_p):           # _null bound at definition: module globals may be gone when __del__ runs at exit
        if getattr(self, "_h", None) and self._h.value:
            self._views = {}
            self._L.shasta_destroy(self._h)
            self._h = _null()

    __del__ = close

    def _chk(self, rc, what):
        if rc != 0:
            raise ShastaError(f"{what} failed ({rc}): {self._L.shasta_last_error(self._h).decode()}")

    def set_option(self, key, value):
        self._chk(self._L.shasta_set_option(self._h, key, float(value)), "shasta_set_option")

    def set_eos_table(self, p2d, e_max, n_max):
        """p2d: CPU float64 tensor or array of shape (nn, ne), p2d[j, i] = P(i e_max/(ne-1), j n_max/(nn-1)); None = analytic."""
        import torch
        if p2d is None:
            self._chk(self._L.shasta_set_eos_table(self._h, None, 0, 0, 0.0, 0.0), "shasta_set_eos_table")
            return
        t = torch.as_tensor(p2d, dtype=torch.float64).contiguous().cpu()
        nn, ne = t.shape
        self._chk(self._L.shasta_set_eos_table(self._h, C.c_void_p(t.data_ptr()), ne, nn, float(e_max), float(n_max)),
                  "shasta_set_eos_table")

    def set_sweep_table(self, axes):
        a = (C.c_int * len(axes))(*axes)
        self._chk(self._L.shasta_set_sweep_table(self._h, a, len(axes)), "shasta_set_sweep_table")

    def set_state(self, e, n, vx, vy, vz, stream=None):
        self._chk(self._L.shasta_set_state(self._h, _dev(e), _dev(n), _dev(vx), _dev(vy), _dev(vz),
                                           _stream_ptr(stream)), "shasta_set_state")

    def set_state_host(self, e, n, vx, vy, vz, stream=None):
        self._chk(self._L.shasta_set_state_host(self._h, _host(e), _host(n), _host(vx), _host(vy), _host(vz),
                                                _stream_ptr(stream)), "shasta_set_state_host")

    def set_conserved(self, E, Mx, My, Mz, R, stream=None):
        self._chk(self._L.shasta_set_conserved(self._h, _dev(E), _dev(Mx), _dev(My), _dev(Mz), _dev(R),
                                               _stream_ptr(stream)), "shasta_set_conserved")

    def step(self, nsteps=1, stream=None):
        self._chk(self._L.shasta_step(self._h, int(nsteps), _stream_ptr(stream)), "shasta_step")

    def sweep(self, axis, emit_primitives=False, stream=None):
        self._chk(self._L.shasta_sweep(self._h, int(axis), int(emit_primitives), _stream_ptr(stream)),
                  "shasta_sweep")

    def get_conserved(self, stream=None):
        import torch
        out = [torch.empty(self.shape, dtype=torch.float64, device="cuda") for _ in range(5)]
        self._chk(self._L.shasta_get_conserved(self._h, *[_dev(t) for t in out], _stream_ptr(stream)),
                  "shasta_get_conserved")
        return dict(zip(("E", "Mx", "My", "Mz", "R"), out))

    def get_planes(self, z0, nplanes, out=None, stream=None):
        """planes z0 .. z0+nplanes-1 of the conserved state as a (5, nplanes, ny, nx) CUDA tensor (fields E, Mx, My, Mz, R)"""
        import torch
        if out is None:
            out = torch.empty((5, int(nplanes), self.ny, self.nx), dtype=torch.float64, device="cuda")
        self._chk(self._L.shasta_get_planes(self._h, int(z0), int(nplanes), *[_dev(out[f]) for f in range(5)],
                                            _stream_ptr(stream)), "shasta_get_planes")
        return out

    def set_planes(self, z0, planes, stream=None):
        """planes: (5, nplanes, ny, nx) CUDA tensor written over planes z0 .. z0+nplanes-1 of the conserved state"""
        self._chk(self._L.shasta_set_planes(self._h, int(z0), int(planes.shape[1]), *[_dev(planes[f]) for f in range(5)],
                                            _stream_ptr(stream)), "shasta_set_planes")

    def set_active_planes(self, z_lo, z_hi):
        self._chk(self._L.shasta_set_active_planes(self._h, int(z_lo), int(z_hi)), "shasta_set_active_planes")

    def plane_views(self, z0, nplanes):
        """shasta_plane_ptr: the planes z0 .. z0+nplanes-1 of the five conserved fields as five CUDA tensors (nplanes, ny, nx)
        that ALIAS the handle's current state buffer (storage dtype); valid until the next sweep / step / set_* call."""
        import torch
        if not (0 <= z0 and nplanes >= 1 and z0 + nplanes <= self.nz):
            raise ValueError("planes outside the grid")
        out = []
        for f in range(5):
            p = _vp()
            self._chk(self._L.shasta_plane_ptr(self._h, f, int(z0), C.byref(p)), "shasta_plane_ptr")
            key = (p.value, int(nplanes))                # the two state buffers live as long as the handle: wrap each once
            t = self._views.get(key)
            if t is None:
                t = torch.as_tensor(_DeviceMemory(p.value, (int(nplanes), self.ny, self.nx), self._typestr), device="cuda")
                self._views[key] = t
            out.append(t)
        return out

    def get_primitives(self, stream=None, out=None):
        import torch
        if out is None:
            out = [torch.empty(self.shape, dtype=torch.float64, device="cuda") for _ in range(6)]
        self._chk(self._L.shasta_get_primitives(self._h, *[_dev(t) for t in out], _stream_ptr(stream)),
                  "shasta_get_primitives")
        return dict(zip(("e", "p", "n", "vx", "vy", "vz"), out))

    def get_primitives_host(self, out, stream=None):
        """out: list of 6 CPU float64 tensors (None = skip), ideally pinned."""
        self._chk(self._L.shasta_get_primitives_host(self._h, *[_host(t) for t in out], _stream_ptr(stream)),
                  "shasta_get_primitives_host")
        return out

    def conserved_totals(self, stream=None):
        t = (C.c_double * (5 * self.batch))()
        self._chk(self._L.shasta_conserved_totals(self._h, t, _stream_ptr(stream)), "shasta_conserved_totals")
        v = [float(x) for x in t]
        return v if self.batch == 1 else [v[5 * b:5 * b + 5] for b in range(self.batch)]

    def diagnostics(self):
        c = (C.c_ulonglong * 4)()
        self._chk(self._L.shasta_diagnostics(self._h, c), "shasta_diagnostics")
        return [int(x) for x in c]

    @property
    def launch_count(self):
        return int(self._L.shasta_launch_count(self._h))

    @property
    def graph_launch_count(self):
        return int(self._L.shasta_graph_launch_count(self._h))

    @property
    def step_index(self):
        return int(self._L.shasta_step_index(self._h))

    def kernel_name(self, axis):
        return self._L.shasta_kernel_name(self._h, axis).decode()
