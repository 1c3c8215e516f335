"""ORACLE — test infrastructure, not the product.

ctypes binding of ``oracle/pic_oracle.cpp`` (the plain serial CPU statement of the PIC step,
see that file's header for citations and pins). Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.
It imports nothing from ``paper_2101_12149_b200`` and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pic_oracle.cpp")
# ORACLE_SANITIZE=1: an AddressSanitizer + UndefinedBehaviorSanitizer build of the same source, loaded instead
# (run python with libasan / libubsan preloaded — command in profiles/oracle_sanitizers.md)
_SANITIZE = os.environ.get("ORACLE_SANITIZE", "") == "1"
_LIB = os.path.join(_HERE, "liboracle_san.so" if _SANITIZE else "liboracle.so")

DIAG = ("field_E", "field_B", "kinetic", "charge", "gauss_max", "rho_max", "deactivated", "steps")


def build(force: bool = False) -> str:
    """Compile the oracle (g++ -O2 -ffp-contract=off -fopenmp). Returns the library path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        extra = ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if _SANITIZE else []
        subprocess.check_call(
            ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC"] + extra +
            ["-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, i32p, i64p, dp = C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_double)
        L.orc_create.restype = vp
        L.orc_create.argtypes = [i32p, dp, C.c_double, C.c_int, C.c_int, i32p, i32p, C.c_int, C.c_int]
        L.orc_destroy.argtypes = [vp]
        L.orc_add_species.argtypes = [vp, C.c_int64] + [vp] * 7 + [C.c_double, C.c_double]
        L.orc_set_fields.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]
        L.orc_step.argtypes = [vp, C.c_int]
        L.orc_step_omp.argtypes = [vp, C.c_int, C.c_int]
        L.orc_step_omp.restype = C.c_int
        L.orc_get_fields.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
        L.orc_num_particles.restype = C.c_int64
        L.orc_num_particles.argtypes = [vp, C.c_int]
        L.orc_get_particles.argtypes = [vp, C.c_int] + [vp] * 7 + [i64p]
        L.orc_get_sort_state.argtypes = [vp, C.c_int, i32p, i32p]
        L.orc_get_diagnostics.argtypes = [vp, dp]
        L.orc_get_rho.argtypes = [vp, dp]
        L.orc_sort_now.argtypes = [vp]
        L.orc_field_step.argtypes = [vp, C.c_int]
        L.orc_particle_step.argtypes = [vp]
        L.orc_shape_f64.argtypes = [C.c_int, C.c_double, i32p, dp]
        L.orc_shape_f32.argtypes = [C.c_int, C.c_float, i32p, C.POINTER(C.c_float)]
        L.orc_create_ex.restype = vp
        L.orc_create_ex.argtypes = L.orc_create.argtypes + [C.c_int]
        L.orc_ckc_coefficients.argtypes = [vp, dp]
        L.orc_set_method.argtypes = [vp, C.c_int, C.c_int]
        L.orc_set_method.restype = C.c_int
        L.orc_vay_f64.argtypes = [C.c_double, dp, dp, dp]
        L.orc_vay_f32.argtypes = [C.c_float] + [C.POINTER(C.c_float)] * 3
        L.orc_boris_f64.argtypes = [C.c_double, dp, dp, dp]
        L.orc_boris_f32.argtypes = [C.c_float] + [C.POINTER(C.c_float)] * 3
        L.orc_gather.argtypes = [vp, C.c_int64, vp, vp, vp, vp]
        L.orc_deposit_moves.argtypes = [vp, C.c_int, C.c_int64, vp, vp, vp]
        L.orc_const_c.restype = C.c_double
        L.orc_const_eps0.restype = C.c_double
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def _i32(v):
    return (C.c_int32 * 3)(*[int(t) for t in v])


def shape(order: int, xi: float, dtype=np.float64):
    """(leftmost index, weights[order+1]) — oracle step 2a."""
    l = C.c_int32()
    if np.dtype(dtype) == np.float64:
        w = (C.c_double * 4)()
        lib().orc_shape_f64(order, float(xi), C.byref(l), w)
    else:
        w = (C.c_float * 4)()
        lib().orc_shape_f32(order, float(xi), C.byref(l), w)
    return l.value, np.array(w[: order + 1], dtype=dtype)


def boris(kq: float, E, B, u, dtype=np.float64):
    """One Boris rotation u^{n-1/2} -> u^{n+1/2} — oracle step 2c. kq = q*dt/(2m)."""
    E = np.ascontiguousarray(E, dtype=dtype)
    B = np.ascontiguousarray(B, dtype=dtype)
    u = np.array(u, dtype=dtype)
    ct = C.c_double if np.dtype(dtype) == np.float64 else C.c_float
    f = lib().orc_boris_f64 if np.dtype(dtype) == np.float64 else lib().orc_boris_f32
    f(ct(kq), E.ctypes.data_as(C.POINTER(ct)), B.ctypes.data_as(C.POINTER(ct)), u.ctypes.data_as(C.POINTER(ct)))
    return u


def vay(kq: float, E, B, u, dtype=np.float64):
    """One Vay push u^{n-1/2} -> u^{n+1/2} (ref [21]). kq = q*dt/(2m)."""
    E = np.ascontiguousarray(E, dtype=dtype)
    B = np.ascontiguousarray(B, dtype=dtype)
    u = np.array(u, dtype=dtype)
    ct = C.c_double if np.dtype(dtype) == np.float64 else C.c_float
    f = lib().orc_vay_f64 if np.dtype(dtype) == np.float64 else lib().orc_vay_f32
    f(ct(kq), E.ctypes.data_as(C.POINTER(ct)), B.ctypes.data_as(C.POINTER(ct)), u.ctypes.data_as(C.POINTER(ct)))
    return u


PUSHER_BORIS, PUSHER_VAY = 0, 1
SOLVER_YEE, SOLVER_CKC = 0, 1
GATHER_UNIFORM, GATHER_GALERKIN = 0, 1


class Oracle:
    """One oracle simulation. Arrays in and out are numpy, x-fastest fields of shape (nz, ny, nx)."""

    def __init__(self, n_cells, dx, dt, order, dtype=np.float64, periodic=(1, 1, 1), tile=(8, 8, 8),
                 sort_interval=4, sort_key_mode=0, pusher=PUSHER_BORIS, gather_mode=GATHER_UNIFORM,
                 solver=SOLVER_YEE):
        self.dtype = np.dtype(dtype)
        self.n_cells = tuple(int(v) for v in n_cells)
        self.dx = tuple(float(v) for v in dx)
        self.dt = float(dt)
        self.order = int(order)
        tile = tuple(min(int(t), n) for t, n in zip(tile, self.n_cells))
        dxa = (C.c_double * 3)(*self.dx)
        self._h = lib().orc_create_ex(_i32(self.n_cells), dxa, self.dt, self.order,
                                   0 if self.dtype == np.float64 else 1, _i32(periodic), _i32(tile),
                                      int(sort_interval), int(sort_key_mode), int(solver))
        if not self._h:
            raise ValueError("orc_create rejected the arguments (order, tile, dx or CFL)")
        self._fshape = (self.n_cells[2], self.n_cells[1], self.n_cells[0])
        if lib().orc_set_method(self._h, int(pusher), int(gather_mode)) != 0:
            raise ValueError("unknown pusher / gather_mode")

    def ckc_coefficients(self):
        """(alpha[3], beta[3][3], gamma[3]) of the CKC solver for this grid."""
        out = (C.c_double * 15)()
        lib().orc_ckc_coefficients(self._h, out)
        v = np.array(out[:])
        return v[:3], v[3:12].reshape(3, 3), v[12:]

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def add_species(self, x, y, z, ux, uy, uz, w, charge, mass) -> int:
        arrs = [np.ascontiguousarray(a, dtype=self.dtype) for a in (x, y, z, ux, uy, uz, w)]
        return lib().orc_add_species(self._h, len(arrs[0]), *[_ptr(a) for a in arrs], float(charge), float(mass))

    def set_fields(self, E, B):
        E = [np.ascontiguousarray(a, dtype=self.dtype).reshape(self._fshape) for a in E]
        B = [np.ascontiguousarray(a, dtype=self.dtype).reshape(self._fshape) for a in B]
        pe = (C.c_void_p * 3)(*[a.ctypes.data for a in E])
        pb = (C.c_void_p * 3)(*[a.ctypes.data for a in B])
        lib().orc_set_fields(self._h, pe, pb)

    def step(self, n=1):
        lib().orc_step(self._h, int(n))

    def step_omp(self, n=1, threads=0) -> int:
        """The OpenMP variant (the paper's CPU scheme: tiles to threads, private J buffers, one atomic per cell;
        PAPER.md:171-173). Same arithmetic per particle as step(); J sums in another order. Returns the thread
        count used (threads <= 0: all that OpenMP offers)."""
        return lib().orc_step_omp(self._h, int(n), int(threads))

    def sort_now(self):
        lib().orc_sort_now(self._h)

    def field_step(self, n=1):
        lib().orc_field_step(self._h, int(n))

    def particle_step(self):
        lib().orc_particle_step(self._h)

    def get_fields(self):
        out = [[np.empty(self._fshape, dtype=self.dtype) for _ in range(3)] for _ in range(3)]
        ps = [(C.c_void_p * 3)(*[a.ctypes.data for a in grp]) for grp in out]
        lib().orc_get_fields(self._h, ps[0], ps[1], ps[2])
        return out[0], out[1], out[2]

    def num_particles(self, species=0) -> int:
        return lib().orc_num_particles(self._h, species)

    def get_particles(self, species=0):
        n = self.num_particles(species)
        arrs = [np.empty(n, dtype=self.dtype) for _ in range(7)]
        ids = np.empty(n, dtype=np.int64)
        lib().orc_get_particles(self._h, species, *[_ptr(a) for a in arrs], ids.ctypes.data_as(C.POINTER(C.c_int64)))
        return dict(zip(("x", "y", "z", "ux", "uy", "uz", "w"), arrs), id=ids)

    def get_sort_state(self, species=0):
        n = self.num_particles(species)
        cell = np.empty(n, dtype=np.int32)
        perm = np.empty(n, dtype=np.int32)
        rc = lib().orc_get_sort_state(self._h, species, cell.ctypes.data_as(C.POINTER(C.c_int32)),
                                      perm.ctypes.data_as(C.POINTER(C.c_int32)))
        if rc != 0:
            raise RuntimeError("species has not been sorted yet")
        return cell, perm

    def diagnostics(self) -> dict:
        out = (C.c_double * len(DIAG))()
        lib().orc_get_diagnostics(self._h, out)
        return dict(zip(DIAG, out))

    def rho(self):
        r = np.empty(self._fshape, dtype=np.float64)
        lib().orc_get_rho(self._h, r.ctypes.data_as(C.POINTER(C.c_double)))
        return r

    def gather(self, x, y, z):
        x, y, z = [np.ascontiguousarray(a, dtype=self.dtype) for a in (x, y, z)]
        out = np.empty((len(x), 6), dtype=self.dtype)
        lib().orc_gather(self._h, len(x), _ptr(x), _ptr(y), _ptr(z), _ptr(out))
        return out

    def deposit_moves(self, species, x0, x1, w):
        """Zero J, Esirkepov-deposit the moves x0[n,3] -> x1[n,3] (x1 unwrapped); returns (Jx,Jy,Jz)."""
        x0 = np.ascontiguousarray(x0, dtype=self.dtype)
        x1 = np.ascontiguousarray(x1, dtype=self.dtype)
        w = np.ascontiguousarray(w, dtype=self.dtype)
        lib().orc_deposit_moves(self._h, species, len(w), _ptr(x0), _ptr(x1), _ptr(w))
        return self.get_fields()[2]
