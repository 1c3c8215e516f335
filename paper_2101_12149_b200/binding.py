"""ctypes binding of libpic.so (include/pic.h): argument marshalling only — every step of the
path runs in the library's CUDA kernels. Functions carry the C names; `Sim` is a thin object
wrapper over the same calls. Arrays may be numpy (host, PIC_HOST) or torch CUDA tensors
(device, PIC_DEVICE). There is no CPU fallback: a missing or unloadable library raises."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpic.so")

PIC_F64, PIC_F32 = 0, 1
PIC_HOST, PIC_DEVICE = 0, 1
PIC_DEPOSIT_AUTO, PIC_DEPOSIT_GLOBAL, PIC_DEPOSIT_COOP, PIC_DEPOSIT_TILE, PIC_DEPOSIT_TILE_MMA = 0, 1, 2, 3, 4
PIC_DEPOSIT_FUSED = 5
PIC_PUSHER_BORIS, PIC_PUSHER_VAY = 0, 1
PIC_STAGE_AUTO, PIC_STAGE_CP_ASYNC, PIC_STAGE_TMA = 0, 1, 2
PIC_GATHER_UNIFORM, PIC_GATHER_GALERKIN = 0, 1
PIC_SOLVER_YEE, PIC_SOLVER_CKC = 0, 1
PIC_NDIAG = 12
PIC_NPHASE = 5
DIAG_NAMES = ("field_E", "field_B", "kinetic", "charge", "gauss_max", "rho_max", "deactivated", "steps",
              "pool_chunks", "pool_bytes", "launches", "step_launches")
PHASE_NAMES = ("sort", "push", "deposit", "stray", "fields")
ERRORS = {-1: "PIC_ERR_INVALID_ARG", -2: "PIC_ERR_CFL", -3: "PIC_ERR_OUT_OF_DOMAIN", -4: "PIC_ERR_OOM",
          -5: "PIC_ERR_CUDA", -6: "PIC_ERR_CAPACITY"}

# every symbol include/pic.h declares (tests check that the library exports each of them)
SYMBOLS = (
    "pic_default_options", "pic_create", "pic_add_species", "pic_set_fields", "pic_step", "pic_synchronize",
    "pic_get_fields", "pic_get_particles", "pic_get_sort_state", "pic_sort_now", "pic_get_diagnostics",
    "pic_get_rho", "pic_enable_phase_timing", "pic_get_phase_times", "pic_num_particles", "pic_num_species",
    "pic_last_error", "pic_ckc_coefficients", "pic_probe_peaks", "pic_destroy", "pic_sort_permutation_noalloc",
)
PIC_NOALLOC_MAX_PARTICLES = 524288


class PicError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("%s (%d): %s" % (ERRORS.get(code, "PIC_ERR"), code, msg))
        self.code = code


class pic_options(C.Structure):
    _fields_ = [("periodic", C.c_int32 * 3), ("tile", C.c_int32 * 3), ("sort_interval", C.c_int32),
                ("sort_key_mode", C.c_int32), ("deposit_mode", C.c_int32), ("pusher", C.c_int32),
                ("gather_mode", C.c_int32), ("solver", C.c_int32),
                ("deterministic", C.c_int32), ("cuda_graph", C.c_int32), ("box_staging", C.c_int32),
                ("cuda_stream", C.c_void_p)]


_lib = None


def lib():
    """The loaded library; raises if it has not been built (python -m paper_2101_12149_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libpic.so is missing: build it with `python -m paper_2101_12149_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, vpp = C.c_void_p, C.POINTER(C.c_void_p)
        i32p, i64p, dp = C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_double)
        L.pic_default_options.argtypes = [C.POINTER(pic_options)]
        L.pic_default_options.restype = None
        L.pic_create.argtypes = [i32p, dp, C.c_double, C.c_int, C.c_int, C.POINTER(pic_options), vpp]
        L.pic_add_species.argtypes = [vp, C.c_int64] + [vp] * 7 + [C.c_double, C.c_double, C.c_int, i32p]
        L.pic_set_fields.argtypes = [vp, vpp, vpp, C.c_int]
        L.pic_step.argtypes = [vp, C.c_int32]
        L.pic_synchronize.argtypes = [vp]
        L.pic_get_fields.argtypes = [vp, vpp, vpp, vpp, C.c_int]
        L.pic_get_particles.argtypes = [vp, C.c_int32, C.c_int64] + [vp] * 7 + [vp, i64p, C.c_int]
        L.pic_get_sort_state.argtypes = [vp, C.c_int32, vp, vp, C.c_int]
        L.pic_sort_now.argtypes = [vp]
        L.pic_get_diagnostics.argtypes = [vp, dp]
        L.pic_get_rho.argtypes = [vp, vp, C.c_int]
        L.pic_enable_phase_timing.argtypes = [vp, C.c_int32]
        L.pic_get_phase_times.argtypes = [vp, C.POINTER(C.c_float), i64p, C.c_int32]
        L.pic_num_particles.argtypes = [vp, C.c_int32]
        L.pic_num_particles.restype = C.c_int64
        L.pic_num_species.argtypes = [vp]
        L.pic_num_species.restype = C.c_int32
        L.pic_last_error.argtypes = [vp]
        L.pic_last_error.restype = C.c_char_p
        L.pic_ckc_coefficients.argtypes = [dp, dp, dp, dp]
        L.pic_probe_peaks.argtypes = [vp, C.c_double, dp]
        L.pic_destroy.argtypes = [vp]
        L.pic_destroy.restype = None
        L.pic_sort_permutation_noalloc.argtypes = [i32p, dp, i32p, C.c_int32, C.c_int, vp, vp, vp, C.c_int64, vp, vp, vp]
        _lib = L
    return _lib


def _is_torch(a):
    return type(a).__module__.startswith("torch")


def _where(arrs):
    kinds = {(_is_torch(a) and a.is_cuda) for a in arrs if a is not None}
    if len(kinds) > 1:
        raise ValueError("mix of host and device arrays in one call")
    return PIC_DEVICE if kinds == {True} else PIC_HOST


def _addr(a, np_dtype, n=None):
    """Pointer of a contiguous array of the right dtype (no copies, no conversion)."""
    if a is None:
        return None
    if _is_torch(a):
        import torch
        want = {np.dtype(np.float64): torch.float64, np.dtype(np.float32): torch.float32,
                np.dtype(np.int64): torch.int64, np.dtype(np.int32): torch.int32}[np.dtype(np_dtype)]
        if a.dtype != want or not a.is_contiguous():
            raise TypeError("tensor must be contiguous %s" % want)
        if n is not None and a.numel() < n:
            raise ValueError("tensor too small")
        return a.data_ptr()
    if not isinstance(a, np.ndarray) or a.dtype != np.dtype(np_dtype) or not a.flags.c_contiguous:
        raise TypeError("array must be a C-contiguous numpy array of dtype %s" % np.dtype(np_dtype))
    if n is not None and a.size < n:
        raise ValueError("array too small")
    return a.ctypes.data


def _check(h, rc):
    if rc != 0:
        raise PicError(rc, (lib().pic_last_error(h) or b"").decode())


# ----------------------------------------------------------------------------- C-named calls
def pic_default_options() -> pic_options:
    o = pic_options()
    lib().pic_default_options(C.byref(o))
    return o


def pic_create(n_cells, dx, dt, shape_order, precision, options: pic_options | None = None):
    h = C.c_void_p()
    n = (C.c_int32 * 3)(*[int(v) for v in n_cells])
    d = (C.c_double * 3)(*[float(v) for v in dx])
    rc = lib().pic_create(n, d, float(dt), int(shape_order), int(precision),
                          C.byref(options) if options is not None else None, C.byref(h))
    _check(None, rc)
    return h


def pic_add_species(h, x, y, z, ux, uy, uz, w, charge, mass, np_dtype) -> int:
    arrs = (x, y, z, ux, uy, uz, w)
    n = int(arrs[0].numel() if _is_torch(arrs[0]) else arrs[0].size)
    sid = C.c_int32(-1)
    rc = lib().pic_add_species(h, n, *[_addr(a, np_dtype, n) for a in arrs], float(charge), float(mass),
                               _where(arrs), C.byref(sid))
    _check(h, rc)
    return sid.value


def pic_set_fields(h, E, B, np_dtype, n_valid):
    pe = (C.c_void_p * 3)(*[_addr(a, np_dtype, n_valid) for a in E])
    pb = (C.c_void_p * 3)(*[_addr(a, np_dtype, n_valid) for a in B])
    _check(h, lib().pic_set_fields(h, pe, pb, _where(list(E) + list(B))))


def pic_step(h, n=1):
    _check(h, lib().pic_step(h, int(n)))


def pic_synchronize(h):
    _check(h, lib().pic_synchronize(h))


def pic_get_fields(h, E, B, J, np_dtype, n_valid):
    def pack(g):
        return None if g is None else (C.c_void_p * 3)(*[_addr(a, np_dtype, n_valid) for a in g])
    allarr = [a for g in (E, B, J) if g is not None for a in g]
    _check(h, lib().pic_get_fields(h, pack(E), pack(B), pack(J), _where(allarr)))


def pic_get_particles(h, species, capacity, x, y, z, ux, uy, uz, w, ids, np_dtype) -> int:
    arrs = (x, y, z, ux, uy, uz, w)
    n_out = C.c_int64(0)
    rc = lib().pic_get_particles(h, int(species), int(capacity), *[_addr(a, np_dtype) for a in arrs],
                                 _addr(ids, np.int64), C.byref(n_out), _where(list(arrs) + [ids]))
    _check(h, rc)
    return n_out.value


def pic_get_sort_state(h, species, cell, perm):
    _check(h, lib().pic_get_sort_state(h, int(species), _addr(cell, np.int32), _addr(perm, np.int32),
                                       _where([cell, perm])))


def pic_sort_now(h):
    _check(h, lib().pic_sort_now(h))


def pic_get_diagnostics(h) -> dict:
    out = (C.c_double * PIC_NDIAG)()
    _check(h, lib().pic_get_diagnostics(h, out))
    return dict(zip(DIAG_NAMES, out))


def pic_get_rho(h, rho):
    _check(h, lib().pic_get_rho(h, _addr(rho, np.float64), _where([rho])))


def pic_enable_phase_timing(h, on=True):
    _check(h, lib().pic_enable_phase_timing(h, 1 if on else 0))


def pic_get_phase_times(h, reset=True) -> dict:
    """{class: (elapsed ms, spans)} since the last reset."""
    ms = (C.c_float * PIC_NPHASE)()
    cnt = (C.c_int64 * PIC_NPHASE)()
    _check(h, lib().pic_get_phase_times(h, ms, cnt, 1 if reset else 0))
    return {k: (float(m), int(c)) for k, m, c in zip(PHASE_NAMES, ms, cnt)}


def pic_num_particles(h, species=0) -> int:
    return lib().pic_num_particles(h, int(species))


def pic_num_species(h) -> int:
    return lib().pic_num_species(h)


def pic_ckc_coefficients(dx):
    """(alpha[3], beta[3][3], gamma[3]) of the CKC solver for cells of size dx (host arithmetic only)."""
    al, be, ga = (C.c_double * 3)(), (C.c_double * 9)(), (C.c_double * 3)()
    rc = lib().pic_ckc_coefficients((C.c_double * 3)(*[float(v) for v in dx]), al, be, ga)
    if rc != 0:
        raise PicError(rc, "dx must be positive and finite")
    return np.array(al[:]), np.array(be[:]).reshape(3, 3), np.array(ga[:])


def pic_sort_permutation_noalloc(n_cells, dx, tile, x, y, z, cell, perm, sort_key_mode=0, stream=None):
    """Allocation-free sort (include/pic.h): x, y, z are device arrays of one dtype (float64 / float32), cell and perm
    int32 device arrays of the same length; asynchronous on `stream`."""
    n = _n_elems(x)
    dt = np.float64 if _elem_size(x) == 8 else np.float32
    rc = lib().pic_sort_permutation_noalloc(
        (C.c_int32 * 3)(*[int(v) for v in n_cells]), (C.c_double * 3)(*[float(v) for v in dx]),
        (C.c_int32 * 3)(*[int(v) for v in tile]), int(sort_key_mode), PIC_F64 if dt == np.float64 else PIC_F32,
        _dev_ptr(x), _dev_ptr(y), _dev_ptr(z), n, _dev_ptr(cell), _dev_ptr(perm), stream)
    _check(None, rc)


def _dev_ptr(t):
    return int(t.data_ptr()) if hasattr(t, "data_ptr") else int(t)


def _n_elems(t):
    return int(t.numel())


def _elem_size(t):
    return int(t.element_size())


PROBE_NAMES = ("fp64_fma_tflops", "fp64_mma_tflops", "smem_tbs", "fp32_fma_tflops", "sm_count", "sm_clock_mhz")


def pic_probe_peaks(stream=None, seconds_per_probe=0.2) -> dict:
    """Measured on-chip ceilings of the current device (see include/pic.h)."""
    out = (C.c_double * len(PROBE_NAMES))()
    rc = lib().pic_probe_peaks(stream, float(seconds_per_probe), out)
    if rc != 0:
        raise PicError(rc, "pic_probe_peaks failed (no CUDA device?)")
    return dict(zip(PROBE_NAMES, out))


def pic_destroy(h):
    lib().pic_destroy(h)


# ----------------------------------------------------------------------------- object wrapper
class Sim:
    """One simulation handle. Field arrays are shaped (nz, ny, nx) (x fastest)."""

    def __init__(self, n_cells, dx, dt, order, dtype=np.float64, periodic=(1, 1, 1), tile=(8, 8, 8),
                 sort_interval=4, sort_key_mode=0, deposit_mode=PIC_DEPOSIT_AUTO, stream=None,
                 pusher=PIC_PUSHER_BORIS, gather_mode=PIC_GATHER_UNIFORM, solver=PIC_SOLVER_YEE, deterministic=False, cuda_graph=True, box_staging=0):
        self.dtype = np.dtype(dtype)
        self.n_cells = tuple(int(v) for v in n_cells)
        self.n_valid = self.n_cells[0] * self.n_cells[1] * self.n_cells[2]
        self.fshape = (self.n_cells[2], self.n_cells[1], self.n_cells[0])
        o = pic_default_options()
        for d in range(3):
            o.periodic[d] = int(periodic[d])
            o.tile[d] = int(tile[d])
        o.sort_interval = int(sort_interval)
        o.sort_key_mode = int(sort_key_mode)
        o.deposit_mode = int(deposit_mode)
        o.pusher = int(pusher)
        o.gather_mode = int(gather_mode)
        o.solver = int(solver)
        o.deterministic = 1 if deterministic else 0
        o.cuda_graph = 1 if cuda_graph else 0
        o.box_staging = int(box_staging)
        o.cuda_stream = stream
        self._h = pic_create(self.n_cells, dx, dt, order, PIC_F64 if self.dtype == np.float64 else PIC_F32, o)

    def close(self):
        if getattr(self, "_h", None):
            pic_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _host(self, a):
        return a if _is_torch(a) else np.ascontiguousarray(a, dtype=self.dtype)

    def add_species(self, x, y, z, ux, uy, uz, w, charge, mass) -> int:
        arrs = [self._host(a) for a in (x, y, z, ux, uy, uz, w)]
        return pic_add_species(self._h, *arrs, charge, mass, self.dtype)

    def set_fields(self, E, B):
        pic_set_fields(self._h, [self._host(a) for a in E], [self._host(a) for a in B], self.dtype, self.n_valid)

    def step(self, n=1):
        pic_step(self._h, n)

    def synchronize(self):
        pic_synchronize(self._h)

    def sort_now(self):
        pic_sort_now(self._h)

    def get_fields(self, with_J=True):
        mk = lambda: [np.empty(self.fshape, dtype=self.dtype) for _ in range(3)]
        E, B, J = mk(), mk(), (mk() if with_J else None)
        pic_get_fields(self._h, E, B, J, self.dtype, self.n_valid)
        return E, B, J

    def num_particles(self, species=0) -> int:
        return pic_num_particles(self._h, species)

    def get_particles(self, species=0):
        n = self.num_particles(species)
        arrs = [np.empty(n, dtype=self.dtype) for _ in range(7)]
        ids = np.empty(n, dtype=np.int64)
        pic_get_particles(self._h, species, n, *arrs, ids, self.dtype)
        return dict(zip(("x", "y", "z", "ux", "uy", "uz", "w"), arrs), id=ids)

    def get_sort_state(self, species=0):
        n = self.num_particles(species)
        cell = np.empty(n, dtype=np.int32)
        perm = np.empty(n, dtype=np.int32)
        pic_get_sort_state(self._h, species, cell, perm)
        return cell, perm

    def diagnostics(self) -> dict:
        return pic_get_diagnostics(self._h)

    def rho(self):
        r = np.empty(self.fshape, dtype=np.float64)
        pic_get_rho(self._h, r)
        return r

    def enable_phase_timing(self, on=True):
        pic_enable_phase_timing(self._h, on)

    def phase_times(self, reset=True) -> dict:
        return pic_get_phase_times(self._h, reset)
