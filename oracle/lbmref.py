"""ctypes binding of oracle/liblbmref.so (CPU oracle; test infrastructure, not the product).

Arrays are numpy float64 / uint8 indexed [z, y, x]; populations [19, z, y, x] in the direction
order of `lattice()`.
"""
import ctypes as C

import numpy as np

from . import build as _build


class _Params(C.Structure):
    _fields_ = [("G", C.c_double), ("tau", C.c_double * 2), ("xi", C.c_double),
                ("accel", C.c_double * 3), ("z_open", C.c_int), ("inlet_kind", C.c_int),
                ("inlet_comp", C.c_int), ("inlet_rho", C.c_double), ("inlet_uz", C.c_double),
                ("outlet_kind", C.c_int), ("outlet_comp", C.c_int), ("outlet_rho", C.c_double),
                ("storage_bits", C.c_int), ("half_force", C.c_int)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        P, D, I = C.c_void_p, C.POINTER(C.c_double), C.c_int
        lib.lbmref_create.argtypes = [C.POINTER(P), C.c_void_p, I, I, I, C.POINTER(_Params)]
        lib.lbmref_destroy.argtypes = [P]
        lib.lbmref_destroy.restype = None
        lib.lbmref_set_density.argtypes = [P, C.c_void_p, C.c_void_p]
        lib.lbmref_set_populations.argtypes = [P, I, C.c_void_p]
        lib.lbmref_get_populations.argtypes = [P, I, C.c_void_p]
        lib.lbmref_step.argtypes = [P, I]
        lib.lbmref_get_macroscopic.argtypes = [P] + [C.c_void_p] * 6
        lib.lbmref_diagnostics.argtypes = [P, D, D]
        lib.lbmref_saturation.argtypes = [P, I, I, I, D]
        lib.lbmref_trapped_volume.argtypes = [P, I, I, I, C.POINTER(C.c_longlong), D]
        lib.lbmref_num_fluid.argtypes = [P]
        lib.lbmref_set_boundary.argtypes = [P, C.c_double, C.c_double]
        lib.lbmref_num_fluid.restype = C.c_longlong
        lib.lbmref_lattice.argtypes = [D, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        lib.lbmref_lattice.restype = None
        _lib = lib
    return _lib


def _params(p):
    s = _Params()
    s.G = p["G"]
    s.tau[0], s.tau[1] = p["tau"]
    s.xi = p["xi"]
    for a in range(3):
        s.accel[a] = p["accel"][a]
    for k in ("z_open", "inlet_kind", "inlet_comp", "outlet_kind", "outlet_comp",
              "storage_bits", "half_force"):
        setattr(s, k, int(p[k]))
    for k in ("inlet_rho", "inlet_uz", "outlet_rho"):
        setattr(s, k, float(p[k]))
    return s


def lattice():
    lib = _load()
    w = (C.c_double * 19)()
    e = (C.c_int * 57)()
    o = (C.c_int * 19)()
    lib.lbmref_lattice(w, e, o)
    return np.array(w), np.array(e).reshape(19, 3), np.array(o)


def threads():
    return int(_load().lbmref_threads())


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"{what} failed with code {rc}")


class LbmRef:
    def __init__(self, mask, params):
        lib = _load()
        mask = np.ascontiguousarray(mask, np.uint8)
        assert mask.ndim == 3
        self.shape = mask.shape
        nz, ny, nx = mask.shape
        self._h = C.c_void_p()
        _chk(lib.lbmref_create(C.byref(self._h), mask.ctypes.data, nx, ny, nz,
                               C.byref(_params(params))), "lbmref_create")
        self.num_fluid = int(lib.lbmref_num_fluid(self._h))

    def close(self):
        if getattr(self, "_h", None):
            _load().lbmref_destroy(self._h)
            self._h = None

    __del__ = close

    def set_density(self, rhoA, rhoB):
        a = np.ascontiguousarray(rhoA, np.float64)
        b = np.ascontiguousarray(rhoB, np.float64)
        assert a.shape == self.shape and b.shape == self.shape
        _chk(_load().lbmref_set_density(self._h, a.ctypes.data, b.ctypes.data), "set_density")

    def set_populations(self, comp, f):
        f = np.ascontiguousarray(f, np.float64)
        assert f.shape == (19,) + self.shape
        _chk(_load().lbmref_set_populations(self._h, comp, f.ctypes.data), "set_populations")

    def get_populations(self, comp):
        f = np.empty((19,) + self.shape, np.float64)
        _chk(_load().lbmref_get_populations(self._h, comp, f.ctypes.data), "get_populations")
        return f

    def step(self, n=1):
        _chk(_load().lbmref_step(self._h, int(n)), "step")

    def set_boundary(self, inlet_value, outlet_rho):
        _chk(_load().lbmref_set_boundary(self._h, float(inlet_value), float(outlet_rho)),
             "set_boundary")

    def get_macroscopic(self):
        out = [np.empty(self.shape, np.float64) for _ in range(6)]
        _chk(_load().lbmref_get_macroscopic(self._h, *[o.ctypes.data for o in out]),
             "get_macroscopic")
        return dict(zip(("rhoA", "rhoB", "ux", "uy", "uz", "P"), out))

    def diagnostics(self):
        m = (C.c_double * 2)()
        j = (C.c_double * 3)()
        _chk(_load().lbmref_diagnostics(self._h, m, j), "diagnostics")
        return np.array(m), np.array(j)

    def saturation(self, comp, z0=0, z1=None):
        z1 = self.shape[0] if z1 is None else z1
        s = C.c_double()
        _chk(_load().lbmref_saturation(self._h, comp, z0, z1, C.byref(s)), "saturation")
        return s.value

    def trapped_volume(self, comp, z0=0, z1=None):
        z1 = self.shape[0] if z1 is None else z1
        n = C.c_longlong()
        m = C.c_double()
        _chk(_load().lbmref_trapped_volume(self._h, comp, z0, z1, C.byref(n), C.byref(m)),
             "trapped_volume")
        return n.value, m.value
