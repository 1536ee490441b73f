"""Thin ctypes binding of include/lbm.h (argument marshalling only: every step of the path runs
in the CUDA kernels of liblbm_b200.so).  Same names as the C ABI.

Arrays are numpy, indexed [z, y, x] (x fastest, i.e. idx = x + nx*(y + ny*z)); populations are
[19, z, y, x] float64 in the canonical D3Q19 order of include/lbm.h.

There is no CPU fallback: if the shared library is missing it is built with nvcc, and if that
fails, or no CUDA device is present at lbm_create time, an exception is raised.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

LBM_OK, LBM_EINVAL, LBM_ENOFLUID, LBM_ESOLIDOPEN, LBM_ENOMEM, LBM_ECUDA, LBM_ENONFINITE = (
    0, -1, -2, -3, -4, -5, -6)

SYMBOLS = [
    "lbm_create", "lbm_destroy", "lbm_set_density", "lbm_set_populations", "lbm_get_populations",
    "lbm_set_boundary", "lbm_step", "lbm_sync", "lbm_get_macroscopic", "lbm_diagnostics",
    "lbm_saturation", "lbm_trapped_volume", "lbm_trapped_volume_static", "lbm_mean_pressure", "lbm_num_fluid", "lbm_num_wall_solid",
    "lbm_memory_bytes", "lbm_set_profiling", "lbm_last_step_profile", "lbm_last_error",
    "lbm_build_index",
    "lbm_options_default", "lbm_create_opt", "lbm_create_slab_opt", "lbm_step_info",
    "lbm_create_slab", "lbm_slab_density", "lbm_slab_collide", "lbm_slab_unpack", "lbm_slab_buffer",
    "lbm_num_owned", "lbm_build_slab_halo",
    "lbm_comm_unique_id", "lbm_slab_comm_init", "lbm_slab_step", "lbm_slab_exchange",
    "lbm_slab_ccl_begin", "lbm_slab_ccl_export", "lbm_slab_ccl_import", "lbm_slab_ccl_finish",
]


class LbmError(RuntimeError):
    def __init__(self, code, what, msg):
        super().__init__(f"{what} failed with code {code}: {msg}")
        self.code = code


class lbm_params(C.Structure):
    _fields_ = [("G", C.c_double), ("tau", C.c_double * 2), ("xi", C.c_double),
                ("accel", C.c_double * 3), ("z_open", C.c_int), ("inlet_kind", C.c_int),
                ("inlet_comp", C.c_int), ("inlet_rho", C.c_double), ("inlet_uz", C.c_double),
                ("outlet_kind", C.c_int), ("outlet_comp", C.c_int), ("outlet_rho", C.c_double),
                ("storage_bits", C.c_int), ("half_force", C.c_int)]


class lbm_options(C.Structure):
    _fields_ = [("graph", C.c_int), ("pdl", C.c_int), ("reverse", C.c_int),
                ("keep_psi_mb", C.c_int)]


_lib = None


def library_path():
    return _build.LIB


def load():
    """Load (building if needed) liblbm_b200.so and declare the prototypes of include/lbm.h."""
    global _lib
    if _lib is not None:
        return _lib
    import torch  # noqa: F401  -- makes libc10/libc10_cuda/libcudart resolvable before dlopen
    path = _build.build()
    if not os.path.exists(path):
        raise RuntimeError("liblbm_b200.so is missing and could not be built; no CPU fallback")
    lib = C.CDLL(path)
    P, D, I, V = C.c_void_p, C.POINTER(C.c_double), C.c_int, C.c_void_p
    LL = C.c_longlong
    lib.lbm_create.argtypes = [C.POINTER(P), V, I, I, I, C.POINTER(lbm_params)]
    lib.lbm_destroy.argtypes = [P]
    lib.lbm_destroy.restype = None
    lib.lbm_set_density.argtypes = [P, V, V]
    lib.lbm_set_populations.argtypes = [P, I, V]
    lib.lbm_get_populations.argtypes = [P, I, V]
    lib.lbm_set_boundary.argtypes = [P, C.c_double, C.c_double]
    lib.lbm_step.argtypes = [P, I]
    lib.lbm_sync.argtypes = [P]
    lib.lbm_get_macroscopic.argtypes = [P] + [V] * 6
    lib.lbm_diagnostics.argtypes = [P, D, D]
    lib.lbm_saturation.argtypes = [P, I, I, I, D]
    lib.lbm_trapped_volume.argtypes = [P, I, I, I, C.POINTER(LL), D]
    lib.lbm_trapped_volume_static.argtypes = [P, I, I, I, C.POINTER(LL), D]
    lib.lbm_trapped_volume_static.restype = I
    lib.lbm_mean_pressure.argtypes = [P, I, I, D]
    lib.lbm_num_fluid.argtypes = [P]
    lib.lbm_num_fluid.restype = LL
    lib.lbm_num_wall_solid.argtypes = [P]
    lib.lbm_num_wall_solid.restype = LL
    lib.lbm_memory_bytes.argtypes = [P, C.POINTER(LL)]
    lib.lbm_set_profiling.argtypes = [P, I]
    lib.lbm_last_step_profile.argtypes = [P, D, C.POINTER(LL)]
    lib.lbm_last_error.argtypes = []
    lib.lbm_last_error.restype = C.c_char_p
    lib.lbm_build_index.argtypes = [V, I, I, I, I, V, V, LL, C.POINTER(LL), C.POINTER(LL)]
    lib.lbm_options_default.argtypes = [C.POINTER(lbm_options)]
    lib.lbm_options_default.restype = None
    lib.lbm_create_opt.argtypes = [C.POINTER(P), V, I, I, I, C.POINTER(lbm_params),
                                   C.POINTER(lbm_options)]
    lib.lbm_create_slab_opt.argtypes = [C.POINTER(P), V, I, I, I, C.POINTER(lbm_params),
                                        C.POINTER(lbm_options), I, I]
    lib.lbm_step_info.argtypes = [P, C.POINTER(I)]
    lib.lbm_create_slab.argtypes = [C.POINTER(P), V, I, I, I, C.POINTER(lbm_params), I, I]
    lib.lbm_slab_density.argtypes = [P, I]
    lib.lbm_slab_collide.argtypes = [P, I]
    lib.lbm_slab_unpack.argtypes = [P]
    lib.lbm_slab_buffer.argtypes = [P, I, C.POINTER(C.c_void_p), C.POINTER(LL)]
    lib.lbm_num_owned.argtypes = [P]
    lib.lbm_num_owned.restype = LL
    lib.lbm_build_slab_halo.argtypes = [V, I, I, I, I, I, I, V, V, LL] + [C.POINTER(LL)] * 5
    lib.lbm_comm_unique_id.argtypes = [C.c_char_p]
    lib.lbm_slab_comm_init.argtypes = [P, C.c_char_p, I, I]
    lib.lbm_slab_step.argtypes = [P, I]
    lib.lbm_slab_exchange.argtypes = [P, I]
    for fn in ("lbm_comm_unique_id", "lbm_slab_comm_init", "lbm_slab_step", "lbm_slab_exchange"):
        getattr(lib, fn).restype = I
    lib.lbm_slab_ccl_begin.argtypes = [P, I, I, I]
    lib.lbm_slab_ccl_export.argtypes = [P]
    lib.lbm_slab_ccl_import.argtypes = [P, I, I, C.POINTER(I)]
    lib.lbm_slab_ccl_finish.argtypes = [P, I, I, C.POINTER(LL), D]
    for fn in ("lbm_slab_ccl_begin", "lbm_slab_ccl_export", "lbm_slab_ccl_import",
               "lbm_slab_ccl_finish"):
        getattr(lib, fn).restype = I
    for fn in ("lbm_create_slab", "lbm_slab_density", "lbm_slab_collide", "lbm_slab_unpack",
               "lbm_slab_buffer", "lbm_build_slab_halo"):
        getattr(lib, fn).restype = I
    for fn in ("lbm_create", "lbm_set_density", "lbm_set_populations", "lbm_get_populations",
               "lbm_set_boundary", "lbm_step", "lbm_sync", "lbm_get_macroscopic",
               "lbm_diagnostics", "lbm_saturation", "lbm_trapped_volume", "lbm_mean_pressure",
               "lbm_memory_bytes",
               "lbm_set_profiling", "lbm_last_step_profile", "lbm_build_index",
               "lbm_create_opt", "lbm_create_slab_opt", "lbm_step_info"):
        getattr(lib, fn).restype = I
    _lib = lib
    return lib


def make_params(p):
    """dict (workloads.default_params layout) -> lbm_params"""
    s = lbm_params()
    s.G = float(p["G"])
    s.tau[0], s.tau[1] = float(p["tau"][0]), float(p["tau"][1])
    s.xi = float(p["xi"])
    for a in range(3):
        s.accel[a] = float(p["accel"][a])
    for k in ("z_open", "inlet_kind", "inlet_comp", "outlet_kind", "outlet_comp", "storage_bits",
              "half_force"):
        setattr(s, k, int(p[k]))
    for k in ("inlet_rho", "inlet_uz", "outlet_rho"):
        setattr(s, k, float(p[k]))
    return s


def make_options(o=None):
    """dict -> lbm_options: the library's defaults (lbm_options_default) with the given fields
    replaced."""
    s = lbm_options()
    load().lbm_options_default(C.byref(s))
    for k, v in (o or {}).items():
        if k not in dict(lbm_options._fields_):
            raise KeyError(f"unknown option {k!r}")
        setattr(s, k, int(v))
    return s


def _chk(rc, what):
    if rc != 0:
        raise LbmError(rc, what, (load().lbm_last_error() or b"").decode())


def lbm_build_index(mask, z_open=0, with_nbr=True):
    """Host-only: the compact index lbm_create builds (no GPU needed). Returns
    (vox2id[z,y,x] int32, nbr[18, N_f] int32 or None, N_f, N_w)."""
    lib = load()
    mask = np.ascontiguousarray(mask, np.uint8)
    nz, ny, nx = mask.shape
    vox2id = np.empty(mask.shape, np.int32)
    nf, nw = C.c_longlong(), C.c_longlong()
    nfluid = int((mask == 0).sum())
    nbr = np.empty((18, max(nfluid, 1)), np.int32) if with_nbr else None
    _chk(lib.lbm_build_index(mask.ctypes.data, nx, ny, nz, int(z_open), vox2id.ctypes.data,
                             nbr.ctypes.data if with_nbr else None, 18 * max(nfluid, 1),
                             C.byref(nf), C.byref(nw)), "lbm_build_index")
    return vox2id, (nbr[:, :nf.value] if with_nbr else None), nf.value, nw.value


LBM_COMM_ID_BYTES = 128


def lbm_comm_unique_id():
    """Rendezvous token of a slab ring (made on one rank, to be handed to every rank)."""
    buf = C.create_string_buffer(LBM_COMM_ID_BYTES)
    _chk(load().lbm_comm_unique_id(buf), "lbm_comm_unique_id")
    return buf.raw


def lbm_build_slab_halo(mask_local, z_open=0, halo=(1, 1)):
    """Host-only: the halo lists lbm_create_slab builds for a local mask [owned + halo planes, y, x];
    halo = (low, high): 1 = that end is a cut with 2 halo planes, 0 = the open box's own end.
    Returns a dict: pack / unpack = per face (low, high) an int32 array [n, 2] of (direction,
    local voxel index); psi_send / psi_recv = fluid nodes per face; n_owned."""
    lib = load()
    mask_local = np.ascontiguousarray(mask_local, np.uint8)
    nz, ny, nx = mask_local.shape
    cap = 2 * 5 * nx * ny
    pk = np.zeros((cap, 2), np.int32)
    up = np.zeros((cap, 2), np.int32)
    arr = lambda: (C.c_longlong * 2)()
    n_pack, n_unpack, ps, pr = arr(), arr(), arr(), arr()
    n_owned = C.c_longlong()
    _chk(lib.lbm_build_slab_halo(mask_local.ctypes.data, nx, ny, nz, int(z_open), int(halo[0]),
                                 int(halo[1]), pk.ctypes.data,
                                 up.ctypes.data, cap, n_pack, n_unpack, ps, pr,
                                 C.byref(n_owned)), "lbm_build_slab_halo")
    return {"pack": (pk[:n_pack[0]].copy(), pk[n_pack[0]:n_pack[0] + n_pack[1]].copy()),
            "unpack": (up[:n_unpack[0]].copy(), up[n_unpack[0]:n_unpack[0] + n_unpack[1]].copy()),
            "psi_send": (int(ps[0]), int(ps[1])), "psi_recv": (int(pr[0]), int(pr[1])),
            "n_owned": int(n_owned.value)}


class Lbm:
    """One simulation on the current CUDA device. Methods mirror the C ABI one to one.
    slab=True: a z-slab context (lbm_create_slab; mask = owned planes + 2 halo planes per cut
    end; halo = (low, high) flags, 0 only at the ends of a z-open box)."""

    def __init__(self, mask, params, slab=False, halo=(1, 1), options=None):
        lib = load()
        import torch
        if torch.cuda.is_available():
            torch.cuda.init()
            torch.empty(1, device="cuda")  # initialises torch's caching allocator and stream
        mask = np.ascontiguousarray(mask, np.uint8)
        if mask.ndim != 3:
            raise ValueError("mask must be [z, y, x]")
        self.shape = mask.shape
        nz, ny, nx = mask.shape
        self.params = dict(params)
        self._h = C.c_void_p()
        ps = make_params(params)
        self.slab = bool(slab)
        if options is None:
            if slab:
                _chk(lib.lbm_create_slab(C.byref(self._h), mask.ctypes.data, nx, ny, nz,
                                         C.byref(ps), int(halo[0]), int(halo[1])),
                     "lbm_create_slab")
            else:
                _chk(lib.lbm_create(C.byref(self._h), mask.ctypes.data, nx, ny, nz, C.byref(ps)),
                     "lbm_create")
        else:
            po = make_options(options)
            if slab:
                _chk(lib.lbm_create_slab_opt(C.byref(self._h), mask.ctypes.data, nx, ny, nz,
                                             C.byref(ps), C.byref(po), int(halo[0]),
                                             int(halo[1])), "lbm_create_slab_opt")
            else:
                _chk(lib.lbm_create_opt(C.byref(self._h), mask.ctypes.data, nx, ny, nz,
                                        C.byref(ps), C.byref(po)), "lbm_create_opt")
        self.num_owned = int(lib.lbm_num_owned(self._h))
        self.num_fluid = int(lib.lbm_num_fluid(self._h))
        self.num_wall_solid = int(lib.lbm_num_wall_solid(self._h))

    def close(self):
        if getattr(self, "_h", None):
            load().lbm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dense(self, a):
        a = np.ascontiguousarray(a, np.float64)
        if a.shape != self.shape:
            raise ValueError(f"expected shape {self.shape}, got {a.shape}")
        return a

    def set_density(self, rhoA, rhoB):
        a, b = self._dense(rhoA), self._dense(rhoB)
        _chk(load().lbm_set_density(self._h, a.ctypes.data, b.ctypes.data), "lbm_set_density")

    def set_populations(self, comp, f):
        f = np.ascontiguousarray(f, np.float64)
        if f.shape != (19,) + self.shape:
            raise ValueError("populations must be [19, z, y, x]")
        _chk(load().lbm_set_populations(self._h, int(comp), f.ctypes.data), "lbm_set_populations")

    def get_populations(self, comp):
        f = np.empty((19,) + self.shape, np.float64)
        _chk(load().lbm_get_populations(self._h, int(comp), f.ctypes.data), "lbm_get_populations")
        return f

    def set_boundary(self, inlet_value, outlet_rho):
        _chk(load().lbm_set_boundary(self._h, float(inlet_value), float(outlet_rho)),
             "lbm_set_boundary")

    def step(self, n=1):
        _chk(load().lbm_step(self._h, int(n)), "lbm_step")

    def slab_density(self, part):
        _chk(load().lbm_slab_density(self._h, int(part)), "lbm_slab_density")

    def slab_collide(self, part):
        _chk(load().lbm_slab_collide(self._h, int(part)), "lbm_slab_collide")

    def slab_unpack(self):
        _chk(load().lbm_slab_unpack(self._h), "lbm_slab_unpack")

    def slab_comm_init(self, comm_id, rank, world):
        if len(comm_id) != LBM_COMM_ID_BYTES:
            raise ValueError("comm_id must be the 128 bytes lbm_comm_unique_id returned")
        _chk(load().lbm_slab_comm_init(self._h, bytes(comm_id), int(rank), int(world)),
             "lbm_slab_comm_init")

    def slab_step(self, n=1):
        _chk(load().lbm_slab_step(self._h, int(n)), "lbm_slab_step")

    def slab_exchange(self, kind):
        _chk(load().lbm_slab_exchange(self._h, int(kind)), "lbm_slab_exchange")

    def slab_ccl_begin(self, comp, mark_lo, mark_hi):
        _chk(load().lbm_slab_ccl_begin(self._h, int(comp), int(bool(mark_lo)), int(bool(mark_hi))),
             "lbm_slab_ccl_begin")

    def slab_ccl_export(self):
        _chk(load().lbm_slab_ccl_export(self._h), "lbm_slab_ccl_export")

    def slab_ccl_import(self, use_lo, use_hi):
        n = C.c_int()
        _chk(load().lbm_slab_ccl_import(self._h, int(bool(use_lo)), int(bool(use_hi)), C.byref(n)),
             "lbm_slab_ccl_import")
        return int(n.value)

    def slab_ccl_finish(self, z0, z1):
        n = C.c_longlong()
        m = C.c_double()
        _chk(load().lbm_slab_ccl_finish(self._h, int(z0), int(z1), C.byref(n), C.byref(m)),
             "lbm_slab_ccl_finish")
        return n.value, m.value

    def slab_buffer(self, which):
        """(device pointer, bytes) of exchange buffer `which` (include/lbm.h lbm_slab_buffer)."""
        ptr = C.c_void_p()
        n = C.c_longlong()
        _chk(load().lbm_slab_buffer(self._h, int(which), C.byref(ptr), C.byref(n)),
             "lbm_slab_buffer")
        return int(ptr.value or 0), int(n.value)

    def step_info(self):
        v = (C.c_int * 8)()
        _chk(load().lbm_step_info(self._h, v), "lbm_step_info")
        return {"graph": bool(v[1]), "pdl": bool(v[2]), "reverse": bool(v[3]),
                "keep_psi": v[4] / 1000.0, "wide_tiles": v[5]}

    def sync(self):
        _chk(load().lbm_sync(self._h), "lbm_sync")

    def get_macroscopic(self, fields=("rhoA", "rhoB", "ux", "uy", "uz", "P"), out=None):
        names = ("rhoA", "rhoB", "ux", "uy", "uz", "P")
        res = {}
        ptrs = []
        for k in names:
            if k in fields:
                res[k] = out[k] if out is not None else np.empty(self.shape, np.float64)
                a = res[k]
                if (not isinstance(a, np.ndarray) or a.dtype != np.float64 or a.shape != self.shape
                        or not a.flags["C_CONTIGUOUS"] or not a.flags["WRITEABLE"]):
                    raise ValueError(f"out[{k!r}] must be a writeable C-contiguous float64 array "
                                     f"of shape {self.shape}")
                ptrs.append(a.ctypes.data)
            else:
                ptrs.append(None)
        _chk(load().lbm_get_macroscopic(self._h, *ptrs), "lbm_get_macroscopic")
        return res

    def diagnostics(self):
        m = (C.c_double * 2)()
        j = (C.c_double * 3)()
        _chk(load().lbm_diagnostics(self._h, m, j), "lbm_diagnostics")
        return np.array(m), np.array(j)

    def saturation(self, comp, z0=0, z1=None):
        z1 = self.shape[0] if z1 is None else z1
        s = C.c_double()
        _chk(load().lbm_saturation(self._h, int(comp), int(z0), int(z1), C.byref(s)),
             "lbm_saturation")
        return s.value

    def trapped_volume(self, comp, z0=0, z1=None):
        z1 = self.shape[0] if z1 is None else z1
        n = C.c_longlong()
        m = C.c_double()
        _chk(load().lbm_trapped_volume(self._h, int(comp), int(z0), int(z1), C.byref(n),
                                       C.byref(m)), "lbm_trapped_volume")
        return n.value, m.value

    def trapped_volume_static(self, comp, z0=0, z1=None):
        z1 = self.shape[0] if z1 is None else z1
        n = C.c_longlong()
        m = C.c_double()
        _chk(load().lbm_trapped_volume_static(self._h, int(comp), int(z0), int(z1), C.byref(n),
                                              C.byref(m)), "lbm_trapped_volume_static")
        return n.value, m.value

    def mean_pressure(self, z0=0, z1=None):
        z1 = self.shape[0] if z1 is None else z1
        v = C.c_double()
        _chk(load().lbm_mean_pressure(self._h, int(z0), int(z1), C.byref(v)), "lbm_mean_pressure")
        return v.value

    def memory_bytes(self):
        b = (C.c_longlong * 4)()
        _chk(load().lbm_memory_bytes(self._h, b), "lbm_memory_bytes")
        return dict(zip(("populations", "psi", "index", "other"), [int(v) for v in b]))

    def set_profiling(self, on):
        _chk(load().lbm_set_profiling(self._h, int(bool(on))), "lbm_set_profiling")

    def last_step_profile(self):
        ms = (C.c_double * 4)()
        n = C.c_longlong()
        _chk(load().lbm_last_step_profile(self._h, ms, C.byref(n)), "lbm_last_step_profile")
        return dict(zip(("density", "wallpsi", "collide_stream", "open_planes"),
                        [float(v) for v in ms])), int(n.value)
