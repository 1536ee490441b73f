"""CPU-side tests of the product library: it loads, exports every symbol include/lbm.h declares,
rejects bad arguments with the documented codes, refuses to run without a GPU (no CPU fallback),
and builds the compact neighbour index correctly (checked against a brute-force numpy index).
No compute entry point is called without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2207_01534_b200 as lbm
from paper_2207_01534_b200 import lbm as binding
from workloads import default_params, make_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

E = np.array([(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1),
              (1, 1, 0), (-1, 1, 0), (1, -1, 0), (-1, -1, 0), (1, 0, 1), (-1, 0, 1), (1, 0, -1),
              (-1, 0, -1), (0, 1, 1), (0, -1, 1), (0, 1, -1), (0, -1, -1)])


def test_library_exports_every_declared_symbol():
    lib = lbm.load()
    header = open(os.path.join(ROOT, "include", "lbm.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(lbm_[a-z_]+)\s*\(", header))
    assert declared == set(lbm.SYMBOLS), declared ^ set(lbm.SYMBOLS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_params_struct_layout_matches_header():
    """The ctypes mirror must have the C struct's size: 4 doubles+3 doubles, ints, ... = 112 B."""
    assert C.sizeof(lbm.lbm_params) == 112
    p = lbm.make_params(default_params(G=3.5, tau=(1.5, 0.6), xi=-0.2, accel=(1, 2, 3)))
    assert (p.G, p.tau[0], p.tau[1], p.xi, p.accel[2], p.storage_bits) == (3.5, 1.5, 0.6, -0.2, 3, 32)


def _create_rc(mask, params):
    lib = lbm.load()
    h = C.c_void_p()
    nz, ny, nx = mask.shape
    ps = lbm.make_params(params)
    rc = lib.lbm_create(C.byref(h), mask.ctypes.data, nx, ny, nz, C.byref(ps))
    if rc == 0:
        lib.lbm_destroy(h)
    return rc, (lib.lbm_last_error() or b"").decode()


def test_bad_arguments_return_documented_codes():
    lib = lbm.load()
    m = np.zeros((6, 4, 4), np.uint8)
    assert _create_rc(m, default_params(tau=(0.5, 1.0)))[0] == binding.LBM_EINVAL
    assert _create_rc(m, default_params(tau=(1.0, float("nan"))))[0] == binding.LBM_EINVAL
    assert _create_rc(m, default_params(storage_bits=16))[0] == binding.LBM_EINVAL
    assert _create_rc(m, default_params(z_open=1, inlet_kind=7))[0] == binding.LBM_EINVAL
    assert _create_rc(m, default_params(z_open=1, inlet_comp=2))[0] == binding.LBM_EINVAL
    assert _create_rc(np.ones((4, 4, 4), np.uint8), default_params())[0] == binding.LBM_ENOFLUID
    ms = m.copy()
    ms[1, 2, 2] = 1
    rc, msg = _create_rc(ms, default_params(z_open=1))
    assert rc == binding.LBM_ESOLIDOPEN and "open plane" in msg
    # NULL pointers / NULL context: codes, never a crash
    h = C.c_void_p()
    assert lib.lbm_create(C.byref(h), None, 4, 4, 4, None) == binding.LBM_EINVAL
    assert lib.lbm_step(None, 1) == binding.LBM_EINVAL
    assert lib.lbm_set_density(None, None, None) == binding.LBM_EINVAL
    assert lib.lbm_num_fluid(None) == -1
    lib.lbm_destroy(None)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    rc, msg = _create_rc(np.zeros((4, 4, 4), np.uint8), default_params())
    assert rc == binding.LBM_ECUDA and "no CPU fallback" in msg
    with pytest.raises(lbm.LbmError):
        lbm.Lbm(np.zeros((4, 4, 4), np.uint8), default_params())


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2207_01534_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".cpp", ".hpp", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "lbmref" not in src and "import oracle" not in src and "from oracle" not in src, fn


def _brute_index(mask, z_open):
    nz, ny, nx = mask.shape
    fluid = mask == 0
    ids = np.full(mask.shape, -1, np.int64)
    nf = int(fluid.sum())
    ids[fluid] = np.arange(nf)                      # raster order, x fastest
    z, y, x = np.nonzero(fluid)
    # wall solids: solid with any fluid neighbour (mirror across open planes)
    def shifted(a, i, fill_mirror):
        out = np.empty_like(a)
        ex, ey, ez = E[i]
        r = np.roll(a, (-ez, -ey, -ex), (0, 1, 2))   # r[z,y,x] = a[z+ez, y+ey, x+ex] periodic
        out[:] = r
        if z_open and ez != 0:
            zb = nz - 1 if ez > 0 else 0
            m = np.roll(a, (ez, -ey, -ex), (0, 1, 2))  # a[z-ez, y+ey, x+ex]
            out[zb] = m[zb]
        return out
    anyfluid = np.zeros(mask.shape, bool)
    for i in range(1, 19):
        anyfluid |= shifted(fluid, i, True)
    wall = (~fluid) & anyfluid
    nw = int(wall.sum())
    ids[wall] = nf + np.arange(nw)
    nbr = np.empty((18, nf), np.int64)
    for i in range(1, 19):
        ex, ey, ez = E[i]
        xn, yn, zn = (x + ex) % nx, (y + ey) % ny, z + ez
        beyond = (zn < 0) | (zn >= nz)
        if z_open:
            zn = np.where(beyond, z - ez, zn)
        else:
            zn = zn % nz
            beyond[:] = False
        t = ids[zn, yn, xn]
        nbr[i - 1] = np.where(beyond, -(t + 1), t)
    return ids, nbr, nf, nw


@pytest.mark.parametrize("z_open", [0, 1])
def test_compact_index_matches_bruteforce(z_open):
    rng = np.random.Generator(np.random.PCG64(17))
    mask = (rng.uniform(size=(9, 7, 10)) < 0.35).astype(np.uint8)
    if z_open:
        mask[:2] = 0
        mask[-2:] = 0
    vox2id, nbr, nf, nw = lbm.lbm_build_index(mask, z_open)
    ids, nbr_ref, nf_ref, nw_ref = _brute_index(mask, z_open)
    assert (nf, nw) == (nf_ref, nw_ref)
    assert np.array_equal(vox2id, ids)
    assert np.array_equal(nbr, nbr_ref)


def test_compact_index_on_config_geometries():
    c = make_config(3, size=32)
    vox2id, nbr, nf, nw = lbm.lbm_build_index(c["mask"], 1)
    ids, nbr_ref, nf_ref, nw_ref = _brute_index(c["mask"], 1)
    assert (nf, nw) == (nf_ref, nw_ref) and np.array_equal(nbr, nbr_ref)
    assert nf == int((c["mask"] == 0).sum())


def test_library_has_no_global_knobs():
    """no global state, no environment variables.  The shared object neither
    imports getenv nor carries an LBM_B200_* string; execution options travel in lbm_options."""
    import subprocess
    path = binding.library_path()
    lbm.load()
    und = subprocess.run(["nm", "-D", "--undefined-only", path], capture_output=True, text=True).stdout
    assert "getenv" not in und
    assert b"LBM_B200_" not in open(path, "rb").read()
    src = "".join(open(os.path.join(ROOT, "paper_2207_01534_b200", "csrc", f)).read()
                  for f in ("lbm.cu", "kernels.cuh", "geometry.cpp", "torch_shim.cpp"))
    assert "getenv" not in src


def test_options_struct_and_defaults():
    assert C.sizeof(lbm.lbm_options) == 16
    o = lbm.make_options()
    assert (o.graph, o.pdl, o.reverse, o.keep_psi_mb) == (-1, 1, 1, 48)
    o = lbm.make_options({"reverse": 0, "graph": 0})
    assert (o.reverse, o.graph) == (0, 0)
    with pytest.raises(KeyError):
        lbm.make_options({"tile": 1287})
    # bad option values are rejected before any device is needed
    h = C.c_void_p()
    m = np.zeros((4, 4, 4), np.uint8)
    ps = lbm.make_params(default_params())
    for bad in ({"reverse": 5}, {"graph": 3}, {"pdl": 2}, {"keep_psi_mb": -1}):
        po = lbm.make_options(bad)
        rc = lbm.load().lbm_create_opt(C.byref(h), m.ctypes.data, 4, 4, 4, C.byref(ps), C.byref(po))
        assert rc == binding.LBM_EINVAL
