"""GPU tests of the z-slab sharded step (include/lbm.h "z-slab sharding").
All slabs of a box live on the one GPU of the test box and are stepped one after another, the
exchanges being device copies of the very buffers NCCL would move (paper_2207_01534_b200/slab.py).

What is checked: the sharded step is BIT-IDENTICAL to the unsharded CUDA path on every population
(same kernels, same summation order, for any number of slabs, fp64 and fp32), and matches the CPU
oracle to the north-star tolerances (fp64: every population 1e-10 relative)."""
import ctypes as C

import numpy as np
import pytest

from oracle import LbmRef
from paper_2207_01534_b200 import Lbm, LbmError, load, make_params
from paper_2207_01534_b200 import lbm as binding
from paper_2207_01534_b200.slab import SlabLbm, local_box
from workloads import default_params, make_config, sphere_pack_mask

pytestmark = pytest.mark.gpu


def _rock_case(n=40, bits=64, seed=21):
    """config 5 recipe at a small edge (periodic sphere pack, body force) plus wetting and a
    viscosity ratio, so that every term of the step is switched on"""
    c = make_config(5, size=n, seed=seed, storage_bits=bits, xi=-0.2, tau=(1.2, 0.7),
                    accel=(1e-6, -2e-6, 3e-6))
    rng = np.random.Generator(np.random.PCG64(seed))
    fl = c["mask"] == 0
    for k in ("rhoA", "rhoB"):
        c[k] = np.where(fl, c[k] * (1.0 + rng.uniform(-1e-3, 1e-3, c[k].shape)), 0.0)
    return c


def _identical_pops(a, b, mask):
    fl = mask == 0
    for s in (0, 1):
        fa, fb = a.get_populations(s)[:, fl], b.get_populations(s)[:, fl]
        assert np.array_equal(fa, fb), (s, np.abs(fa - fb).max())


@pytest.mark.parametrize("parts", [1, 2, 3])
def test_slab_fp64_bit_identical_to_unsharded_and_matches_oracle(parts):
    c = _rock_case(40, 64)
    g = Lbm(c["mask"], c["params"])
    s = SlabLbm(c["mask"], c["params"], parts=parts)
    assert s.num_fluid == g.num_fluid
    g.set_density(c["rhoA"], c["rhoB"])
    s.set_density(c["rhoA"], c["rhoB"])
    g.step(60)
    s.step(60)
    _identical_pops(s, g, c["mask"])
    if parts == 3:
        o = LbmRef(c["mask"], c["params"])
        o.set_density(c["rhoA"], c["rhoB"])
        o.step(60)
        fl = c["mask"] == 0
        for comp in (0, 1):
            a, b = s.get_populations(comp)[:, fl], o.get_populations(comp)[:, fl]
            assert (np.abs(a - b) / np.abs(b)).max() <= 1e-10
    # macroscopic fields and sums over slabs
    mg, ms = g.get_macroscopic(), s.get_macroscopic()
    for k in mg:
        assert np.array_equal(mg[k], ms[k]), k
    m_g, j_g = g.diagnostics()
    m_s, j_s = s.diagnostics()
    assert np.max(np.abs(m_s - m_g) / m_g) < 1e-13 and np.max(np.abs(j_s - j_g)) < 1e-10
    # stepping continues correctly after the getters
    g.step(5)
    s.step(5)
    _identical_pops(s, g, c["mask"])
    s.close()
    g.close()


@pytest.mark.parametrize("parts", [2, 4])
def test_slab_fp32_bit_identical_to_unsharded(parts):
    c = _rock_case(48, 32, seed=22)
    g = Lbm(c["mask"], c["params"])
    s = SlabLbm(c["mask"], c["params"], parts=parts)
    g.set_density(c["rhoA"], c["rhoB"])
    s.set_density(c["rhoA"], c["rhoB"])
    g.step(100)
    s.step(100)
    _identical_pops(s, g, c["mask"])
    mg, ms = g.get_macroscopic(("rhoA", "rhoB", "uz")), s.get_macroscopic(("rhoA", "rhoB", "uz"))
    for k in mg:
        assert np.array_equal(mg[k], ms[k]), k
    s.close()
    g.close()


def test_slab_no_solids_and_thinnest_slabs():
    """config 1 (no solids: empty wall pass, full planes) cut into slabs of exactly 2 planes: every
    owned plane is a boundary plane and both halo planes of a face come from different slabs'
    planes."""
    c = make_config(1, size=16)
    g = Lbm(c["mask"], c["params"])
    s = SlabLbm(c["mask"], c["params"], parts=8)
    assert all(z1 - z0 == 2 for z0, z1 in s.ranges)
    g.set_density(c["rhoA"], c["rhoB"])
    s.set_density(c["rhoA"], c["rhoB"])
    g.step(40)
    s.step(40)
    _identical_pops(s, g, c["mask"])
    s.close()
    g.close()


def test_slab_index_variants_agree():
    """Plain (non-PDL) launches, forward tile order and plain psi stores give the same sharded
    result as the default path (boundary tiles read the compact wide-tile table there)."""
    c = _rock_case(32, 32, seed=23)
    ref = None
    for opt in (None, {"pdl": 0}, {"reverse": 0}, {"keep_psi_mb": 0}):
        s = SlabLbm(c["mask"], c["params"], parts=2, options=opt)
        s.set_density(c["rhoA"], c["rhoB"])
        s.step(30)
        f = [s.get_populations(k) for k in (0, 1)]
        s.close()
        if ref is None:
            ref = f
        else:
            for a, b in zip(f, ref):
                assert np.array_equal(a, b), opt


def test_slab_checkpoint_roundtrip():
    c = _rock_case(32, 64, seed=24)
    a = SlabLbm(c["mask"], c["params"], parts=2)
    a.set_density(c["rhoA"], c["rhoB"])
    a.step(10)
    f = [a.get_populations(k) for k in (0, 1)]
    b = SlabLbm(c["mask"], c["params"], parts=3)     # restore onto a different cut
    for k in (0, 1):
        b.set_populations(k, f[k])
    a.step(10)
    b.step(10)
    _identical_pops(a, b, c["mask"])
    a.close()
    b.close()


def test_slab_error_paths():
    lib = load()
    m = sphere_pack_mask(16, 5, 3.0, 4.0)[0]
    ml = local_box(m, 0, 8)
    p = default_params()
    s = Lbm(ml, p, slab=True)
    with pytest.raises(LbmError) as e:
        s.step(1)                                   # lbm_step is not the slab step
    assert e.value.code == binding.LBM_EINVAL
    with pytest.raises(LbmError):
        s.slab_collide(0)                           # density pass + psi exchange come first
    with pytest.raises(LbmError):
        s.slab_unpack()
    with pytest.raises(LbmError):
        s.saturation(0)
    with pytest.raises(LbmError):
        s.get_macroscopic()                         # psi of the current state is missing
    with pytest.raises(LbmError):
        s.slab_density(1)                           # boundary part first
    s.slab_density(0)
    with pytest.raises(LbmError):
        s.slab_collide(0)
    s.slab_density(1)
    s.slab_density(0)                               # a step may restart after its density pass
    s.slab_density(1)
    with pytest.raises(LbmError):
        s.slab_collide(1)
    s.slab_collide(0)
    s.slab_collide(1)
    with pytest.raises(LbmError):
        s.slab_density(0)                           # unpack of the running step is missing
    s.slab_unpack()
    with pytest.raises(LbmError):
        s.slab_buffer(12)
    sizes = [s.slab_buffer(w)[1] for w in range(12)]
    assert all(b % 8 == 0 for b in sizes) and sizes[0] > 0 and sizes[8:] == [16 * 16 * 4] * 4
    with pytest.raises(LbmError):
        s.slab_ccl_export()                         # no lbm_slab_ccl_begin
    with pytest.raises(LbmError):
        s.slab_ccl_begin(0, 1, 1)                   # psi of the current state is missing
    s.close()
    g = Lbm(m, p)
    with pytest.raises(LbmError):
        g.slab_density(0)                           # not a slab context
    g.close()
    h = C.c_void_p()
    ps = make_params(p)
    # a z-periodic box has no end of its own: both ends of every slab are cuts
    assert lib.lbm_create_slab(C.byref(h), ml.ctypes.data, 16, 16, 12, C.byref(ps), 0, 1) == binding.LBM_EINVAL
    assert lib.lbm_create_slab(C.byref(h), ml.ctypes.data, 16, 16, 12, C.byref(ps), 1, 2) == binding.LBM_EINVAL
    thin = np.zeros((5, 4, 4), np.uint8)
    assert lib.lbm_create_slab(C.byref(h), thin.ctypes.data, 4, 4, 5, C.byref(ps), 1, 1) == binding.LBM_EINVAL
    # the open end of a slab must be solid-free like the open planes of lbm_create (reading R12)
    po = make_params(default_params(z_open=1, inlet_kind=1, outlet_kind=1))
    mo = np.zeros((8, 4, 4), np.uint8)
    mo[1, 2, 2] = 1
    assert lib.lbm_create_slab(C.byref(h), mo.ctypes.data, 4, 4, 8, C.byref(po), 0, 1) == binding.LBM_ESOLIDOPEN
    assert lib.lbm_create_slab(C.byref(h), mo.ctypes.data, 4, 4, 8, C.byref(po), 1, 1) == binding.LBM_OK
    lib.lbm_destroy(h)


# ------------------------------------------------------------------ z-open boxes (configs 3, 4)

def _open_case(k, n, bits, **kw):
    c = make_config(k, size=n, storage_bits=bits, **kw)
    rng = np.random.Generator(np.random.PCG64(100 + k))
    fl = c["mask"] == 0
    for key in ("rhoA", "rhoB"):
        c[key] = np.where(fl, c[key] * (1.0 + rng.uniform(-1e-3, 1e-3, c[key].shape)), 0.0)
    return c


@pytest.mark.parametrize("k,parts,kinds", [(3, 2, None), (3, 3, (4, 3)), (4, 2, None), (4, 4, (3, 3))])
def test_open_box_slabs_fp64_bit_identical_and_oracle(k, parts, kinds):
    """configs 3 (velocity inlet) and 4 (pressure inlet, viscosity ratio 10) at 40^3: the inlet
    plane lives on the first slab, the outlet plane on the last, middle slabs have none; NEEM
    (kinds 1, 2) and Zou-He (kinds 3, 4) planes; boundary ramp between the steps."""
    kw = {} if kinds is None else {"inlet_kind": kinds[0], "outlet_kind": kinds[1]}
    c = _open_case(k, 40, 64, **kw)
    g = Lbm(c["mask"], c["params"])
    s = SlabLbm(c["mask"], c["params"], parts=parts)
    assert s.halo[0] == (0, 1) and s.halo[-1] == (1, 0)
    g.set_density(c["rhoA"], c["rhoB"])
    s.set_density(c["rhoA"], c["rhoB"])
    g.step(30)
    s.step(30)
    _identical_pops(s, g, c["mask"])
    iv = 1.03 if c["params"]["inlet_kind"] in (1, 3) else 2e-4
    g.set_boundary(iv, 0.99)
    s.set_boundary(iv, 0.99)
    g.step(30)
    s.step(30)
    _identical_pops(s, g, c["mask"])
    mg, ms = g.get_macroscopic(), s.get_macroscopic()
    for key in mg:
        assert np.array_equal(mg[key], ms[key]), key
    nz = c["mask"].shape[0]
    for z0, z1 in ((0, nz), (8, nz - 8), (0, 1), (nz - 1, nz), (5, 23)):
        assert abs(s.saturation(1, z0, z1) - g.saturation(1, z0, z1)) < 1e-12
        assert abs(s.mean_pressure(z0, z1) - g.mean_pressure(z0, z1)) < 1e-12
    g.step(3)
    s.step(3)
    _identical_pops(s, g, c["mask"])
    if parts == 2:
        o = LbmRef(c["mask"], c["params"])
        o.set_density(c["rhoA"], c["rhoB"])
        o.step(30)
        o.set_boundary(iv, 0.99)
        o.step(33)
        fl = c["mask"] == 0
        for comp in (0, 1):
            a, b = s.get_populations(comp)[:, fl], o.get_populations(comp)[:, fl]
            assert (np.abs(a - b) / np.abs(b)).max() <= 1e-10
    s.close()
    g.close()


@pytest.mark.parametrize("k,parts", [(3, 3), (4, 2)])
def test_open_box_slabs_fp32_bit_identical(k, parts):
    c = _open_case(k, 48, 32)
    g = Lbm(c["mask"], c["params"])
    s = SlabLbm(c["mask"], c["params"], parts=parts)
    g.set_density(c["rhoA"], c["rhoB"])
    s.set_density(c["rhoA"], c["rhoB"])
    g.step(100)
    s.step(100)
    _identical_pops(s, g, c["mask"])
    m_g, _ = g.diagnostics()
    m_s, _ = s.diagnostics()
    assert np.max(np.abs(m_s - m_g) / m_g) < 1e-12
    s.close()
    g.close()


# ------------------------------------------------------------------ two processes, one GPU

def _rank_worker(rank, world, port, out):
    """One rank of the distributed driver: owns slab `rank`, exchanges through torch.distributed
    (gloo, messages staged through pinned host memory -- NCCL refuses two ranks on one device; no
    kernel ever waits on another rank, the waits are on the host), and compares its owned planes
    with an unsharded run of the same box that it makes itself."""
    import os
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch
    import torch.distributed as dist
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ok, msg = True, ""
    try:
        for k, bits in ((5, 64), (4, 32)):
            c = make_config(k, size=32, storage_bits=bits)
            s = SlabLbm(c["mask"], c["params"], rank=rank, world=world)
            g = Lbm(c["mask"], c["params"])
            s.set_density(c["rhoA"], c["rhoB"])
            g.set_density(c["rhoA"], c["rhoB"])
            s.step(25)
            g.step(25)
            z0, z1 = s.ranges[rank]
            fl = c["mask"][z0:z1] == 0
            for comp in (0, 1):
                a = s.get_populations(comp)[:, fl]
                b = g.get_populations(comp)[:, z0:z1][:, fl]
                if not np.array_equal(a, b):
                    ok, msg = False, f"cfg {k} comp {comp}: populations differ"
            ms = s.get_macroscopic(("rhoA", "uz"))
            mg = g.get_macroscopic(("rhoA", "uz"))
            for key in ms:
                if not np.array_equal(ms[key], mg[key][z0:z1]):
                    ok, msg = False, f"cfg {k}: {key} differs"
            m_s, j_s = s.diagnostics()          # all_reduce over ranks
            m_g, j_g = g.diagnostics()
            if np.max(np.abs(m_s - m_g) / m_g) > 1e-12:
                ok, msg = False, f"cfg {k}: mass {m_s} vs {m_g}"
            nz = c["mask"].shape[0]
            if abs(s.saturation(1, 3, nz - 3) - g.saturation(1, 3, nz - 3)) > 1e-12:
                ok, msg = False, f"cfg {k}: saturation"
            s.step(3)
            g.step(3)
            a = s.get_populations(0)[:, fl]
            b = g.get_populations(0)[:, z0:z1][:, fl]
            if not np.array_equal(a, b):
                ok, msg = False, f"cfg {k}: populations differ after the getters"
            s.close()
            g.close()
        dist.barrier()
    except Exception as e:  # noqa: BLE001 -- reported to the parent
        ok, msg = False, repr(e)
    out.put((rank, ok, msg))
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_distributed_driver_ranks_share_one_gpu(world):
    import os
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 32500 + os.getpid() % 2000 + world
    procs = [ctx.Process(target=_rank_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=600) for _ in procs)
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    assert all(ok for _, ok, _ in res), res


# ------------------------------------------------------------------ trapped volume across cuts

def _blob_state(shape, seed, solid, z_open):
    """Smooth random two-phase field on a random solid mask: many clusters of both phases, some
    touching the ends, many cut by slab boundaries."""
    rng = np.random.Generator(np.random.PCG64(seed))
    mask = (rng.uniform(size=shape) < solid).astype(np.uint8)
    if z_open:
        mask[:2] = 0
        mask[-2:] = 0
    f = rng.standard_normal(shape)
    k = [np.fft.fftfreq(n) for n in shape]
    kk = k[0][:, None, None] ** 2 + k[1][None, :, None] ** 2 + k[2][None, None, :] ** 2
    f = np.real(np.fft.ifftn(np.fft.fftn(f) * np.exp(-2 * (np.pi * 2.5) ** 2 * kk)))
    f /= f.std()
    rA = np.where(f > 0.3, 0.9, 0.1) + 0.01 * rng.uniform(size=shape)
    return mask, rA, 1.0 - rA


@pytest.mark.parametrize("shape,solid,z_open,parts", [((40, 36, 44), 0.25, 0, 2),
                                                      ((40, 36, 44), 0.15, 0, 5),
                                                      ((48, 32, 32), 0.2, 1, 3),
                                                      ((64, 24, 24), 0.3, 1, 8)])
def test_slab_trapped_volume_matches_unsharded(shape, solid, z_open, parts):
    mask, rA, rB = _blob_state(shape, 41, solid, z_open)
    kw = dict(storage_bits=64)
    if z_open:
        kw.update(z_open=1, inlet_kind=1, inlet_comp=1, inlet_rho=1.0, outlet_kind=1, outlet_comp=0,
                  outlet_rho=1.0)
    p = default_params(**kw)
    g = Lbm(mask, p)
    s = SlabLbm(mask, p, parts=parts)
    g.set_density(rA, rB)
    s.set_density(rA, rB)
    nz = shape[0]
    seen = 0
    for comp in (0, 1):
        for z0, z1 in ((0, nz), (nz // 4, 3 * nz // 4), (nz - 1, nz), (0, 1), (5, 6)):
            ng, mg = g.trapped_volume(comp, z0, z1)
            ns, ms = s.trapped_volume(comp, z0, z1)
            assert ns == ng, (comp, z0, z1, ns, ng)
            assert abs(ms - mg) <= 1e-12 * max(1.0, mg)
            seen += ng
    assert seen > 0
    g.step(3)
    s.step(3)
    assert s.trapped_volume(0) == pytest.approx(g.trapped_volume(0), rel=1e-12)
    s.step(2)                                      # stepping goes on after the query
    g.step(2)
    _identical_pops(s, g, mask)
    s.close()
    g.close()


def test_slab_trapped_volume_serpentine_crosses_every_cut_many_times():
    """A single phase-A channel that winds up and down through the whole box: its end-connected
    flag has to travel across every cut several times before the iteration settles.  A second,
    closed loop of the same shape but detached from the end planes is trapped."""
    nz, ny, nx = 32, 12, 40
    mask = np.zeros((nz, ny, nx), np.uint8)
    A = np.zeros((nz, ny, nx), bool)
    for k, x in enumerate(range(2, 38, 4)):        # vertical legs, joined alternately at top/bottom
        A[3:29, 2, x] = True
        if x + 4 < 38:
            A[28 if k % 2 == 0 else 3, 2, x:x + 5] = True
    A[0:4, 2, 2] = True                            # the first leg reaches z = 0
    B = np.zeros_like(A)
    for k, x in enumerate(range(2, 38, 4)):        # same serpentine at y = 8, not reaching an end
        B[3:29, 8, x] = True
        if x + 4 < 38:
            B[28 if k % 2 == 0 else 3, 8, x:x + 5] = True
    rA = np.where(A | B, 0.9, 0.1)
    p = default_params(storage_bits=64)
    g = Lbm(mask, p)
    g.set_density(rA, 1.0 - rA)
    want = g.trapped_volume(0)
    assert want[0] == int(B.sum())
    for parts in (2, 4, 8):
        s = SlabLbm(mask, p, parts=parts)
        s.set_density(rA, 1.0 - rA)
        got = s.trapped_volume(0)
        assert got[0] == want[0] and abs(got[1] - want[1]) < 1e-9
        s.close()
    g.close()


@pytest.mark.parametrize("k,bits", [(5, 64), (5, 32), (4, 32), (3, 64)])
def test_native_slab_step_ring_of_one(k, bits):
    """lbm_slab_step: the sharded step sequenced inside the library, exchanges as grouped
    ncclSend / ncclRecv on a side stream.  One GPU can host one NCCL rank, so the ring has one
    slab: in a z-periodic box (config 5) it exchanges both faces with itself -- every pack /
    send / receive / unpack path runs, with the message matching of a 1- or 2-rank ring --, in a
    z-open box (configs 3, 4) it owns both open planes and has nothing to exchange.  Bit-identical
    to the unsharded step and to the call-by-call sequence driven from Python, across getters in
    between."""
    c = make_config(k, size=40, storage_bits=bits)
    ref = Lbm(c["mask"], c["params"])
    ref.set_density(c["rhoA"], c["rhoB"])
    ref.step(25)
    want = [ref.get_populations(s) for s in (0, 1)]
    want_sat = ref.saturation(1)
    want_trapped = ref.trapped_volume(0)
    want_p = ref.mean_pressure(0, c["mask"].shape[0])
    ref.close()
    for native in (True, False):
        s = SlabLbm(c["mask"], c["params"], rank=0, world=1, native=native)
        assert s.native == native
        s.set_density(c["rhoA"], c["rhoB"])
        s.step(10)
        s.saturation(0)                       # a query between steps (density + psi halo, phase 2)
        s.step(15)
        for comp in (0, 1):
            assert np.array_equal(s.get_populations(comp), want[comp]), (native, comp)
        assert s.saturation(1) == want_sat
        assert s.trapped_volume(0) == want_trapped      # cluster flags cross the (self-)cut by kind 2
        assert abs(s.mean_pressure(0, c["mask"].shape[0]) - want_p) < 1e-12
        s.close()


def test_native_slab_step_needs_a_communicator():
    from paper_2207_01534_b200 import LbmError
    c = make_config(5, size=24)
    s = SlabLbm(c["mask"], c["params"], parts=1)           # in-process slabs: no communicator
    with pytest.raises(LbmError) as e:
        s.sims[0].slab_step(1)
    assert e.value.code == -1
    s.close()
