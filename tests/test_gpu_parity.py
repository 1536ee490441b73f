"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Run with `-m gpu` on a B200.

Tolerances (BASELINE.json north_star; norms are reading R22, stated here):
  fp64 build : every population, relative  abs(a-b)/abs(b) <= 1e-10 after 200 steps;
  fp32 build : component densities element-wise relative <= 1e-4 after 100 steps; velocities
               max-norm of the difference / max-norm of the oracle field <= 1e-4;
               total mass per component relative <= 1e-6.
"""
import numpy as np
import pytest

from oracle import LbmRef
from paper_2207_01534_b200 import Lbm
from workloads import default_params, make_config

pytestmark = pytest.mark.gpu


def _pair(mask, rhoA, rhoB, params):
    o = LbmRef(mask, params)
    g = Lbm(mask, params)
    o.set_density(rhoA, rhoB)
    g.set_density(rhoA, rhoB)
    return o, g


def _pop_rel(o, g, mask):
    fl = mask == 0
    worst = 0.0
    for s in (0, 1):
        a, b = g.get_populations(s), o.get_populations(s)
        assert np.all(a[:, ~fl] == 0.0)
        rel = np.abs(a[:, fl] - b[:, fl]) / np.abs(b[:, fl])
        worst = max(worst, float(rel.max()))
    return worst


def _check_fp32(o, g, mask, rho_tol=1e-4, u_tol=1e-4, mass_tol=1e-6):
    fl = mask == 0
    mo, mg = o.get_macroscopic(), g.get_macroscopic()
    for k in ("rhoA", "rhoB"):
        rel = np.abs(mg[k][fl] - mo[k][fl]) / np.abs(mo[k][fl])
        assert rel.max() <= rho_tol, (k, rel.max())
        assert np.all(mg[k][~fl] == 0.0)
    uo = np.stack([mo[k][fl] for k in ("ux", "uy", "uz")])
    ug = np.stack([mg[k][fl] for k in ("ux", "uy", "uz")])
    assert np.abs(ug - uo).max() <= u_tol * np.abs(uo).max(), np.abs(ug - uo).max() / np.abs(uo).max()
    rel = np.abs(mg["P"][fl] - mo["P"][fl]) / np.abs(mo["P"][fl])
    assert rel.max() <= 1e-4
    m_o, _ = o.diagnostics()
    m_g, _ = g.diagnostics()
    assert np.max(np.abs(m_g - m_o) / m_o) <= mass_tol, np.abs(m_g - m_o) / m_o


# ------------------------------------------------------------------ config 1: fp64, 1e-10

def test_cfg1_fp64_every_population_200_steps():
    c = make_config(1)
    assert c["params"]["storage_bits"] == 64
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    assert _pop_rel(o, g, c["mask"]) == 0.0            # identical initial state
    o.step(200)
    g.step(200)
    assert _pop_rel(o, g, c["mask"]) <= 1e-10
    m_o, j_o = o.diagnostics()
    m_g, j_g = g.diagnostics()
    assert np.max(np.abs(m_g - m_o) / m_o) < 1e-13 and np.max(np.abs(j_g - j_o)) < 1e-11


def test_cfg1_fp32_build():
    c = make_config(1, storage_bits=32)
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(100)
    g.step(100)
    _check_fp32(o, g, c["mask"])


# ------------------------------------------------------------------ all features, fp64, ragged sizes

@pytest.mark.parametrize("shape,seed", [((5, 6, 8), 1), ((9, 33, 67), 2), ((23, 17, 130), 3)])
def test_random_porous_fp64_all_features(shape, seed):
    """Random solids (bounce-back + IVSD), unequal tau, wetting, body force; sizes that are not
    multiples of the block size and span several blocks."""
    rng = np.random.Generator(np.random.PCG64(seed))
    mask = (rng.uniform(size=shape) < 0.3).astype(np.uint8)
    rA = np.where(mask == 0, rng.uniform(0.05, 1.0, shape), 0.0)
    rB = np.where(mask == 0, rng.uniform(0.05, 1.0, shape), 0.0)
    p = default_params(G=3.5, tau=(1.2, 0.7), xi=0.25, accel=(1e-5, -2e-5, 3e-5), storage_bits=64)
    o, g = _pair(mask, rA, rB, p)
    o.step(20)
    g.step(20)
    assert _pop_rel(o, g, mask) <= 1e-10
    mo, mg = o.get_macroscopic(), g.get_macroscopic()
    for k in mo:
        assert np.max(np.abs(mo[k] - mg[k])) <= 1e-12, k


def test_worked_example_on_gpu():
    """SURVEY.md App. C set-up (the oracle is pinned to its printed values in the CPU suite)."""
    nx, ny, nz = 8, 6, 5
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    mask = ((x + 2 * y + 3 * z) % 7 == 0).astype(np.uint8)
    rA = 0.5 + 0.4 * np.sin(2 * np.pi * x / 8) * np.cos(2 * np.pi * y / 6) + 0.05 * np.cos(2 * np.pi * z / 5)
    p = default_params(G=3.5, tau=(1.0, 0.7), xi=0.2, accel=(0.0, 0.0, 1e-5), storage_bits=64)
    o, g = _pair(mask, rA, 1.03 - rA, p)
    o.step(5)
    g.step(5)
    assert _pop_rel(o, g, mask) <= 1e-12
    m, j = g.diagnostics()
    assert abs(m[0] - 1.032080772877051e+02) < 1e-11 and abs(j[0] - 1.316643580760437e-01) < 1e-12


def test_half_force_off_negative_control_matches_too():
    c = make_config(1, size=16, half_force=0)
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(30)
    g.step(30)
    assert _pop_rel(o, g, c["mask"]) <= 1e-11


# ------------------------------------------------------------------ config 2: walls + wetting, fp32

@pytest.mark.parametrize("xi", [-0.3, 0.0, 0.3])
def test_cfg2_contact_fp32_100_steps(xi):
    c = make_config(2, size=32, xi=xi)
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(100)
    g.step(100)
    _check_fp32(o, g, c["mask"])


def test_cfg2_contact_fp64():
    c = make_config(2, size=24, xi=-0.3, storage_bits=64)
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(100)
    g.step(100)
    assert _pop_rel(o, g, c["mask"]) <= 1e-10


# ------------------------------------------------------------------ configs 3, 4: open planes

def test_cfg3_drainage_open_fp64():
    c = make_config(3, size=32, storage_bits=64)
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(60)
    g.step(60)
    assert _pop_rel(o, g, c["mask"]) <= 1e-10


def test_cfg3_drainage_open_fp32():
    c = make_config(3, size=48)
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(100)
    g.step(100)
    _check_fp32(o, g, c["mask"])


@pytest.mark.parametrize("G", [3.5, 3.0])
def test_cfg4_imbibition_open_fp32(G):
    c = make_config(4, size=48, G=G)
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(100)
    g.step(100)
    _check_fp32(o, g, c["mask"])
    # Saturation is an integer decision (rho_c > rho_other) taken by the GPU in fp32 and by the
    # oracle in fp64: it may differ only on nodes whose two densities agree to fp32 accuracy.
    mo = o.get_macroscopic()
    fl = c["mask"][8:40] == 0
    a, b = mo["rhoA"][8:40][fl], mo["rhoB"][8:40][fl]
    ambiguous = int((np.abs(a - b) <= 2e-4 * (a + b)).sum())
    for comp in (0, 1):
        dS = abs(o.saturation(comp, 8, 40) - g.saturation(comp, 8, 40))
        assert dS * fl.sum() <= ambiguous + 1e-9, (dS * fl.sum(), ambiguous)


def test_cfg4_imbibition_open_fp64():
    c = make_config(4, size=32, storage_bits=64)
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(60)
    g.step(60)
    assert _pop_rel(o, g, c["mask"]) <= 1e-10


# ------------------------------------------------------------------ config 5: periodic pack + body force

def test_cfg5_spherepack_bodyforce_fp32():
    c = make_config(5, size=64)
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(100)
    g.step(100)
    _check_fp32(o, g, c["mask"])


# ------------------------------------------------------------------ interfaces and edge cases

def test_checkpoint_roundtrip_and_restart():
    c = make_config(3, size=24, storage_bits=64)
    a = Lbm(c["mask"], c["params"])
    a.set_density(c["rhoA"], c["rhoB"])
    a.step(7)
    b = Lbm(c["mask"], c["params"])
    for s in (0, 1):
        b.set_populations(s, a.get_populations(s))
    a.step(5)
    b.step(5)
    for s in (0, 1):
        assert np.array_equal(a.get_populations(s), b.get_populations(s))


def test_step_zero_and_split_steps_are_identical():
    c = make_config(1, size=16)
    a = Lbm(c["mask"], c["params"])
    b = Lbm(c["mask"], c["params"])
    a.set_density(c["rhoA"], c["rhoB"])
    b.set_density(c["rhoA"], c["rhoB"])
    a.step(0)
    a.step(6)
    for n in (1, 2, 3):
        b.step(n)
    for s in (0, 1):
        assert np.array_equal(a.get_populations(s), b.get_populations(s))   # deterministic


def test_single_fluid_voxel_and_single_component():
    mask = np.ones((3, 3, 3), np.uint8)
    mask[1, 1, 1] = 0
    p = default_params(G=3.5, tau=(1.0, 0.8), xi=0.1, storage_bits=64)
    rA = np.where(mask == 0, 0.7, 0.0)
    o, g = _pair(mask, rA, np.zeros_like(rA), p)          # rho_B = 0 everywhere (R4)
    o.step(5)
    g.step(5)
    a, b = g.get_populations(0), o.get_populations(0)
    assert np.max(np.abs(a - b)) <= 1e-15 and np.isfinite(a).all()
    assert np.all(g.get_populations(1) == 0.0)


def test_diagnostics_saturation_trapped_volume_match_oracle():
    rng = np.random.Generator(np.random.PCG64(9))
    shape = (14, 10, 12)
    mask = (rng.uniform(size=shape) < 0.3).astype(np.uint8)
    rA = np.where(mask == 0, rng.uniform(0.0, 1.0, shape), 0.0)
    rB = np.where(mask == 0, rng.uniform(0.0, 1.0, shape), 0.0)
    p = default_params(storage_bits=64)
    o, g = _pair(mask, rA, rB, p)
    m_o, j_o = o.diagnostics()
    m_g, j_g = g.diagnostics()
    assert np.allclose(m_o, m_g, rtol=1e-14) and np.allclose(j_o, j_g, atol=1e-13)
    for comp in (0, 1):
        for z0, z1 in ((0, 14), (3, 9)):
            assert abs(o.saturation(comp, z0, z1) - g.saturation(comp, z0, z1)) < 1e-15
            no, mo = o.trapped_volume(comp, z0, z1)
            ng, mg = g.trapped_volume(comp, z0, z1)
            assert no == ng and abs(mo - mg) < 1e-12 * max(1.0, mo)


def test_set_boundary_changes_inlet_density():
    c = make_config(4, size=24, storage_bits=64)
    g = Lbm(c["mask"], c["params"])
    g.set_density(c["rhoA"], c["rhoB"])
    g.set_boundary(1.05, 0.98)
    g.step(3)
    m = g.get_macroscopic(fields=("rhoA", "rhoB"))
    assert np.allclose(m["rhoB"][0], 1.05, atol=1e-12)      # inlet Dirichlet on B (config 4)
    assert np.allclose(m["rhoA"][-1], 0.98, atol=1e-12)     # outlet Dirichlet on A


@pytest.mark.parametrize("shape", [(1, 1, 64), (1, 40, 41), (3, 1, 5), (2, 2, 2)])
def test_degenerate_box_shapes_fp64(shape):
    """Boxes that are one voxel thick along one or two axes (a voxel is then its own periodic
    neighbour) and a 2x2x2 box (every neighbour pair wraps): fp64, with solids and wetting."""
    rng = np.random.Generator(np.random.PCG64(sum(shape)))
    mask = (rng.uniform(size=shape) < 0.2).astype(np.uint8)
    mask.flat[0] = 0
    rA = np.where(mask == 0, rng.uniform(0.1, 1.0, shape), 0.0)
    rB = np.where(mask == 0, rng.uniform(0.1, 1.0, shape), 0.0)
    p = default_params(G=2.0, tau=(0.9, 1.3), xi=-0.2, accel=(1e-5, 2e-5, -1e-5), storage_bits=64)
    o, g = _pair(mask, rA, rB, p)
    o.step(15)
    g.step(15)
    assert _pop_rel(o, g, mask) <= 1e-10


def test_periodic_box_larger_than_15_bit_offsets_fp64():
    """48^3 periodic box (110 592 nodes): tiles that straddle the z wrap have neighbour-id ranges
    wider than the 15-bit offsets of the tile-relative index and take the int32 fallback rows."""
    c = make_config(1, size=48)
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(8)
    g.step(8)
    assert _pop_rel(o, g, c["mask"]) <= 1e-12


def test_fp32_run_is_deterministic():
    c = make_config(4, size=40)
    res = []
    for _ in range(2):
        g = Lbm(c["mask"], c["params"])
        g.set_density(c["rhoA"], c["rhoB"])
        g.step(50)
        res.append([g.get_populations(s) for s in (0, 1)])
        g.close()
    for s in (0, 1):
        assert np.array_equal(res[0][s], res[1][s])


def test_velocity_inlet_on_component_b_and_extreme_parameters_fp64():
    c = make_config(3, size=24, storage_bits=64, inlet_comp=1, outlet_comp=0, inlet_uz=5e-4,
                    tau=(0.55, 3.5), xi=0.5)
    o, g = _pair(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(40)
    g.step(40)
    assert _pop_rel(o, g, c["mask"]) <= 1e-10


@pytest.mark.parametrize("bits", [64, 32])
def test_execution_options_are_bit_identical(bits):
    """lbm_options select how the step is scheduled -- never what is computed: forward tile order,
    no programmatic dependent launch, no L2 priority for psi, CUDA-graph replay all give the default
    path's populations bit for bit (fp64 and fp32 builds), and those match the oracle."""
    c = make_config(3, size=32, storage_bits=bits)
    sims = {}
    for name, opt in (("prod", None), ("fwd", {"reverse": 0}),
                      ("nopdl", {"pdl": 0}), ("nokeep", {"keep_psi_mb": 0}), ("graph", {"graph": 1}),
                      ("nograph", {"graph": 0})):
        g = Lbm(c["mask"], c["params"], options=opt)
        g.set_density(c["rhoA"], c["rhoB"])
        g.step(30)
        info = g.step_info()
        assert info["pdl"] == (name != "nopdl") and info["reverse"] == (name != "fwd")
        sims[name] = [g.get_populations(s) for s in (0, 1)]
        g.close()
    for name in sims:
        for s in (0, 1):
            assert np.array_equal(sims["prod"][s], sims[name][s]), name
    o = LbmRef(c["mask"], c["params"])
    o.set_density(c["rhoA"], c["rhoB"])
    o.step(30)
    fl = c["mask"] == 0
    for s in (0, 1):
        b = o.get_populations(s)[:, fl]
        assert (np.abs(sims["prod"][s][:, fl] - b) / np.abs(b)).max() < (1e-10 if bits == 64 else 1e-4)


def test_options_are_validated():
    from paper_2207_01534_b200 import LbmError
    c = make_config(1, size=8)
    for bad in ({"graph": 2}, {"pdl": 3}, {"reverse": -1}, {"keep_psi_mb": -5}):
        with pytest.raises(LbmError) as e:
            Lbm(c["mask"], c["params"], options=bad)
        assert e.value.code == -1


def test_context_used_from_several_streams():
    """A context may be stepped and queried from different torch streams in turn (each call is
    ordered after the work the context enqueued before, on whatever stream) and destroyed while
    another stream than the current one holds its last kernels."""
    import torch
    c = make_config(4, size=32, storage_bits=64)
    ref = Lbm(c["mask"], c["params"])
    ref.set_density(c["rhoA"], c["rhoB"])
    ref.step(24)
    want = [ref.get_populations(s) for s in (0, 1)]
    ref.close()
    g = Lbm(c["mask"], c["params"])
    g.set_density(c["rhoA"], c["rhoB"])
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for k in range(6):
        with torch.cuda.stream(s1 if k % 2 == 0 else s2):
            g.step(4)
    got = [g.get_populations(s) for s in (0, 1)]        # on the default stream
    for a, b in zip(want, got):
        assert np.array_equal(a, b)
    with torch.cuda.stream(s1):
        g.step(50)
    g.close()                                            # outside the stream block
    torch.cuda.synchronize()


# ------------------------------------------------------------------ CUDA-graph replay of lbm_step

@pytest.mark.parametrize("k,bits", [(1, 64), (3, 32), (4, 64)])
def test_graph_replay_is_bit_identical_to_host_launches(k, bits):
    """lbm_step through replayed CUDA graphs of 16 steps (the default on launch-bound boxes) gives
    the populations of plain host launches bit for bit: periodic and open boxes, with getters and
    a boundary change (which drops the captured graphs) in between, odd step counts."""
    c = make_config(k, size=32 if k == 1 else 36, storage_bits=bits)
    res = []
    for mode in (0, 1):
        g = Lbm(c["mask"], c["params"], options={"graph": mode})
        g.set_density(c["rhoA"], c["rhoB"])
        g.step(53)                       # 1 direct + 3 graphs + 4 direct
        m1, _ = g.diagnostics()          # applies a pending open-plane fix: next step runs direct
        g.step(37)
        if c["params"]["z_open"]:
            g.set_boundary(1.01 if c["params"]["inlet_kind"] in (1, 3) else 2e-4, 0.995)
        g.step(64)
        g.step(0)
        _, launches = g.last_step_profile()
        assert launches == 0
        g.step(33)
        _, launches = g.last_step_profile()
        assert launches == 33 * (3 if g.num_wall_solid else 2)
        res.append([g.get_populations(s) for s in (0, 1)] + [m1])
        g.close()
    for a, b in zip(res[0], res[1]):
        assert np.array_equal(a, b)


# ------------------------------------------------------------------ the pins of R12 iv and R14, through the C ABI

def test_open_plane_psi_mirror_on_gpu():
    """The oracle pin of reading R12 iv (tests/test_oracle_diag_open.py) through
    lbm_get_macroscopic: with f = w_i rho on a solid-free open box the plane-normal force cancels
    term by term on both open planes, so u_z = 0 there for any density field; fp64 and fp32."""
    rng = np.random.Generator(np.random.PCG64(113))
    shape = (9, 6, 7)
    rA = rng.uniform(0.05, 1.0, shape)
    rB = rng.uniform(0.05, 1.0, shape)
    for bits, zero in ((64, 1e-15), (32, 2e-7)):
        p = default_params(G=3.5, tau=(1.0, 1.0), z_open=1, inlet_kind=1, inlet_comp=0,
                           inlet_rho=1.0, outlet_kind=1, outlet_comp=0, outlet_rho=1.0,
                           storage_bits=bits)
        g = Lbm(np.zeros(shape, np.uint8), p)
        g.set_density(rA, rB)
        m = g.get_macroscopic()
        o = LbmRef(np.zeros(shape, np.uint8), p)
        o.set_density(rA, rB)
        mo = o.get_macroscopic()
        for z in (0, shape[0] - 1):
            assert np.max(np.abs(m["uz"][z])) < zero
            assert np.max(np.abs(m["ux"][z])) > 1e-3
        assert np.max(np.abs(m["uz"][1])) > 1e-3
        for k in ("ux", "uy", "uz"):
            assert np.max(np.abs(m[k] - mo[k])) < (1e-13 if bits == 64 else 1e-6)
        g.close()


def test_saturation_tie_goes_to_component_one_on_gpu():
    """Reading R14 through lbm_saturation and lbm_trapped_volume: identical populations of the two
    components on a node (an exact tie) count for component index 1, never for index 0."""
    rng = np.random.Generator(np.random.PCG64(14))
    shape = (6, 5, 4)
    mask = np.zeros(shape, np.uint8)
    mask[2, 1, 1] = 1
    f = rng.uniform(0.01, 0.1, (19,) + shape)
    clear_a = rng.uniform(size=shape) < 0.3
    clear_b = ~clear_a & (rng.uniform(size=shape) < 0.4)
    gpop = f.copy()
    gpop[:, clear_a] *= 0.5
    gpop[:, clear_b] *= 2.0
    fluid = mask == 0
    tie = fluid & ~clear_a & ~clear_b
    tot = fluid.sum()
    for bits in (64, 32):
        g = Lbm(mask, default_params(storage_bits=bits))
        o = LbmRef(mask, default_params(storage_bits=bits))
        for s in (g, o):
            s.set_populations(0, f)
            s.set_populations(1, gpop)
        assert g.saturation(0) == (fluid & clear_a).sum() / tot == o.saturation(0)
        assert g.saturation(1) == ((fluid & clear_b).sum() + tie.sum()) / tot == o.saturation(1)
        g.set_populations(1, f)
        assert g.saturation(0) == 0.0 and g.saturation(1) == 1.0
        assert g.trapped_volume(0)[0] == 0 and g.trapped_volume(1)[0] == 0
        g.close()


def test_get_macroscopic_validates_output_arrays():
    c = make_config(1, size=8)
    g = Lbm(c["mask"], c["params"])
    g.set_density(c["rhoA"], c["rhoB"])
    for bad in (np.empty(c["mask"].shape, np.float32), np.empty((8, 8, 9)),
                np.empty((8, 8, 16))[:, :, ::2]):
        with pytest.raises(ValueError):
            g.get_macroscopic(fields=("rhoA",), out={"rhoA": bad})
    g.close()


def test_neem_extrapolates_the_collision_operators_nonequilibrium_part_on_gpu():
    """The oracle pin of reading R12 iii (tests/test_oracle_neem.py), through the C ABI in fp64: on
    a force-free state with different component momenta, the plane populations NEEM writes equal
    (rho_b / rho(x_f)) f^eq(x_f) + f(x_f) - f^eq(x_f) with f^eq read off the library's own collision
    step of a z-periodic copy: f^eq = f - tau (f - f*)."""
    W = np.array([1 / 3] + [1 / 18] * 6 + [1 / 36] * 12)
    E = np.array([(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1),
                  (1, 1, 0), (-1, 1, 0), (1, -1, 0), (-1, -1, 0), (1, 0, 1), (-1, 0, 1), (1, 0, -1),
                  (-1, 0, -1), (0, 1, 1), (0, -1, 1), (0, 1, -1), (0, -1, -1)])
    shape = (8, 4, 5)
    nz, tau = shape[0], 0.8
    mask = np.zeros(shape, np.uint8)
    rng = np.random.Generator(np.random.PCG64(12))
    f0 = []
    for s in range(2):
        rho = rng.uniform(0.3, 1.0, shape)
        f0.append(np.stack([W[i] * rho * (1.0 + 0.2 * rng.uniform(-1, 1, shape)) for i in range(19)]))
    f0[0] = f0[0] * (1.0 + 0.05 * E[:, 2].reshape(19, 1, 1, 1))
    f0[1] = f0[1] * (1.0 - 0.05 * E[:, 0].reshape(19, 1, 1, 1))
    p = default_params(G=0.0, tau=(tau, tau), xi=0.0, z_open=1, inlet_kind=1, inlet_comp=0,
                       inlet_rho=1.03, outlet_kind=1, outlet_comp=1, outlet_rho=0.97,
                       storage_bits=64)
    g = Lbm(mask, p)
    for s in range(2):
        g.set_populations(s, f0[s])
    g.step(1)
    f = [g.get_populations(s) for s in range(2)]
    g.close()
    q = Lbm(mask, dict(p, z_open=0))
    for s in range(2):
        q.set_populations(s, f[s])
    q.step(1)
    h = [q.get_populations(s) for s in range(2)]
    q.close()
    for zb, zf, dc, rho_b in ((0, 1, 0, 1.03), (nz - 1, nz - 2, 1, 0.97)):
        fstar = np.empty_like(f[dc][:, zf])
        for i in range(19):
            fstar[i] = np.roll(h[dc][i], (-E[i][2], -E[i][1], -E[i][0]), (0, 1, 2))[zf]
        feq = f[dc][:, zf] - tau * (f[dc][:, zf] - fstar)
        rho_f = f[dc][:, zf].sum(0)
        want = (rho_b / rho_f) * feq + f[dc][:, zf] - feq
        assert np.abs(f[dc][:, zb] - want).max() < 1e-14


def test_getters_decode_the_tile_index_including_wide_tiles():
    """lbm_get_macroscopic and the connected-component query read neighbour ids through the same
    16-bit rows as the fused pass (no separate int32 table); tiles whose offsets do not fit 15 bits
    ("wide": periodic wraps inside a tile) read the compact wide-tile table.  Forces, hence
    velocities, see every neighbour id: fp64 fields against the oracle on boxes made of wide
    tiles, after a few steps."""
    rng = np.random.Generator(np.random.PCG64(77))
    wide_seen = 0
    for shape, solid in (((1, 40, 41), 0.2), ((3, 1, 5), 0.0), ((2, 2, 2), 0.0), ((40, 40, 40), 0.35),
                         ((6, 300, 7), 0.3)):
        mask = (rng.uniform(size=shape) < solid).astype(np.uint8)
        rA = rng.uniform(0.1, 1.0, shape)
        rB = rng.uniform(0.1, 1.0, shape)
        p = default_params(G=1.5, tau=(1.0, 0.8), xi=0.2, accel=(1e-5, 0, 2e-5), storage_bits=64)
        o, g = LbmRef(mask, p), Lbm(mask, p)
        for s in (o, g):
            s.set_density(rA, rB)
            s.step(3)
        wide_seen += g.step_info()["wide_tiles"]
        mo, mg = o.get_macroscopic(), g.get_macroscopic()
        for k in ("rhoA", "rhoB", "ux", "uy", "uz", "P"):
            assert np.max(np.abs(mg[k] - mo[k])) < 1e-12, (shape, k)
        for comp in (0, 1):
            assert g.trapped_volume(comp)[0] == o.trapped_volume(comp)[0]
        g.close()
    assert wide_seen > 0
