"""GPU parity of the pieces the drainage protocol of Sec. 4 adds to the hot
path: the plane-mean pressure query, and the whole staged protocol against the same sequence of
calls made on the oracle."""
import numpy as np
import pytest

from oracle import LbmRef
from paper_2207_01534_b200 import Lbm
from paper_2207_01534_b200.drainage import primary_drainage
from workloads import make_config

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("bits,tol", [(64, 1e-13), (32, 2e-6)])
def test_mean_pressure_matches_oracle_field(bits, tol):
    c = make_config(4, size=40, storage_bits=bits)
    mask = c["mask"]
    o, g = LbmRef(mask, c["params"]), Lbm(mask, c["params"])
    o.set_density(c["rhoA"], c["rhoB"])
    g.set_density(c["rhoA"], c["rhoB"])
    o.step(25)
    g.step(25)
    P = o.get_macroscopic()["P"]
    fl = mask == 0
    nz = mask.shape[0]
    for z0, z1 in ((0, 1), (nz - 1, nz), (0, nz), (7, 23), (20, 21)):
        want = P[z0:z1][fl[z0:z1]].mean()          # Eq. (12) averaged over the fluid nodes
        got = g.mean_pressure(z0, z1)
        assert abs(got - want) <= tol * abs(want), (z0, z1, got, want)
    assert g.mean_pressure(0, nz) == g.mean_pressure(0, nz)       # fixed-order reduction


def test_mean_pressure_rejects_bad_ranges():
    c = make_config(2, size=16)
    g = Lbm(c["mask"], c["params"])
    g.set_density(c["rhoA"], c["rhoB"])
    nz = c["mask"].shape[0]
    for z0, z1 in ((-1, 3), (3, 3), (5, 2), (0, nz + 1)):
        with pytest.raises(RuntimeError):
            g.mean_pressure(z0, z1)
    solid_planes = np.nonzero(c["mask"].reshape(nz, -1).all(axis=1))[0]
    if len(solid_planes):                                          # config 2: the channel walls
        z = int(solid_planes[0])
        with pytest.raises(RuntimeError):
            g.mean_pressure(z, z + 1)


def test_staged_drainage_protocol_matches_oracle():
    """Three pressure stages on a 40^3 rock, fp64: the CUDA path driven by
    `primary_drainage` against the oracle driven by the same sequence written out here."""
    c = make_config(4, size=40, storage_bits=64)
    mask, p = c["mask"], c["params"]
    layers, nz = 8, mask.shape[0]
    stages, rho_out = [1.0, 1.04, 1.08], 1.0
    check_every, tol, max_steps = 60, 2e-4, 240
    defending = p["outlet_comp"]

    g = Lbm(mask, p)
    g.set_density(c["rhoA"], c["rhoB"])
    curve = primary_drainage(g, stages, rho_out, defending_comp=defending, layers=layers,
                             check_every=check_every, plateau_tol=tol,
                             max_steps_per_stage=max_steps)

    o = LbmRef(mask, p)
    o.set_density(c["rhoA"], c["rhoB"])
    fl = mask == 0
    s_prev = o.saturation(defending, layers, nz - layers)
    for k, rho_in in enumerate(stages):
        o.set_boundary(rho_in, rho_out)
        steps, settled = 0, False
        while steps + check_every <= max_steps and not settled:
            o.step(check_every)
            steps += check_every
            s = o.saturation(defending, layers, nz - layers)
            settled = abs(s - s_prev) < tol
            s_prev = s
        P = o.get_macroscopic()["P"]
        p_in, p_out = P[0][fl[0]].mean(), P[-1][fl[-1]].mean()
        nodes, mass = o.trapped_volume(defending, layers, nz - layers)
        pt = curve[k]
        assert (pt.steps, pt.settled) == (steps, settled), k
        assert pt.S_w == s_prev, k
        assert abs(pt.P_c - (p_in - p_out)) <= 1e-10 * max(abs(p_in), 1e-3), k
        assert pt.trapped_nodes == nodes and abs(pt.trapped_mass - mass) <= 1e-9 * max(1.0, mass)
    # the ramp does something: the inlet pressure follows the imposed density
    assert curve[2].P_in > curve[1].P_in > curve[0].P_in
    assert curve[2].P_c > 0.0


def test_staged_drainage_protocol_on_slabs_matches_unsharded():
    """The same protocol driven on the box cut into 3 z-slabs (SlabLbm has the calls
    `primary_drainage` makes): stage lengths, S_w and trapped node counts identical to the
    unsharded run, pressures and trapped mass to rounding of the per-slab sums."""
    from paper_2207_01534_b200.slab import SlabLbm
    c = make_config(4, size=40, storage_bits=64)
    mask, p = c["mask"], c["params"]
    kw = dict(defending_comp=p["outlet_comp"], layers=8, check_every=60, plateau_tol=2e-4,
              max_steps_per_stage=240)
    stages = [1.0, 1.04, 1.08]
    curves = []
    for make in (lambda: Lbm(mask, p), lambda: SlabLbm(mask, p, parts=3)):
        sim = make()
        sim.set_density(c["rhoA"], c["rhoB"])
        curves.append(primary_drainage(sim, stages, 1.0, **kw))
        sim.close()
    for a, b in zip(*curves):
        assert (a.steps, a.settled, a.trapped_nodes) == (b.steps, b.settled, b.trapped_nodes)
        assert abs(a.S_w - b.S_w) < 1e-12
        assert abs(a.P_in - b.P_in) < 1e-12 and abs(a.P_out - b.P_out) < 1e-12
        assert abs(a.trapped_mass - b.trapped_mass) <= 1e-10 * max(1.0, a.trapped_mass)
