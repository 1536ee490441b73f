"""GPU parity of the Zou-He variant of the open-plane condition (reading R31;
inlet_kind / outlet_kind 3, 4) against the oracle, element by element."""
import numpy as np
import pytest

from oracle import LbmRef
from paper_2207_01534_b200 import Lbm
from workloads import make_config

pytestmark = pytest.mark.gpu


def _pair(c, **over):
    p = dict(c["params"])
    p.update(over)
    o, g = LbmRef(c["mask"], p), Lbm(c["mask"], p)
    o.set_density(c["rhoA"], c["rhoB"])
    g.set_density(c["rhoA"], c["rhoB"])
    return o, g, p


def _pop_rel(o, g, mask):
    fl = mask == 0
    worst = 0.0
    for s in (0, 1):
        a, b = g.get_populations(s), o.get_populations(s)
        assert np.all(a[:, ~fl] == 0.0)
        worst = max(worst, float((np.abs(a[:, fl] - b[:, fl]) / np.abs(b[:, fl])).max()))
    return worst


@pytest.mark.parametrize("cfg,size,inlet_kind", [(3, 40, 4), (3, 40, 3), (4, 40, 3), (4, 36, 4)])
def test_zou_he_fp64_every_population_200_steps(cfg, size, inlet_kind):
    c = make_config(cfg, size=size, storage_bits=64)
    o, g, p = _pair(c, inlet_kind=inlet_kind, outlet_kind=3, inlet_uz=1e-4)
    o.step(200)
    g.step(200)
    assert _pop_rel(o, g, c["mask"]) <= 1e-10
    m_o, j_o = o.diagnostics()
    m_g, j_g = g.diagnostics()
    assert np.allclose(m_o, m_g, rtol=1e-12) and np.allclose(j_o, j_g, atol=1e-10)


@pytest.mark.parametrize("cfg,inlet_kind", [(3, 4), (4, 3)])
def test_zou_he_fp32_100_steps(cfg, inlet_kind):
    c = make_config(cfg, size=48)
    assert c["params"]["storage_bits"] == 32
    o, g, p = _pair(c, inlet_kind=inlet_kind, outlet_kind=3, inlet_uz=1e-4)
    o.step(100)
    g.step(100)
    fl = c["mask"] == 0
    mo, mg = o.get_macroscopic(), g.get_macroscopic()
    for k in ("rhoA", "rhoB"):
        assert (np.abs(mg[k][fl] - mo[k][fl]) / np.abs(mo[k][fl])).max() <= 1e-4
    uo = np.stack([mo[k][fl] for k in ("ux", "uy", "uz")])
    ug = np.stack([mg[k][fl] for k in ("ux", "uy", "uz")])
    assert np.abs(ug - uo).max() <= 1e-4 * np.abs(uo).max()
    m_o, _ = o.diagnostics()
    m_g, _ = g.diagnostics()
    assert np.max(np.abs(m_g - m_o) / m_o) <= 1e-6


def test_zou_he_mixed_with_neem_and_boundary_ramp():
    """NEEM inlet with a Zou-He outlet (and the other way round), with the imposed values changed
    between steps through lbm_set_boundary."""
    c = make_config(4, size=32, storage_bits=64)
    for ik, ok in ((1, 3), (3, 1), (4, 1), (2, 3)):
        o, g, p = _pair(c, inlet_kind=ik, outlet_kind=ok, inlet_uz=2e-4)
        for val in (1.01, 1.03) if ik in (1, 3) else (2e-4, 5e-4):
            o.set_boundary(val, 0.99)
            g.set_boundary(val, 0.99)
            o.step(30)
            g.step(30)
        assert _pop_rel(o, g, c["mask"]) <= 1e-10, (ik, ok)


def test_zou_he_properties_through_the_cuda_path():
    """What defines the condition, read back from the GPU state: imposed density met, no
    transverse momentum of the Dirichlet component on its plane; imposed velocity met."""
    c = make_config(4, size=32, storage_bits=64)
    o, g, p = _pair(c, inlet_kind=3, outlet_kind=3, inlet_rho=1.04, outlet_rho=0.98)
    g.step(25)
    from oracle import lattice
    _, E, _ = lattice()
    fin = g.get_populations(p["inlet_comp"])[:, 0]
    fout = g.get_populations(p["outlet_comp"])[:, -1]
    assert np.max(np.abs(fin.sum(0) - 1.04)) < 1e-13 and np.max(np.abs(fout.sum(0) - 0.98)) < 1e-13
    for f in (fin, fout):
        for a in (0, 1):
            assert np.max(np.abs(np.tensordot(E[:, a].astype(float), f, axes=(0, 0)))) < 1e-14
    o, g, p = _pair(c, inlet_kind=4, outlet_kind=3, inlet_uz=3e-4)
    g.step(25)
    fin = g.get_populations(p["inlet_comp"])[:, 0]
    uz = np.tensordot(E[:, 2].astype(float), fin, axes=(0, 0)) / fin.sum(0)
    assert np.max(np.abs(uz - 3e-4)) < 1e-14


def test_zou_he_all_step_paths_agree():
    """Forward tile order, graph replay and plain launches run the same arithmetic as the default
    path (bit-identical).  All share the open-plane code."""
    c = make_config(4, size=40, storage_bits=64)
    p = dict(c["params"], inlet_kind=3, outlet_kind=3)

    def run(opt=None):
        g = Lbm(c["mask"], p, options=opt)
        g.set_density(c["rhoA"], c["rhoB"])
        g.step(37)
        f = [g.get_populations(s) for s in (0, 1)]
        g.close()
        return f

    base = run()
    for opt in ({"reverse": 0}, {"graph": 1}, {"graph": 0, "pdl": 0}):
        other = run(opt)
        for s in (0, 1):
            assert np.array_equal(base[s], other[s]), opt


def test_bad_kinds_are_rejected():
    c = make_config(4, size=24)
    for bad in (dict(inlet_kind=0), dict(inlet_kind=5), dict(outlet_kind=2), dict(outlet_kind=4)):
        with pytest.raises(RuntimeError):
            Lbm(c["mask"], dict(c["params"], **bad))
