"""Host logic of the drainage protocol driver (paper_2207_01534_b200/drainage.py) on a scripted
stand-in for the simulation object: staging, plateau detection (reading R30), the planes and
z-ranges it queries (R28, R29).  No GPU, no oracle."""
import pytest

from paper_2207_01534_b200.drainage import primary_drainage


class _Scripted:
    """S_w relaxes geometrically towards a target that depends on the inlet density."""

    def __init__(self, nz=40):
        self.shape = (nz, 4, 4)
        self.s = 1.0
        self.rho_in = 1.0
        self.rho_out = 1.0
        self.calls = []

    def set_boundary(self, a, b):
        self.rho_in, self.rho_out = a, b
        self.calls.append(("set_boundary", a, b))

    def step(self, n):
        target = max(0.2, 1.0 - 10.0 * (self.rho_in - 1.0))
        for _ in range(n // 100):
            self.s += 0.5 * (target - self.s)
        self.calls.append(("step", n))

    def saturation(self, comp, z0, z1):
        self.calls.append(("saturation", comp, z0, z1))
        return self.s

    def mean_pressure(self, z0, z1):
        self.calls.append(("mean_pressure", z0, z1))
        return (self.rho_in if z0 == 0 else self.rho_out) / 3.0

    def trapped_volume(self, comp, z0, z1):
        self.calls.append(("trapped_volume", comp, z0, z1))
        return 7, 6.5


def test_stages_settle_and_record_the_curve():
    sim = _Scripted()
    seen = []
    curve = primary_drainage(sim, [1.0, 1.03, 1.06, 1.2], 1.0, defending_comp=0, layers=8,
                             check_every=100, plateau_tol=1e-3, max_steps_per_stage=5000,
                             on_check=lambda k, n, s: seen.append((k, n, s)))
    assert [p.stage for p in curve] == [0, 1, 2, 3]
    assert curve[0].steps == 100 and curve[0].settled and curve[0].S_w == 1.0
    assert all(p.settled for p in curve)
    assert curve[1].S_w == pytest.approx(0.7, abs=2e-3)
    assert curve[2].S_w == pytest.approx(0.4, abs=2e-3)
    assert curve[3].S_w == pytest.approx(0.2, abs=2e-3)          # irreducible saturation
    for p, rho in zip(curve, [1.0, 1.03, 1.06, 1.2]):
        assert p.P_c == pytest.approx((rho - 1.0) / 3.0) and p.inlet_rho == rho
        assert p.trapped_nodes == 7 and p.trapped_mass == 6.5
    # halving the distance per check: |dS| < 1e-3 first holds at the 9th check of stage 1
    assert curve[1].steps == 900
    assert [s for s in seen if s[0] == 1][-1][1] == 900
    # what it asked the library for: rock region only, boundary planes for the pressures
    assert ("saturation", 0, 8, 32) in sim.calls and ("trapped_volume", 0, 8, 32) in sim.calls
    assert ("mean_pressure", 0, 1) in sim.calls and ("mean_pressure", 39, 40) in sim.calls
    assert [c for c in sim.calls if c[0] == "set_boundary"] == [
        ("set_boundary", r, 1.0) for r in (1.0, 1.03, 1.06, 1.2)]


def test_stage_stops_at_max_steps_when_not_settled():
    sim = _Scripted()
    curve = primary_drainage(sim, [1.05], 1.0, defending_comp=0, layers=8, check_every=100,
                             plateau_tol=1e-9, max_steps_per_stage=350)
    assert curve[0].steps == 300 and not curve[0].settled     # never oversteps the budget


@pytest.mark.parametrize("kw", [dict(layers=20), dict(layers=-1), dict(check_every=0),
                                dict(check_every=200, max_steps_per_stage=100)])
def test_bad_arguments(kw):
    args = dict(defending_comp=0, layers=8, check_every=100, max_steps_per_stage=1000)
    args.update(kw)
    with pytest.raises(ValueError):
        primary_drainage(_Scripted(), [1.0], 1.0, **args)


def test_displacement_run_sequences_queries():
    """paper_2207_01534_b200/displacement.py: samples at step 0 and after every block, the last
    block shortened to the step count; saturations over the rock only (R29), P_c from the two end
    planes (R28), trapped volume of the DISPLACED component (R15)."""
    from paper_2207_01534_b200.displacement import displacement_run

    class S(_Scripted):
        def diagnostics(self):
            return (1.0, 2.0), (0.0, 0.0, 0.0)

    sim = S(nz=40)
    seen = []
    samples, final = displacement_run(sim, 2500, 1000, invading_comp=1, layers=8,
                                      on_sample=lambda k, s, pc: seen.append(k))
    assert [k for k, _, _ in samples] == [0, 1000, 2000, 2500] == seen
    assert [c for c in sim.calls if c[0] == "step"] == [("step", 1000), ("step", 1000), ("step", 500)]
    assert all(c[2:] == (8, 32) for c in sim.calls if c[0] == "saturation")
    assert ("mean_pressure", 0, 1) in sim.calls and ("mean_pressure", 39, 40) in sim.calls
    assert ("trapped_volume", 0, 8, 32) in sim.calls
    assert final["trapped_nodes"] == 7 and final["mass"] == (1.0, 2.0)
