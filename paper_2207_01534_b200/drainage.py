"""Primary-drainage protocol of Sec. 4 (Fig. 5 and Fig. 8), driven through the
C ABI: the inlet density of the invading component is raised in stages while the outlet density
of the defending component is kept constant; after each stage has settled, one point of the
capillary pressure - saturation curve is recorded.

Everything numerical happens in the library (`lbm_set_boundary`, `lbm_step`, `lbm_saturation`,
`lbm_mean_pressure`, `lbm_trapped_volume`); this module only sequences the calls.

Readings (the paper gives the protocol in words only, R28-R30):
  R28  P_in, P_out are the means of Eq. (12) over the fluid nodes of the boundary planes z = 0 and
       z = nz-1 ("the first (last) slice of the inlet (outlet) layer is used to implement the
       boundary conditions", L219; "P_c = P_in - P_out", L223).
  R29  S_w is the saturation (reading R14) of the defending component over the rock, i.e. without
       the `layers` reservoir layers at either end (L219: they "represent pure reservoir fluid").
  R30  a stage has settled when S_w changed by less than `plateau_tol` over `check_every` steps
       (the paper does not state its criterion), or after `max_steps_per_stage`.
"""
from dataclasses import dataclass, asdict


@dataclass
class DrainagePoint:
    stage: int
    inlet_rho: float
    steps: int            # steps spent in this stage
    settled: bool         # False: stopped by max_steps_per_stage
    P_in: float
    P_out: float
    P_c: float
    S_w: float
    trapped_nodes: int    # defending-phase nodes cut off from both ends (reading R15), in the rock
    trapped_mass: float

    def as_dict(self):
        return asdict(self)


def primary_drainage(sim, inlet_rho_stages, outlet_rho, *, defending_comp, layers,
                     check_every=500, plateau_tol=1e-4, max_steps_per_stage=20000,
                     on_check=None):
    """Run the staged protocol on `sim` (a `paper_2207_01534_b200.Lbm` created with z_open=1 and
    density Dirichlet planes, already initialised with `set_density`).  Returns one
    `DrainagePoint` per entry of `inlet_rho_stages`.

    on_check(stage, steps_in_stage, S_w), if given, is called after every saturation check."""
    nz = sim.shape[0]
    if not 0 <= layers < nz // 2:
        raise ValueError("layers must leave a rock region")
    if check_every <= 0 or max_steps_per_stage < check_every:
        raise ValueError("need 0 < check_every <= max_steps_per_stage")
    z0, z1 = layers, nz - layers
    curve = []
    s_prev = sim.saturation(defending_comp, z0, z1)
    for k, rho_in in enumerate(inlet_rho_stages):
        sim.set_boundary(float(rho_in), float(outlet_rho))
        steps, settled = 0, False
        while steps + check_every <= max_steps_per_stage:
            sim.step(check_every)
            steps += check_every
            s = sim.saturation(defending_comp, z0, z1)
            if on_check is not None:
                on_check(k, steps, s)
            settled = abs(s - s_prev) < plateau_tol
            s_prev = s
            if settled:
                break
        p_in = sim.mean_pressure(0, 1)
        p_out = sim.mean_pressure(nz - 1, nz)
        nodes, mass = sim.trapped_volume(defending_comp, z0, z1)
        curve.append(DrainagePoint(k, float(rho_in), steps, settled, p_in, p_out, p_in - p_out,
                                   s_prev, int(nodes), float(mass)))
    return curve


def _main(argv=None):
    """python -m paper_2207_01534_b200.drainage --config 4 --size 128 ...
    Runs the protocol on one of the seeded synthetic rocks (workloads/generators.py) and prints
    the P_c - S_w table as markdown."""
    import argparse
    import time

    from workloads import make_config

    from .lbm import Lbm

    ap = argparse.ArgumentParser(description=_main.__doc__)
    ap.add_argument("--config", type=int, default=4, choices=(3, 4, 5))
    ap.add_argument("--size", type=int, default=None)
    ap.add_argument("--xi", type=float, default=0.2,
                    help="wettability; the defending component must be the wetting one for drainage")
    ap.add_argument("--tau", type=float, nargs=2, default=None, metavar=("TAU_A", "TAU_B"),
                    help="relaxation times (default: the config's)")
    ap.add_argument("--rho-in", type=float, nargs=3, default=(1.0, 1.10, 0.01),
                    metavar=("FIRST", "LAST", "STEP"))
    ap.add_argument("--rho-out", type=float, default=1.0)
    ap.add_argument("--layers", type=int, default=8)
    ap.add_argument("--check-every", type=int, default=1000)
    ap.add_argument("--plateau-tol", type=float, default=5e-4)
    ap.add_argument("--max-steps-per-stage", type=int, default=20000)
    a = ap.parse_args(argv)

    over = dict(xi=a.xi, inlet_kind=1, outlet_kind=1)
    if a.tau is not None:
        over["tau"] = tuple(a.tau)
    c = make_config(a.config, size=a.size, **over)
    p = c["params"]
    sim = Lbm(c["mask"], p)
    sim.set_density(c["rhoA"], c["rhoB"])
    first, last, step = a.rho_in
    stages = [first + k * step for k in range(int(round((last - first) / step)) + 1)]
    t0 = time.perf_counter()
    curve = primary_drainage(sim, stages, a.rho_out, defending_comp=p["outlet_comp"],
                             layers=a.layers, check_every=a.check_every,
                             plateau_tol=a.plateau_tol,
                             max_steps_per_stage=a.max_steps_per_stage)
    wall = time.perf_counter() - t0
    total = sum(pt.steps for pt in curve)
    print(f"config {a.config}, shape {c['mask'].shape}, N_f = {sim.num_fluid}, xi = {a.xi}, "
          f"tau = {tuple(p['tau'])}, G = {p['G']}, invading component {p['inlet_comp']}, "
          f"defending {p['outlet_comp']}; {total} steps in {wall:.1f} s "
          f"({total * sim.num_fluid / wall / 1e6:.0f} MLUPS including the queries)")
    print("| stage | rho_in | steps | settled | P_in | P_out | P_c | S_w | trapped nodes |")
    print("|---|---|---|---|---|---|---|---|---|")
    for pt in curve:
        print(f"| {pt.stage} | {pt.inlet_rho:.3f} | {pt.steps} | {'yes' if pt.settled else 'no'} | "
              f"{pt.P_in:.5f} | {pt.P_out:.5f} | {pt.P_c:.5f} | {pt.S_w:.4f} | {pt.trapped_nodes} |")


if __name__ == "__main__":
    _main()
