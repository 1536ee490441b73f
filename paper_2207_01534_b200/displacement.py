"""The two displacement runs BASELINE.json names, driven through the C ABI and reported as the
paper reports its own (Sec. 4): saturation against time, and the trapped volume of the displaced
phase at the end.

  config 3  drainage: non-wetting A injected at constant velocity 1e-4 through the z = 0 inlet
            into a 128^3 sphere pack filled with wetting B, constant-pressure outlet; 20 000 steps;
            S_B(t) (S_w = nodes occupied by water / pore nodes).
  config 4  imbibition: wetting B displaces A in the 256^3 sandstone-like mask from a pressure
            inlet to a pressure outlet, viscosity ratio A:B = 10; 10 000 steps at G = 3.5 and at
            G = 3.0 (reading R26: the paper's surface-tension knob is G, L105); S_B(t) and the
            trapped volume of A (residual non-wetting saturation).

Everything numerical happens in the library (`lbm_step`, `lbm_saturation`, `lbm_trapped_volume`,
`lbm_mean_pressure`, `lbm_diagnostics`); this module sequences the calls and prints markdown.

    python -m paper_2207_01534_b200.displacement --config 3
    python -m paper_2207_01534_b200.displacement --config 4 --G 3.5
"""
import time


def displacement_run(sim, steps, every, *, invading_comp, layers, on_sample=None):
    """Step `sim` (an initialised z-open `Lbm`) `steps` times, sampling every `every` steps.
    Returns (samples, final) where a sample is (step, S_invading over the rock, P_in - P_out by
    reading R28) and final = dict(trapped nodes and mass of the displaced component in the rock
    (reading R15), its saturation, the masses).  Saturations exclude the `layers` reservoir
    layers at either end (reading R29)."""
    nz = sim.shape[0]
    z0, z1 = layers, nz - layers
    displaced = 1 - invading_comp

    def sample(k):
        s = sim.saturation(invading_comp, z0, z1)
        pc = sim.mean_pressure(0, 1) - sim.mean_pressure(nz - 1, nz)
        if on_sample is not None:
            on_sample(k, s, pc)
        return (k, s, pc)

    samples = [sample(0)]
    done = 0
    while done < steps:
        n = min(every, steps - done)
        sim.step(n)
        done += n
        samples.append(sample(done))
    nodes, mass = sim.trapped_volume(displaced, z0, z1)
    m, _ = sim.diagnostics()                      # also the non-finite check
    final = dict(trapped_nodes=int(nodes), trapped_mass=float(mass),
                 displaced_saturation=sim.saturation(displaced, z0, z1),
                 mass=(float(m[0]), float(m[1])))
    return samples, final


def _main(argv=None):
    import argparse

    from workloads import make_config

    from .lbm import Lbm

    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--config", type=int, required=True, choices=(3, 4))
    ap.add_argument("--size", type=int, default=None)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--every", type=int, default=1000)
    ap.add_argument("--G", type=float, default=3.5, help="config 4 only: 3.5 or 3.0")
    a = ap.parse_args(argv)
    c = make_config(a.config, size=a.size, **({"G": a.G} if a.config == 4 else {}))
    p = c["params"]
    steps = a.steps if a.steps is not None else c["steps"]
    sim = Lbm(c["mask"], p)
    sim.set_density(c["rhoA"], c["rhoB"])
    inv = p["inlet_comp"]
    name = "AB"
    t0 = time.perf_counter()
    samples, final = displacement_run(sim, steps, a.every, invading_comp=inv, layers=8)
    sim.sync()
    wall = time.perf_counter() - t0
    pore = int((c["mask"][8:-8] == 0).sum())
    print(f"{c['name']}: shape {c['mask'].shape}, N_f = {sim.num_fluid} ({pore} in the rock), "
          f"G = {p['G']}, tau = {tuple(p['tau'])}, xi = {p['xi']}, invading {name[inv]} "
          f"(inlet kind {p['inlet_kind']}), displaced {name[1 - inv]}; {steps} steps + "
          f"{len(samples)} x 3 queries in {wall:.2f} s = "
          f"{steps * sim.num_fluid / wall / 1e6:.0f} MLUPS including the queries")
    print(f"| step | S_{name[inv]} (rock) | P_in - P_out |")
    print("|---|---|---|")
    for k, s, pc in samples:
        print(f"| {k} | {s:.5f} | {pc:+.6f} |")
    print(f"end: S_{name[1 - inv]} = {final['displaced_saturation']:.5f}; trapped {name[1 - inv]} "
          f"(clusters touching neither end plane, reading R15): {final['trapped_nodes']} nodes = "
          f"{final['trapped_nodes'] / pore:.5f} of the pore space, mass {final['trapped_mass']:.3f}; "
          f"total mass A {final['mass'][0]:.3f}, B {final['mass'][1]:.3f}")
    sim.close()


if __name__ == "__main__":
    _main()
