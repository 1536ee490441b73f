"""Pins of the CPU oracle, part 1: what the mathematics fixes (SURVEY.md §8c "pins").

None of these compares the oracle with itself through a retyped formula: they are lattice
identities, conservation laws, symmetries of the lattice, and an independently produced
worked example.
"""
import itertools
import os

import numpy as np
import pytest

from oracle import LbmRef, lattice
from workloads import default_params, make_config

HERE = os.path.dirname(os.path.abspath(__file__))


def _run(mask, rhoA, rhoB, params, steps):
    o = LbmRef(mask, params)
    o.set_density(rhoA, rhoB)
    o.step(steps)
    return o


# ------------------------------------------------------------------ lattice (reading R1)

def test_lattice_identities():
    """D3Q19 isotropy: sum w = 1, sum w e = 0, sum w e e = I/3, 4th-order isotropic tensor
    (c_s^2 = 1/3; weights PAPER.md L67)."""
    w, e, opp = lattice()
    assert abs(w.sum() - 1.0) < 1e-15
    assert np.allclose(w @ e, 0.0, atol=1e-16)
    assert np.allclose(np.einsum("i,ia,ib->ab", w, e, e), np.eye(3) / 3.0, atol=1e-15)
    d = np.eye(3)
    iso = (np.einsum("ab,cd->abcd", d, d) + np.einsum("ac,bd->abcd", d, d)
           + np.einsum("ad,bc->abcd", d, d)) / 9.0
    assert np.allclose(np.einsum("i,ia,ib,ic,id->abcd", w, e, e, e, e), iso, atol=1e-15)
    assert np.allclose(np.einsum("i,ia,ib,ic->abc", w, e, e, e), 0.0, atol=1e-16)
    # 19 distinct vectors: rest, 6 axis (w=1/18), 12 face diagonals (w=1/36)
    assert len({tuple(v) for v in e}) == 19
    n2 = (e * e).sum(1)
    assert np.allclose(w[n2 == 0], 1 / 3) and np.allclose(w[n2 == 1], 1 / 18)
    assert np.allclose(w[n2 == 2], 1 / 36) and sorted(np.bincount(n2)) == [1, 6, 12]
    with open(os.path.join(HERE, "golden", "paper_values.txt")) as fh:
        printed = [l.split("#")[0].split()[1:] for l in fh if l.startswith("weights")][0]
    assert np.allclose(sorted(set(np.round(w, 15)), reverse=True), [float(v) for v in printed])
    for i in range(19):
        assert np.array_equal(e[opp[i]], -e[i])
    # what PAPER.md L152-154 and L113 reveal about the numbering (flow axis = z here)
    assert sorted(np.nonzero(e[:, 2] == 1)[0]) == [5, 11, 12, 15, 16]


# ------------------------------------------------------------------ invariants

def test_uniform_state_is_stationary():
    n = 6
    mask = np.zeros((n, n, n), np.uint8)
    p = default_params(G=3.5, tau=(1.0, 0.7))
    o = LbmRef(mask, p)
    o.set_density(np.full(mask.shape, 0.8), np.full(mask.shape, 0.3))
    f0 = [o.get_populations(s) for s in (0, 1)]
    o.step(25)
    for s in (0, 1):
        assert np.max(np.abs(o.get_populations(s) - f0[s])) < 1e-15
    m = o.get_macroscopic()
    assert np.max(np.abs(m["ux"])) < 1e-15 and np.max(np.abs(m["uz"])) < 1e-15
    # Eq. (12) with reading R13: P = (rho1+rho2)/3 + (G/3) rho1 rho2
    assert np.allclose(m["P"], 1.1 / 3 + 3.5 / 3 * 0.8 * 0.3, atol=1e-14)


def test_mass_and_momentum_conservation_periodic_no_solids():
    """Config 1 (reduced steps): each component's mass and the total bare momentum are
    invariants on a periodic solid-free box (sum_i feq = rho, sum_i S_i = 0, Eq. 11 pairwise
    antisymmetric)."""
    c = make_config(1)
    o = LbmRef(c["mask"], c["params"])
    o.set_density(c["rhoA"], c["rhoB"])
    m0, j0 = o.diagnostics()
    assert np.allclose(m0, [c["rhoA"].sum(), c["rhoB"].sum()], rtol=1e-14)
    o.step(40)
    m1, j1 = o.diagnostics()
    assert np.max(np.abs(m1 - m0) / m0) < 1e-13
    assert np.max(np.abs(j1 - j0)) < 1e-11
    mac = o.get_macroscopic()
    assert mac["rhoA"].min() > 0 and np.isfinite(mac["ux"]).all()
    # something must actually have happened
    assert np.max(np.abs(mac["rhoA"] - c["rhoA"])) > 1e-3


def test_mass_conservation_with_walls_and_wetting():
    """Halfway bounce-back (R10) permutes populations: mass is exact with solids too."""
    rng = np.random.Generator(np.random.PCG64(11))
    shape = (7, 8, 9)
    mask = (rng.uniform(size=shape) < 0.3).astype(np.uint8)
    rA = rng.uniform(0.1, 1.0, shape)
    rB = rng.uniform(0.1, 1.0, shape)
    p = default_params(G=3.5, tau=(1.3, 0.62), xi=0.25, accel=(1e-5, -2e-5, 3e-5))
    o = LbmRef(mask, p)
    o.set_density(rA, rB)
    m0, _ = o.diagnostics()
    o.step(30)
    m1, _ = o.diagnostics()
    assert np.max(np.abs(m1 - m0) / m0) < 1e-13


# ------------------------------------------------------------------ lattice symmetries

def _random_case(seed, shape=(6, 7, 8)):
    rng = np.random.Generator(np.random.PCG64(seed))
    mask = (rng.uniform(size=shape) < 0.25).astype(np.uint8)
    rA = rng.uniform(0.05, 1.0, shape)
    rB = rng.uniform(0.05, 1.0, shape)
    return mask, rA, rB


def _macro(mask, rA, rB, p, steps=6):
    o = _run(mask, rA, rB, p, steps)
    return o.get_macroscopic()


@pytest.mark.parametrize("perm,flip", [((1, 0, 2), (False, False, False)),   # swap y<->z
                                        ((0, 2, 1), (False, False, False)),   # swap x<->y
                                        ((2, 1, 0), (False, False, False)),   # swap x<->z
                                        ((0, 1, 2), (True, False, False)),    # mirror z
                                        ((0, 1, 2), (False, False, True)),    # mirror x
                                        ((1, 2, 0), (False, True, False))])   # rotation + mirror
def test_lattice_symmetry(perm, flip):
    """Transforming the input by a symmetry of the cubic lattice transforms the output the
    same way (catches a wrong direction table, weight or opposite index)."""
    mask, rA, rB = _random_case(5)
    g = np.array([1e-5, -2e-5, 3e-5])               # (gx, gy, gz)
    p = default_params(G=3.5, tau=(1.0, 0.7), xi=0.15, accel=tuple(g))
    base = _macro(mask, rA, rB, p)

    def T(a):                                         # arrays are [z, y, x]
        a = np.transpose(a, perm)
        for ax, fl in enumerate(flip):
            if fl:
                a = np.flip(a, ax)
        return np.ascontiguousarray(a)

    # vector components: array axes (z,y,x) carry components (uz,uy,ux)
    names = ["uz", "uy", "ux"]
    g_zyx = g[::-1]
    g_new_zyx = np.array([g_zyx[perm[a]] * (-1 if flip[a] else 1) for a in range(3)])
    p2 = default_params(G=3.5, tau=(1.0, 0.7), xi=0.15, accel=tuple(g_new_zyx[::-1]))
    out = _macro(T(mask), T(rA), T(rB), p2)
    for k in ("rhoA", "rhoB", "P"):
        assert np.max(np.abs(out[k] - T(base[k]))) < 1e-13
    for a in range(3):
        expect = T(base[names[perm[a]]]) * (-1 if flip[a] else 1)
        assert np.max(np.abs(out[names[a]] - expect)) < 1e-13


def test_translation_invariance():
    mask, rA, rB = _random_case(6)
    p = default_params(G=3.5, tau=(0.8, 1.4), xi=-0.2)
    base = _macro(mask, rA, rB, p)
    sh = (2, 3, 5)
    roll = lambda a: np.roll(a, sh, (0, 1, 2))
    out = _macro(roll(mask), roll(rA), roll(rB), p)
    for k in base:
        assert np.max(np.abs(out[k] - roll(base[k]))) < 1e-13


def test_component_swap_symmetry():
    """Swapping the components with xi -> -xi and tau1 <-> tau2 swaps the output; this is why
    xi = 0 is neutral wetting."""
    mask, rA, rB = _random_case(7)
    a = _macro(mask, rA, rB, default_params(G=3.5, tau=(1.0, 0.7), xi=0.2, accel=(0, 0, 1e-5)))
    b = _macro(mask, rB, rA, default_params(G=3.5, tau=(0.7, 1.0), xi=-0.2, accel=(0, 0, 1e-5)))
    assert np.max(np.abs(a["rhoA"] - b["rhoB"])) < 1e-13
    assert np.max(np.abs(a["rhoB"] - b["rhoA"])) < 1e-13
    for k in ("ux", "uy", "uz", "P"):
        assert np.max(np.abs(a[k] - b[k])) < 1e-13


# ------------------------------------------------------------------ independent worked example

def test_worked_example_golden():
    """values produced by the survey's independent numpy restatement of
    Eq. (1)-(15) (NOT by this oracle, NOT by the CUDA path). Every feature is switched on."""
    rows = {}
    with open(os.path.join(HERE, "golden", "worked_example_appC.txt")) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, a, b = line.split()
            rows[k] = (float(a), float(b))
    nx, ny, nz = 8, 6, 5
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    mask = ((x + 2 * y + 3 * z) % 7 == 0).astype(np.uint8)
    assert mask.sum() == 34
    rA = 0.5 + 0.4 * np.sin(2 * np.pi * x / 8) * np.cos(2 * np.pi * y / 6) + 0.05 * np.cos(2 * np.pi * z / 5)
    rB = 1.03 - rA
    p = default_params(G=3.5, tau=(1.0, 0.7), xi=0.2, accel=(0.0, 0.0, 1e-5))
    o = LbmRef(mask, p)
    o.set_density(rA, rB)
    for col, nstep in ((0, 1), (1, 4)):
        o.step(nstep)
        m, j = o.diagnostics()
        mac = o.get_macroscopic()
        fA, fB = o.get_populations(0), o.get_populations(1)
        got = {"massA": m[0], "massB": m[1], "momx": j[0], "momy": j[1], "momz": j[2],
               "rhoA_321": mac["rhoA"][1, 2, 3], "rhoB_321": mac["rhoB"][1, 2, 3],
               "rhoA_754": mac["rhoA"][4, 5, 7], "rhoB_754": mac["rhoB"][4, 5, 7]}
        for i in (0, 1, 7, 14, 18):
            got[f"fA{i}_321"] = fA[i, 1, 2, 3]
            got[f"fB{i}_321"] = fB[i, 1, 2, 3]
        for k, v in got.items():
            ref = rows[k][col]
            assert abs(v - ref) <= 2e-13 * max(1.0, abs(ref)), (k, col, v, ref)
