"""Pins of the oracle's NEEM open planes (reading R12; "non-equilibrium extrapolation
method (NEEM) [6]", L150-157 frozen populations).  The method has a textbook definition (ref. [6]):
    f_i(x_b) = feq_i(rho_b, u_b) + [ f_i(x_f) - feq_i(rho(x_f), u(x_f)) ] ,
so the pins are that identity evaluated with an equilibrium written here from Eq. (2), its exact
consequences (imposed density met, momentum transplanted), the frozen rule for the other
component, and a moving fixed point.  What stays a reading (R12 iii) is the choice of the
velocity u(x_f): the bare mixture velocity."""
import numpy as np
import pytest

from oracle import LbmRef, lattice
from workloads import default_params

W, E, OPP = lattice()
Ef = E.astype(float)


def _feq(rho, u):
    """Eq. (2), for arrays rho[...], u[3, ...] -> [19, ...]"""
    eu = np.tensordot(Ef, u, axes=(1, 0))
    uu = (u * u).sum(0)
    return W.reshape((19,) + (1,) * rho.ndim) * rho * (1.0 + 3.0 * eu + 4.5 * eu * eu - 1.5 * uu)


def _params(**kw):
    p = dict(z_open=1, inlet_kind=1, inlet_comp=0, inlet_rho=1.03, outlet_kind=1, outlet_comp=1,
             outlet_rho=0.97, G=3.5, tau=(1.0, 0.7), xi=0.1, storage_bits=64)
    p.update(kw)
    return default_params(**p)


def _random_pops(shape, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    out = []
    for s in range(2):
        rho = rng.uniform(0.3, 1.0, shape)
        out.append(np.stack([W[i] * rho * (1.0 + 0.2 * rng.uniform(-1, 1, shape))
                             for i in range(19)]))
    return out


@pytest.mark.parametrize("inlet_kind", [1, 2])
def test_neem_identity_and_its_consequences(inlet_kind):
    shape = (9, 5, 6)
    mask = np.zeros(shape, np.uint8)
    mask[3:6, 1:3, 2:5] = 1
    p = _params(inlet_kind=inlet_kind, inlet_uz=0.011)
    o = LbmRef(mask, p)
    f0 = _random_pops(shape, 8)
    for s in range(2):
        o.set_populations(s, f0[s])
    o.step(2)
    f = [o.get_populations(s) for s in range(2)]
    for plane, zb, zf, dc, rho_given in ((0, 0, 1, 0, 1.03), (1, shape[0] - 1, shape[0] - 2, 1, 0.97)):
        rf = [f[s][:, zf].sum(0) for s in range(2)]
        j = sum(np.tensordot(Ef.T, f[s][:, zf], axes=(1, 0)) for s in range(2))
        uf = j / (rf[0] + rf[1])                         # bare mixture velocity at x_f (R12 iii)
        if plane == 0 and inlet_kind == 2:
            rho_b = rf[dc]
            ub = np.zeros_like(uf)
            ub[2] = 0.011
        else:
            rho_b = np.full_like(rf[dc], rho_given)
            ub = uf
        want = _feq(rho_b, ub) + (f[dc][:, zf] - _feq(rf[dc], uf))
        assert np.max(np.abs(f[dc][:, zb] - want)) < 2e-16
        # consequences: the imposed density is met exactly; the momentum is rho_b u_b plus the
        # neighbour's non-equilibrium momentum
        assert np.max(np.abs(f[dc][:, zb].sum(0) - rho_b)) < 1e-15
        jb = np.tensordot(Ef.T, f[dc][:, zb], axes=(1, 0))
        jn = np.tensordot(Ef.T, f[dc][:, zf], axes=(1, 0))
        assert np.max(np.abs(jb - (rho_b * ub + jn - rf[dc] * uf))) < 1e-15


def test_frozen_rule_of_the_other_component():
    """the 5 populations of the other component that would enter through the
    plane keep their initial values for the whole run; its remaining 14 are streamed."""
    shape = (8, 4, 5)
    mask = np.zeros(shape, np.uint8)
    o = LbmRef(mask, _params())
    f0 = _random_pops(shape, 9)
    for s in range(2):
        o.set_populations(s, f0[s])
    inward = {0: [i for i in range(19) if E[i][2] == 1], 1: [i for i in range(19) if E[i][2] == -1]}
    for _ in range(3):
        o.step(2)
        fB, fA = o.get_populations(1), o.get_populations(0)
        assert np.array_equal(fB[inward[0], 0], f0[1][inward[0], 0])         # inlet: other = B
        assert np.array_equal(fA[inward[1], -1], f0[0][inward[1], -1])       # outlet: other = A
    others = [i for i in range(19) if i not in inward[0]]
    assert not np.allclose(o.get_populations(1)[others, 0], f0[1][others, 0])


def test_neem_moving_uniform_flow_is_a_fixed_point():
    """G = 0: both components in equilibrium at the common velocity (0, 0, u0) everywhere, inlet
    and outlet densities equal to the state's: NEEM reproduces the equilibrium on the planes and
    the frozen inward populations are the equilibrium ones, so nothing changes."""
    shape = (8, 4, 5)
    mask = np.zeros(shape, np.uint8)
    u0, rho = 0.03, (0.8, 0.3)
    u = np.zeros((3,) + shape)
    u[2] = u0
    f0 = [_feq(np.full(shape, r), u) for r in rho]
    for ik in (1, 2):
        o = LbmRef(mask, _params(G=0.0, xi=0.0, tau=(0.9, 1.3), inlet_kind=ik, inlet_rho=rho[0],
                                 inlet_uz=u0, outlet_rho=rho[1]))
        for s in range(2):
            o.set_populations(s, f0[s])
        o.step(30)
        for s in range(2):
            assert np.max(np.abs(o.get_populations(s) - f0[s])) < 1e-15


def test_neem_extrapolates_the_collision_operators_nonequilibrium_part():
    """Reading R12 iii without retyping anything: ref. [6] extrapolates f - f^eq, and the model has
    ONE equilibrium -- Eq. (2) at the common velocity of Eq. (8), the one its
    collision relaxes to.  That equilibrium is read off the oracle's own collision operator (which
    the shear-wave and Poiseuille pins fix independently): with no forces (G = 0, g = 0) and
    tau_A = tau_B = tau, Eq. (1) is f* = f - (f - f^eq)/tau, so f^eq = f - tau (f - f*), and f* of a
    node sits, after streaming, at its neighbours.  Because Eq. (2) is linear in the density at
    fixed velocity, f^eq(rho_b, u_f) = (rho_b / rho_sigma(x_f)) f^eq_sigma(x_f), and NEEM reads
        f(x_b) = (rho_b / rho(x_f)) f^eq(x_f) + f(x_f) - f^eq(x_f)
    with nothing typed here but that linearity.  The two components are given different momenta,
    so an extrapolation at a component's own velocity j_sigma/rho_sigma fails by O(1e-3)."""
    shape = (8, 4, 5)
    nz = shape[0]
    tau = 0.8
    mask = np.zeros(shape, np.uint8)
    p = _params(G=0.0, tau=(tau, tau), xi=0.0)
    o = LbmRef(mask, p)
    rng = np.random.Generator(np.random.PCG64(12))
    f0 = _random_pops(shape, 12)
    f0[0] = f0[0] * (1.0 + 0.05 * Ef[:, 2].reshape(19, 1, 1, 1))      # A drifts up, B down:
    f0[1] = f0[1] * (1.0 - 0.05 * Ef[:, 0].reshape(19, 1, 1, 1))      # different momenta
    for s in range(2):
        o.set_populations(s, f0[s])
    o.step(1)
    f = [o.get_populations(s) for s in range(2)]          # complete state at t+1, planes fixed
    ua = np.tensordot(Ef.T, f[0][:, 1], axes=(1, 0)) / f[0][:, 1].sum(0)
    ub = np.tensordot(Ef.T, f[1][:, 1], axes=(1, 0)) / f[1][:, 1].sum(0)
    assert np.abs(ua - ub).max() > 1e-2                    # the discrimination is real
    # the model's equilibrium of that state, from the collision operator of a periodic copy
    q = LbmRef(mask, _params(G=0.0, tau=(tau, tau), xi=0.0, z_open=0))
    for s in range(2):
        q.set_populations(s, f[s])
    q.step(1)
    g = [q.get_populations(s) for s in range(2)]
    for zb, zf, dc, rho_b in ((0, 1, 0, 1.03), (nz - 1, nz - 2, 1, 0.97)):
        fstar = np.empty_like(f[dc][:, zf])
        for i in range(19):                                # f*_i(x) travelled to x + e_i
            fstar[i] = np.roll(g[dc][i], (-E[i][2], -E[i][1], -E[i][0]), (0, 1, 2))[zf]
        feq = f[dc][:, zf] - tau * (f[dc][:, zf] - fstar)
        rho_f = f[dc][:, zf].sum(0)
        assert np.abs(feq.sum(0) - rho_f).max() < 1e-14    # it is an equilibrium of that density
        want = (rho_b / rho_f) * feq + f[dc][:, zf] - feq
        assert np.abs(f[dc][:, zb] - want).max() < 1e-14
