"""Pins of the CPU oracle, part 2: closed forms, textbook reductions and the numbers the paper
prints (SURVEY.md §8c "pins").

Sizes are reduced from the paper's (128^3 Laplace, 200x100x200 contact angle) to quasi-2-D
slabs so the whole CPU suite stays within minutes; the tolerances state what that costs.
"""
import numpy as np
import pytest

import os

from oracle import LbmRef, lattice
from workloads import default_params, tanh_profile


def _paper_values():
    """tests/golden/paper_values.txt: numbers printed in the paper, each with its citation."""
    out = {}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_values.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if line:
                out[line[0]] = [float(v) for v in line[1:]]
    return out


PAPER = _paper_values()


# ------------------------------------------------------------------ G = 0: textbook SRT-LBM

def test_g0_shear_wave_decays_with_nu():
    """With G=0 and tau1=tau2 the sum of the components is single-component SRT-LBM: a shear
    wave decays as exp(-nu k^2 t) with nu=(tau-1/2)/3 (reading R2 of Eq. 7)."""
    w, e, _ = lattice()
    ny, tau, u0 = 48, 0.8, 1e-4
    k = 2 * np.pi / ny
    shape = (1, ny, 1)
    y = np.arange(ny)[None, :, None] * np.ones(shape)
    ux = u0 * np.sin(k * y)
    f = []
    for rho in (0.7, 0.3):
        eu = e[:, 0][:, None, None, None] * ux[None]
        f.append(w[:, None, None, None] * rho * (1 + 3 * eu + 4.5 * eu * eu - 1.5 * ux[None] ** 2))
    o = LbmRef(np.zeros(shape, np.uint8), default_params(G=0.0, tau=(tau, tau)))
    o.set_populations(0, f[0])
    o.set_populations(1, f[1])
    T = 400
    a0 = np.abs(np.fft.fft(o.get_macroscopic()["ux"][0, :, 0])[1])
    o.step(T)
    m = o.get_macroscopic()
    a1 = np.abs(np.fft.fft(m["ux"][0, :, 0])[1])
    nu = (tau - 0.5) / 3.0
    rate = -np.log(a1 / a0) / T
    assert abs(rate / (nu * k * k) - 1.0) < 5e-3
    # the mixture fractions are advected passively and stay uniform
    assert np.allclose(m["rhoA"], 0.7, atol=1e-9) and np.allclose(m["rhoB"], 0.3, atol=1e-9)


# ------------------------------------------------------------------ Poiseuille closed form

@pytest.mark.parametrize("tau", [1.0, 0.62, 0.5 + np.sqrt(3.0) / 4.0])
def test_poiseuille_discrete_closed_form(tau):
    """Single component (rho_B = 0, legal by R4), body force rho*g through Eq. (9) (R8), halfway
    bounce-back (R10). Discrete steady solution of SRT + this forcing: an exact parabola with
    curvature -g/nu whose wall lies half a link outside the last fluid node, plus the textbook
    slip g(16 tau^2 - 16 tau + 1)/(24 nu) = g(48 nu^2 - 1)/(8 nu); zero at tau = 1/2 + sqrt(3)/4."""
    H, g = 12, 1e-6
    nu = (tau - 0.5) / 3.0
    shape = (1, H + 2, 1)
    mask = np.zeros(shape, np.uint8)
    mask[0, 0, 0] = mask[0, H + 1, 0] = 1
    o = LbmRef(mask, default_params(G=3.5, tau=(tau, tau), accel=(g, 0.0, 0.0)))
    o.set_density(np.ones(shape), np.zeros(shape))
    o.step(int(12 * H * H / nu / 9.87) + 2000)          # ~12 viscous decay times
    u = o.get_macroscopic()["ux"][0, 1:H + 1, 0]
    yj = np.arange(1, H + 1) - 0.5
    exact = g / (2 * nu) * yj * (H - yj) + g * (16 * tau * tau - 16 * tau + 1) / (24 * nu)
    assert np.max(np.abs(u - exact)) < 1e-6 * exact.max()
    d2 = u[:-2] - 2 * u[1:-1] + u[2:]
    assert np.max(np.abs(d2 + g / nu)) < 1e-6 * g / nu


# ------------------------------------------------------------------ coexistence

def test_flat_interface_coexistence():
    """G=3.5: the paper initialises with rho_in=1, rho_out=0.027 (L173). A flat
    interface must stay demixed with the minority density near 0.027 (the exact value depends
    weakly on the enclosed mass: 0.0246-0.0275 over the set-ups used here, hence +-0.003) and
    with equal bulk pressures (Eq. 12, R13) on both sides -- a slab of A filling 1/4 of the box,
    so that neither check is trivial by component-swap symmetry."""
    nz = 96
    shape = (nz, 1, 1)
    zc = np.arange(nz)[:, None, None]
    rA = np.where((zc >= nz // 8) & (zc < 3 * nz // 8), 1.0, 0.027) * np.ones(shape)
    rB = 1.027 - rA
    o = LbmRef(np.zeros(shape, np.uint8), default_params(G=3.5, tau=(1.0, 1.0)))
    o.set_density(rA, rB)
    o.step(8000)
    m = o.get_macroscopic()
    a, b = m["rhoA"][:, 0, 0], m["rhoB"][:, 0, 0]
    zin, zout = nz // 4, 3 * nz // 4
    assert abs(a[zout] - 0.027) < 0.003 and abs(b[zin] - 0.027) < 0.003
    assert abs(a[zin] - 1.0) < 0.03 and abs(b[zout] - 1.0) < 0.03
    assert np.max(np.abs(m["uz"])) < 1e-5
    assert abs(m["P"][zin, 0, 0] - m["P"][zout, 0, 0]) < 2e-6


# ------------------------------------------------------------------ Laplace law

def _laplace_2d(n, r0, tau, steps, half_force=1):
    shape = (1, n, n)
    c = (n - 1) / 2.0
    rA = tanh_profile(shape, (c, c, None), r0)                      # Eq. (16)
    o = LbmRef(np.zeros(shape, np.uint8), default_params(G=3.5, tau=tau, half_force=half_force))
    o.set_density(rA, 1.027 - rA)
    o.step(steps)
    m = o.get_macroscopic()
    if not np.isfinite(m["P"]).all():
        return np.nan, np.nan
    d = (m["rhoA"] - m["rhoB"])[0]
    row = 0.5 * (d[n // 2 - 1] + d[n // 2])
    i = np.nonzero((row[:-1] > 0) & (row[1:] <= 0))[0][0]
    R = i + row[i] / (row[i] - row[i + 1]) - c                      # rho_A = rho_B crossing (R25)
    P = m["P"][0]
    Pin = 0.25 * (P[n // 2 - 1, n // 2 - 1] + P[n // 2, n // 2] + P[n // 2 - 1, n // 2] + P[n // 2, n // 2 - 1])
    return R, Pin - P[0, 0]


def test_laplace_surface_tension_matches_paper():
    """2-D slab (cylinder) Laplace law dP = gamma/R with P from Eq. (12): the paper's regression
    gives gamma = 0.071 at G=3.5 for every viscosity ratio.  SURVEY.md 8(c):
    three radii within 5 % of 0.071 each, the regression slope of dP against 1/R within 5 %, and
    equality across M = 1 and M = 25 within 2 % at every radius (measured: +2.7..+3.1 % at M = 1,
    +1.6..+2.5 % at M = 25; reduced size 96^2, R = 12..24, against the paper's 128^3, R = 30)."""
    cases = ((12, 4000), (16, 4500), (24, 6000))
    g1, invR, dPs = [], [], []
    for r0, steps in cases:
        R, dP = _laplace_2d(96, r0, (1.0, 1.0), steps)
        assert abs(R - r0) < 1.0 and dP > 0
        g1.append(dP * R)
        invR.append(1.0 / R)
        dPs.append(dP)
    assert all(abs(v / PAPER["gamma"][0] - 1.0) < 0.05 for v in g1), g1
    slope, icpt = np.polyfit(invR, dPs, 1)                           # Laplace law is linear (L165, L183)
    assert abs(slope / PAPER["gamma"][0] - 1.0) < 0.05, slope
    assert abs(icpt) < 0.02 * dPs[-1], icpt
    # independent of the viscosity ratio: M = 25 <=> tau = (3.5, 0.62)
    for (r0, steps), ref in zip(cases, g1):
        R, dP = _laplace_2d(96, r0, tuple(PAPER["tau_M25"]), steps)
        assert abs(dP * R / PAPER["gamma"][0] - 1.0) < 0.05
        assert abs(dP * R / ref - 1.0) < 0.02, (r0, dP * R, ref)
    # M = 1/25 is M = 25 with the components' relaxation times exchanged
    R, dP = _laplace_2d(96, 16, tuple(PAPER["tau_M25"])[::-1], 4500)
    assert abs(dP * R / g1[1] - 1.0) < 0.02


@pytest.mark.skipif(not os.environ.get("LBM_ORACLE_SLOW"),
                    reason="6 minutes of oracle time: set LBM_ORACLE_SLOW=1 (result recorded in DESIGN.md section 3)")
def test_laplace_3d_point():
    """one 3-D point at R >= 15 within 10 % of gamma = 0.071 (dP = 2 gamma / R,
    PAPER.md L165, L181).  64^3, r0 = 20, 4000 steps."""
    n, r0 = 64, 20
    shape = (n, n, n)
    c = (n - 1) / 2.0
    rA = tanh_profile(shape, (c, c, c), r0)
    o = LbmRef(np.zeros(shape, np.uint8), default_params(G=3.5, tau=(1.0, 1.0)))
    o.set_density(rA, 1.027 - rA)
    o.step(4000)
    m = o.get_macroscopic()
    d = (m["rhoA"] - m["rhoB"])
    row = 0.25 * (d[n // 2 - 1, n // 2 - 1] + d[n // 2, n // 2] + d[n // 2 - 1, n // 2] + d[n // 2, n // 2 - 1])
    i = np.nonzero((row[:-1] > 0) & (row[1:] <= 0))[0][0]
    R = i + row[i] / (row[i] - row[i + 1]) - c
    P = m["P"]
    Pin = P[n // 2 - 1:n // 2 + 1, n // 2 - 1:n // 2 + 1, n // 2 - 1:n // 2 + 1].mean()
    gamma = (Pin - P[0, 0, 0]) * R / 2.0
    print("3-D Laplace point: R = %.3f, gamma = %.5f" % (R, gamma))
    assert R >= 15 and abs(gamma / PAPER["gamma"][0] - 1.0) < 0.10, (R, gamma)


def test_laplace_negative_control_literal_eq4():
    """Reading R3: without the F/2 shift of the equilibrium velocity (literal Eq. 4) the pressure
    jump of Eq. (12) has the wrong sign -- contradicting PAPER.md L183 -- so the shift is needed."""
    R, dP = _laplace_2d(64, 16, (1.0, 1.0), 3000, half_force=0)
    assert not (dP > 1e-3)
    R, dP = _laplace_2d(64, 16, (1.0, 1.0), 3000, half_force=1)
    assert dP * R > 0.06


# ------------------------------------------------------------------ contact angle

def _contact_angle_through_B(nx, nz, r0, xi, tau, steps):
    """Sessile 2-D droplet of A on the bottom wall; circle fit of the rho_A = rho_B contour
    (linear interpolation) at least 5 l.u. above the halfway wall plane (R24)."""
    shape = (nz, 1, nx)
    mask = np.zeros(shape, np.uint8)
    mask[0] = mask[-1] = 1
    rA = tanh_profile(shape, ((nx - 1) / 2.0, None, 0.5), r0)
    o = LbmRef(mask, default_params(G=3.5, tau=tau, xi=xi))
    o.set_density(rA, np.where(mask == 0, 1.027 - rA, 0.0))
    o.step(steps)
    m = o.get_macroscopic()
    d = (m["rhoA"] - m["rhoB"])[:, 0, :]
    pts = []
    zmin = 0.5 + 5.0
    for z in range(1, nz - 1):
        r = d[z]
        if z >= zmin:
            for i in np.nonzero(r[:-1] * r[1:] < 0)[0]:
                pts.append((i + r[i] / (r[i] - r[i + 1]), float(z)))
    for x in range(nx):
        c = d[1:nz - 1, x]
        for k in np.nonzero(c[:-1] * c[1:] < 0)[0]:
            zz = 1 + k + c[k] / (c[k] - c[k + 1])
            if zz >= zmin:
                pts.append((float(x), zz))
    p = np.array(pts)
    A = np.c_[2 * p[:, 0], 2 * p[:, 1], np.ones(len(p))]
    (xc, zc, cc), *_ = np.linalg.lstsq(A, (p ** 2).sum(1), rcond=None)
    R = np.sqrt(cc + xc * xc + zc * zc)
    theta_A = np.degrees(np.arccos(-(zc - 0.5) / R))
    return 180.0 - theta_A


def _paper_fit(xi):
    a, b, c, d = PAPER["theta_fit"]
    return a * xi ** 3 + b * xi ** 2 + c * xi + d


@pytest.mark.parametrize("xi", [-0.2, 0.0, 0.2])
def test_contact_angle_follows_paper_fit(xi):
    """IVSD wetting (Eq. 13-15) with chi = 1 +- xi: theta through component 2
    follows the paper's cubic (L199; ~70 deg at xi=-0.2, L221; ~108 deg at +0.2, L249).
    Reduced 2-D slab at M=1 instead of 200x100x200 at M=25: tolerance 3 degrees."""
    th = _contact_angle_through_B(80, 40, 16, xi, (1.0, 1.0), 5000)
    assert abs(th - _paper_fit(xi)) < 3.0, th
