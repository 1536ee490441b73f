"""Physics checks run through the CUDA path at the sizes BASELINE.json names (too slow for the CPU
oracle): config 2's static contact angle against the paper's calibration curve, and the 3-D
Laplace law.  The oracle is pinned to the same numbers on 2-D slabs in the CPU suite."""
import numpy as np
import pytest

from paper_2207_01534_b200 import Lbm
from workloads import default_params, make_config, tanh_profile

pytestmark = pytest.mark.gpu


def _paper_fit(xi):
    return 47.4136 * xi ** 3 - 23.4513 * xi ** 2 + 89.7938 * xi + 91.2324


def _cap_angle_through_B(rhoA, rhoB, wall_z=0.5, zmin=5.5):
    """Sphere-cap fit of the rho_A = rho_B surface (linear interpolation along z) at least 5 l.u.
    above the halfway wall plane; theta through component 2 (R24)."""
    d = rhoA - rhoB
    nz, ny, nx = d.shape
    pts = []
    for z in range(1, nz - 2):
        a, b = d[z], d[z + 1]
        cross = a * b < 0
        if not cross.any():
            continue
        yy, xx = np.nonzero(cross)
        zz = z + a[cross] / (a[cross] - b[cross])
        keep = zz >= zmin
        pts.append(np.c_[xx[keep], yy[keep], zz[keep]])
    p = np.concatenate(pts)
    p = p[p[:, 2] < nz / 2]                      # lower wall's droplet only
    A = np.c_[2 * p, np.ones(len(p))]
    (xc, yc, zc, cc), *_ = np.linalg.lstsq(A, (p ** 2).sum(1), rcond=None)
    R = np.sqrt(cc + xc * xc + yc * yc + zc * zc)
    theta_A = np.degrees(np.arccos(-(zc - wall_z) / R))
    return 180.0 - theta_A


def test_cfg2_contact_angles_follow_the_papers_calibration():
    """BASELINE.json config 2: 64^3, walls at z=0 and z=63, hemispherical droplet of A (r=16),
    fp32, 5 000 steps; xi in {-0.3, 0, +0.3} -> about 61, 91, 117 degrees through B (
    the fit was made at M=25, here M=1: +-5 degrees), and theta(-xi) = 180 - theta(xi)."""
    th = {}
    for xi in (-0.3, 0.0, 0.3):
        c = make_config(2, xi=xi)
        g = Lbm(c["mask"], c["params"])
        g.set_density(c["rhoA"], c["rhoB"])
        m0, _ = g.diagnostics()
        g.step(c["steps"])
        m1, _ = g.diagnostics()
        assert np.max(np.abs(m1 - m0) / m0) < 1e-5          # fp32 rounding drift over 5 000 steps (6e-10 per step)
        m = g.get_macroscopic(fields=("rhoA", "rhoB", "ux", "uy", "uz"))
        assert np.isfinite(m["rhoA"]).all()
        assert max(np.abs(m[k]).max() for k in ("ux", "uy", "uz")) < 0.02
        th[xi] = _cap_angle_through_B(m["rhoA"], m["rhoB"])
        g.close()
    for xi, v in th.items():
        assert abs(v - _paper_fit(xi)) < 5.0, th
    assert abs(th[-0.3] + th[0.3] - 180.0) < 1.5, th
    assert th[-0.3] < th[0.0] < th[0.3]


def test_laplace_law_3d():
    """3-D droplet, G=3.5, M=1: dP * R / 2 from Eq. (12) approaches the paper's gamma = 0.071
     from above as R grows (under-resolved radii read high): 64^3, r0 = 20."""
    n, r0 = 64, 20
    shape = (n, n, n)
    c = (n - 1) / 2.0
    rA = tanh_profile(shape, (c, c, c), r0)
    g = Lbm(np.zeros(shape, np.uint8), default_params(G=3.5, tau=(1.0, 1.0), storage_bits=32))
    g.set_density(rA, 1.027 - rA)
    g.step(4000)
    m = g.get_macroscopic(fields=("rhoA", "rhoB", "P"))
    d = (m["rhoA"] - m["rhoB"])
    row = 0.25 * (d[n // 2 - 1, n // 2 - 1] + d[n // 2, n // 2] + d[n // 2 - 1, n // 2] + d[n // 2, n // 2 - 1])
    i = np.nonzero((row[:-1] > 0) & (row[1:] <= 0))[0][0]
    R = i + row[i] / (row[i] - row[i + 1]) - c
    P = m["P"]
    Pin = P[n // 2 - 1:n // 2 + 1, n // 2 - 1:n // 2 + 1, n // 2 - 1:n // 2 + 1].mean()
    gamma = (Pin - P[0, 0, 0]) * R / 2.0
    assert abs(R - r0) < 1.5
    assert 0.068 < gamma < 0.080, gamma


def _laplace_3d(n, r0, tau, steps):
    shape = (n, n, n)
    c = (n - 1) / 2.0
    rA = tanh_profile(shape, (c, c, c), r0)                     # Eq. (16)
    g = Lbm(np.zeros(shape, np.uint8), default_params(G=3.5, tau=tau, storage_bits=32))
    g.set_density(rA, 1.027 - rA)
    g.step(steps)
    m = g.get_macroscopic(fields=("rhoA", "rhoB", "P"))
    g.close()
    d = m["rhoA"] - m["rhoB"]
    h = n // 2
    row = 0.25 * (d[h - 1, h - 1] + d[h, h] + d[h - 1, h] + d[h, h - 1])
    i = np.nonzero((row[:-1] > 0) & (row[1:] <= 0))[0][0]
    R = i + row[i] / (row[i] - row[i + 1]) - c
    P = m["P"]
    dP = P[h - 1:h + 1, h - 1:h + 1, h - 1:h + 1].mean() - P[0, 0, 0]
    return R, dP


def test_laplace_paper_size_128_cubed():
    """PAPER.md Sec. 3.1 at the paper's own size: 128^3 periodic box, droplets up to r0 = 30,
    G = 3.5.  The regression of dP against 2/R gives the surface tension: the paper reports
    gamma = 0.071 for M = 1, 25 and 1/25 alike (L175-183)."""
    pts = [_laplace_3d(128, r0, (1.0, 1.0), 12000) for r0 in (18, 24, 30)]
    x = np.array([2.0 / R for R, _ in pts])
    y = np.array([dP for _, dP in pts])
    slope, icpt = np.polyfit(x, y, 1)
    assert abs(slope / 0.071 - 1.0) < 0.08, (slope, icpt, pts)
    assert abs(icpt) < 6e-4                                    # dP -> 0 as R -> infinity
    # independent of the viscosity ratio: same droplet at M = 25 and M = 1/25
    g1 = pts[2][1] * pts[2][0] / 2.0
    for tau in ((3.5, 0.62), (0.62, 3.5)):
        R, dP = _laplace_3d(128, 30, tau, 12000)
        assert abs(dP * R / 2.0 / g1 - 1.0) < 0.03, (tau, dP * R / 2.0, g1)


PAPER_FIT = (47.4136, -23.4513, 89.7938, 91.2324)           # cubic, linear ... constant


def test_contact_angle_calibration_paper_size():
    """PAPER.md Sec. 3.2 at the paper's own size and viscosity ratio: 200 x 100 x 200 (wall-normal
    extent 100), droplet r0 = 30 on the bottom wall, M = 25 (tau = 3.5 / 0.62), G = 3.5, over the
    paper's whole range xi in [-0.5, 0.5] (Fig. 2).  theta (through component 2) against the
    printed cubic (L199) point by point, and the cubic re-fitted from these runs against the
    printed coefficients ("regenerating ... cubic coefficients")."""
    nz, ny, nx = 100, 200, 200
    shape = (nz, ny, nx)
    mask = np.zeros(shape, np.uint8)
    mask[0] = mask[-1] = 1
    rA = tanh_profile(shape, ((nx - 1) / 2.0, (ny - 1) / 2.0, 0.5), 30.0)
    rA = np.where(mask == 0, rA, 0.0)
    rB = np.where(mask == 0, 1.027 - rA, 0.0)
    got = {}
    for xi in (-0.5, -0.4, -0.3, -0.2, -0.1, 0.0, 0.1, 0.2, 0.3, 0.4, 0.5):
        g = Lbm(mask, default_params(G=3.5, tau=(3.5, 0.62), xi=xi, storage_bits=32))
        g.set_density(rA, rB)
        g.step(15000 if abs(xi) < 0.45 else 30000)          # the far ends spread / retract furthest
        m = g.get_macroscopic(fields=("rhoA", "rhoB"))
        g.close()
        assert np.isfinite(m["rhoA"]).all()
        got[xi] = _cap_angle_through_B(m["rhoA"], m["rhoB"])
    print("contact angles (xi: theta, paper fit):",
          {xi: (round(th, 2), round(_paper_fit(xi), 2)) for xi, th in got.items()})
    for xi, th in got.items():
        assert abs(th - _paper_fit(xi)) < (3.0 if abs(xi) < 0.45 else 4.0), got
    xs = np.array(sorted(got))
    coef = np.polyfit(xs, np.array([got[x] for x in xs]), 3)
    print("re-fitted cubic:", coef, "paper:", PAPER_FIT)
    assert abs(coef[3] - PAPER_FIT[3]) < 1.5, coef           # theta(0): neutral wetting, ~91 degrees
    assert abs(coef[2] / PAPER_FIT[2] - 1.0) < 0.05, coef    # slope at xi = 0 within 5 %
    assert abs(coef[1] - PAPER_FIT[1]) < 12.0 and abs(coef[0] - PAPER_FIT[0]) < 25.0, coef
    grid = np.linspace(-0.5, 0.5, 41)                        # the two curves agree over the range
    # measured: 42.43 xi^3 - 13.70 xi^2 + 87.65 xi + 90.49; largest gap to the paper's curve 3.0
    # degrees, at xi = -0.5 (37.5 against 34.5: the most strongly wetted, flattest cap)
    assert np.max(np.abs(np.polyval(coef, grid) - np.polyval(PAPER_FIT, grid))) < 4.0, coef
