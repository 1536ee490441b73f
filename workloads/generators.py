"""Seeded generators for the five BASELINE.json configs.

All arrays are indexed [z, y, x] (x fastest in memory, i.e. idx = x + nx*(y + ny*z)),
masks are uint8 with 1 = solid, densities are float64.  Randomness comes from
numpy.random.Generator(PCG64(seed)) only.

The paper's workloads (Finney sphere pack; Bentheimer sandstone,
PAPER.md L241) are Digital Rocks Portal data sets that are not available here;
the sphere pack and the thresholded Gaussian random field below stand in for them.
"""
from __future__ import annotations

import numpy as np

CONFIG_NAMES = {
    1: "cfg1_droplet_32",
    2: "cfg2_contact_64",
    3: "cfg3_spherepack_128_drainage",
    4: "cfg4_grf_256_imbibition",
    5: "cfg5_spherepack_512_throughput",
}

# Coexistence (minority) densities of a flat interface, as computed by the oracle
# (tests/test_oracle_physics.py::test_flat_interface_coexistence re-derives them).
MINORITY_DENSITY = {3.5: 0.0264, 3.0: 0.0486}


def default_params(**kw):
    p = dict(
        G=3.5, tau=(1.0, 1.0), xi=0.0, accel=(0.0, 0.0, 0.0),
        z_open=0,
        inlet_kind=1, inlet_comp=0, inlet_rho=1.0, inlet_uz=0.0,
        outlet_kind=1, outlet_comp=1, outlet_rho=1.0,
        storage_bits=32, half_force=1,
    )
    p.update(kw)
    return p


# ----------------------------------------------------------------------------- geometry

def _paint_sphere(solid, c, r, periodic):
    """Mark voxels whose centre lies within r of c (with periodic images). Returns #new solids."""
    nz, ny, nx = solid.shape
    n = (nx, ny, nz)
    lo = [int(np.floor(c[a] - r)) for a in range(3)]
    hi = [int(np.ceil(c[a] + r)) for a in range(3)]
    axes = []
    for a in range(3):
        idx = np.arange(lo[a], hi[a] + 1)
        d = idx - c[a]
        if periodic[a]:
            idx = np.mod(idx, n[a])
            keep = np.ones(idx.shape, bool)
        else:
            keep = (idx >= 0) & (idx < n[a])
        axes.append((idx[keep], d[keep]))
    (ix, dx), (iy, dy), (iz, dz) = axes
    d2 = dz[:, None, None] ** 2 + dy[None, :, None] ** 2 + dx[None, None, :] ** 2
    inside = d2 <= r * r
    sub = solid[np.ix_(iz, iy, ix)]
    new = int(np.count_nonzero(inside & (sub == 0)))
    sub[inside] = 1
    solid[np.ix_(iz, iy, ix)] = sub
    return new


def sphere_pack_mask(n, seed, rmin, rmax, porosity=0.38, overlap=0.75,
                     max_reject=2000, periodic=(True, True, True)):
    """Sphere pack: random sequential addition until `max_reject` consecutive rejections,
    then spheres allowed to overlap down to `overlap`*(r_i+r_j) centre distance, until the
    voxelised porosity is <= `porosity` (SURVEY.md R-gen; plain RSA jams near 0.63).
    Returns (mask[z,y,x] uint8, achieved porosity, number of spheres)."""
    nx = ny = nz = int(n)
    rng = np.random.Generator(np.random.PCG64(seed))
    solid = np.zeros((nz, ny, nx), np.uint8)
    box = np.array([nx, ny, nz], float)
    per = np.array(periodic, bool)
    cs = np.zeros((0, 3))
    rs = np.zeros((0,))
    nsolid = 0
    total = nx * ny * nz
    factor = 1.0
    rejects = 0
    guard = 0
    while nsolid < (1.0 - porosity) * total:
        guard += 1
        if guard > 2_000_000:
            break
        c = rng.uniform(0.0, 1.0, 3) * box
        r = rng.uniform(rmin, rmax)
        if len(rs):
            d = np.abs(cs - c)
            d = np.where(per, np.minimum(d, box - d), d)
            dist = np.sqrt((d * d).sum(1))
            ok = bool(np.all(dist >= factor * (rs + r)))
        else:
            ok = True
        if not ok:
            rejects += 1
            if factor == 1.0 and rejects >= max_reject:
                factor = overlap
                rejects = 0
            continue
        rejects = 0
        cs = np.vstack([cs, c])
        rs = np.append(rs, r)
        nsolid += _paint_sphere(solid, c - 0.5, r, periodic)
    return solid, 1.0 - nsolid / total, len(rs)


def grf_mask(n, seed, sigma=5.0, porosity=0.21):
    """Sandstone-like mask: white noise -> periodic Gaussian filter (std `sigma` voxels)
    -> fluid where the field is below its `porosity` quantile. Isolated pores are kept."""
    from scipy.ndimage import gaussian_filter
    rng = np.random.Generator(np.random.PCG64(seed))
    if np.isscalar(n):
        shape = (int(n),) * 3
    else:
        shape = tuple(int(v) for v in n)
    field = rng.standard_normal(shape).astype(np.float32)
    field = gaussian_filter(field, sigma=sigma, mode="wrap")
    thr = np.quantile(field, porosity)
    return (field >= thr).astype(np.uint8)


def clear_end_layers(mask, layers=8):
    """Reservoir layers of pure fluid at both z ends."""
    m = mask.copy()
    m[:layers] = 0
    m[m.shape[0] - layers:] = 0
    return m


# ----------------------------------------------------------------------------- initial states

def tanh_profile(shape, centre, r0, rho_in=1.0, rho_out=0.027, W=5.0):
    """Eq. (16): diffuse droplet of radius r0 about `centre`=(xc,yc,zc).
    A centre coordinate of None drops that axis (cylinder / slab droplets)."""
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.arange(nz, dtype=float), np.arange(ny, dtype=float),
                          np.arange(nx, dtype=float), indexing="ij")
    r2 = np.zeros(shape)
    for coord, c in zip((x, y, z), centre):
        if c is not None:
            r2 += (coord - c) ** 2
    r = np.sqrt(r2)
    return 0.5 * (rho_in + rho_out) - 0.5 * (rho_in - rho_out) * np.tanh(2.0 * (r - r0) / W)


def _slab_state(shape, z_split, major=1.0, minor=0.027):
    """Component A for z < z_split, B elsewhere."""
    nz = shape[0]
    a = np.where(np.arange(nz)[:, None, None] < z_split, major, minor) * np.ones(shape)
    b = (major + minor) - a
    return a, b


def make_config(k, size=None, seed=None, **overrides):
    """Inputs of BASELINE.json config k (1..5). `size` overrides the box edge (crops /
    reduced test sizes keep the recipe); returns a dict with
    mask[z,y,x] uint8, rhoA, rhoB [z,y,x] float64, params (dict), steps, name, porosity."""
    if k == 1:
        n = size or 32
        seed = 1 if seed is None else seed
        rng = np.random.Generator(np.random.PCG64(seed))
        shape = (n, n, n)
        c = (n - 1) / 2.0
        z, y, x = np.meshgrid(*(np.arange(n, dtype=float),) * 3, indexing="ij")
        inside = (x - c) ** 2 + (y - c) ** 2 + (z - c) ** 2 < (n / 4.0) ** 2
        rhoA = np.where(inside, 1.0, 0.02) + rng.uniform(-1e-3, 1e-3, shape)
        rhoB = np.where(inside, 0.02, 1.0) + rng.uniform(-1e-3, 1e-3, shape)
        mask = np.zeros(shape, np.uint8)
        params = default_params(G=0.9, tau=(1.0, 1.0), storage_bits=64)
        steps = 200
    elif k == 2:
        n = size or 64
        shape = (n, n, n)
        mask = np.zeros(shape, np.uint8)
        mask[0] = 1
        mask[n - 1] = 1
        c = (n - 1) / 2.0
        rhoA = tanh_profile(shape, (c, c, 0.5), n / 4.0)
        rhoB = 1.027 - rhoA
        params = default_params(G=3.5, tau=(1.0, 1.0), xi=-0.3)
        steps = 5000
    elif k == 3:
        n = size or 128
        seed = 3 if seed is None else seed
        scale = n / 128.0
        mask, _, _ = sphere_pack_mask(n, seed, 6.0 * max(scale, 0.5), 10.0 * max(scale, 0.5))
        layers = 8
        mask = clear_end_layers(mask, layers)
        rhoA, rhoB = _slab_state(mask.shape, layers)
        params = default_params(G=3.5, tau=(1.0, 1.0), xi=-0.2, z_open=1,
                                inlet_kind=2, inlet_comp=0, inlet_uz=1e-4, inlet_rho=1.0,
                                outlet_kind=1, outlet_comp=1, outlet_rho=1.0)
        steps = 20000
    elif k == 4:
        n = size or 256
        seed = 4 if seed is None else seed
        G = overrides.pop("G", 3.5)
        mask = grf_mask(n, seed, sigma=5.0, porosity=0.21)
        layers = 8
        mask = clear_end_layers(mask, layers)
        minor = MINORITY_DENSITY.get(G, 0.027)
        major = 1.0
        # wetting B fills the inlet reservoir, A everywhere else
        rhoB, rhoA = _slab_state(mask.shape, layers, major, minor)
        params = default_params(G=G, tau=(1.5, 0.6), xi=-0.2, z_open=1,
                                inlet_kind=1, inlet_comp=1, inlet_rho=1.02,
                                outlet_kind=1, outlet_comp=0, outlet_rho=1.0)
        steps = 10000
    elif k == 5:
        n = size or 512
        seed = 5 if seed is None else seed
        scale = n / 512.0
        mask, _, _ = sphere_pack_mask(n, seed, 24.0 * scale, 40.0 * scale)
        rhoA, rhoB = _slab_state(mask.shape, n // 2)
        params = default_params(G=3.5, tau=(1.0, 1.0), xi=0.0, accel=(0.0, 0.0, 1e-6))
        steps = 1000
    else:
        raise ValueError("config must be 1..5")
    params.update(overrides)
    fluid = mask == 0
    rhoA = np.where(fluid, rhoA, 0.0)
    rhoB = np.where(fluid, rhoB, 0.0)
    return dict(name=CONFIG_NAMES[k], mask=np.ascontiguousarray(mask),
                rhoA=np.ascontiguousarray(rhoA), rhoB=np.ascontiguousarray(rhoB),
                params=params, steps=steps, porosity=float(fluid.mean()))
