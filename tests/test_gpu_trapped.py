"""GPU parity of the trapped-volume query (reading R15): connected-component labelling on the GPU
(union-find over the compact ids, k_ccl_* in kernels.cuh) against the oracle's definition, and
against constructions whose answer is known without either."""
import numpy as np
import pytest

from oracle import LbmRef
from paper_2207_01534_b200 import Lbm
from workloads import default_params, make_config

pytestmark = pytest.mark.gpu


def _both(mask, rA, rB, p):
    o, g = LbmRef(mask, p), Lbm(mask, p)
    o.set_density(rA, rB)
    g.set_density(rA, rB)
    return o, g


def _blobs(shape, seed, sigma):
    """Smooth random two-phase field: many clusters of both phases, some touching the ends."""
    rng = np.random.Generator(np.random.PCG64(seed))
    f = rng.standard_normal(shape)
    k = [np.fft.fftfreq(n) for n in shape]
    kk = k[0][:, None, None] ** 2 + k[1][None, :, None] ** 2 + k[2][None, None, :] ** 2
    f = np.real(np.fft.ifftn(np.fft.fftn(f) * np.exp(-2 * (np.pi * sigma) ** 2 * kk)))
    return f / f.std()


@pytest.mark.parametrize("shape,solid,bits,z_open", [((40, 36, 44), 0.0, 64, 0),
                                                     ((40, 36, 44), 0.25, 64, 0),
                                                     ((33, 47, 29), 0.35, 32, 0),
                                                     ((48, 32, 32), 0.2, 32, 1),
                                                     ((130, 20, 150), 0.3, 32, 0)])
def test_trapped_volume_matches_oracle(shape, solid, bits, z_open):
    rng = np.random.Generator(np.random.PCG64(31))
    mask = (rng.uniform(size=shape) < solid).astype(np.uint8)
    if z_open:
        mask[:2] = 0                    # reading R12: the two layers at either end are fluid
        mask[-2:] = 0
    f = _blobs(shape, 32, 2.5)
    rA = np.where(f > 0.3, 0.9, 0.1) + 0.01 * rng.uniform(size=shape)
    rB = 1.0 - rA
    if bits == 32:                      # exactly representable: the phase decision cannot differ
        rA, rB = rA.astype(np.float32).astype(np.float64), rB.astype(np.float32).astype(np.float64)
    kw = dict(storage_bits=bits)
    if z_open:
        kw.update(z_open=1, inlet_kind=1, inlet_comp=1, inlet_rho=1.0, outlet_kind=1, outlet_comp=0,
                  outlet_rho=1.0)
    p = default_params(**kw)
    o, g = _both(mask, rA, rB, p)
    nz = shape[0]
    seen = 0
    for comp in (0, 1):
        for z0, z1 in ((0, nz), (nz // 4, 3 * nz // 4), (nz - 1, nz), (0, 1)):
            no, mo = o.trapped_volume(comp, z0, z1)
            ng, mg = g.trapped_volume(comp, z0, z1)
            assert no == ng, (comp, z0, z1, no, ng)
            # fp32 storage: rho = sum_i f_i carries fp32 rounding; the node set is still exact
            assert abs(mo - mg) <= (1e-12 if bits == 64 else 1e-6) * max(1.0, mo)
            seen += no
    assert seen > 0                     # the case does contain trapped clusters
    # same answer after a few steps too (state no longer the initial one)
    o.step(3)
    g.step(3)
    if bits == 64:
        assert o.trapped_volume(0, 0, nz)[0] == g.trapped_volume(0, 0, nz)[0]


def test_trapped_volume_known_constructions():
    """Answers fixed by construction: an isolated droplet is trapped, one that reaches an end
    plane is not, one that reaches the other side only through the periodic wrap in z is trapped,
    one that is joined through the periodic wrap in x is one cluster."""
    nz, ny, nx = 24, 20, 28
    mask = np.zeros((nz, ny, nx), np.uint8)
    A = np.zeros((nz, ny, nx), bool)
    A[8:12, 5:9, 10:15] = True                    # isolated: 4*4*5 = 80 nodes, trapped
    A[0:5, 14:16, 2:4] = True                     # touches z=0: 20 nodes, not trapped
    A[20:24, 2:4, 20:22] = True                   # touches z=nz-1: not trapped
    A[15:17, 10:12, 0:3] = True                   # wraps in x: 2*2*3 + 2*2*2 = one cluster of 20
    A[15:17, 10:12, 26:28] = True
    rA = np.where(A, 0.9, 0.1)
    rB = 1.0 - rA
    g = Lbm(mask, default_params(storage_bits=64))
    g.set_density(rA, rB)
    n, m = g.trapped_volume(0, 0, nz)
    assert n == 80 + 20 and abs(m - 100 * 0.9) < 1e-12
    assert g.trapped_volume(0, 8, 12)[0] == 80
    assert g.trapped_volume(0, 15, 16)[0] == 10
    assert g.trapped_volume(1, 0, nz)[0] == 0     # the B phase is one cluster touching both ends
    # a thin wall of solid splits the B phase: the enclosed B pocket becomes trapped
    mask2 = mask.copy()
    mask2[6, 3:11, 8:17] = mask2[13, 3:11, 8:17] = 1
    mask2[6:14, 3, 8:17] = mask2[6:14, 10, 8:17] = 1
    mask2[6:14, 3:11, 8] = mask2[6:14, 3:11, 16] = 1
    g2 = Lbm(mask2, default_params(storage_bits=64))
    g2.set_density(rA, rB)
    inside = np.zeros_like(A)
    inside[7:13, 4:10, 9:16] = True
    assert g2.trapped_volume(1, 0, nz)[0] == int((inside & ~A).sum())
    # a column of A from z=nz-1 wrapping to z=0 is NOT joined across the z ends, but both pieces
    # touch an end plane, so neither is trapped; a droplet adjacent to z=0 only via the wrap is
    A3 = np.zeros_like(A)
    A3[1:4, 5:8, 5:8] = True                      # does not touch z=0 itself -> trapped (27)
    rA3 = np.where(A3, 0.9, 0.1)
    g3 = Lbm(mask, default_params(storage_bits=64))
    g3.set_density(rA3, 1.0 - rA3)
    assert g3.trapped_volume(0, 0, nz)[0] == 27


@pytest.mark.parametrize("shape", [(1, 9, 11), (12, 1, 1), (7, 1, 13), (2, 2, 2)])
def test_trapped_volume_degenerate_shapes(shape):
    rng = np.random.Generator(np.random.PCG64(5))
    mask = (rng.uniform(size=shape) < 0.2).astype(np.uint8)
    if mask.all():
        mask.flat[0] = 0
    rA = rng.uniform(0.0, 1.0, shape)
    rB = rng.uniform(0.0, 1.0, shape)
    o, g = _both(mask, rA, rB, default_params(storage_bits=64))
    for comp in (0, 1):
        no, mo = o.trapped_volume(comp, 0, shape[0])
        ng, mg = g.trapped_volume(comp, 0, shape[0])
        assert no == ng and abs(mo - mg) <= 1e-12 * max(1.0, mo)


def test_trapped_volume_snake_cluster_and_repeatability():
    """One long serpentine cluster (worst case for pointer chasing: the union-find chains are as
    long as the cluster) and a full-size-like rock; repeated calls return the same numbers."""
    nz, ny, nx = 64, 64, 64
    mask = np.zeros((nz, ny, nx), np.uint8)
    A = np.zeros((nz, ny, nx), bool)
    for z in range(2, nz - 2, 2):                 # rows joined alternately at either end
        A[z, 10, 4:60] = True
        A[z + 1, 10, 59 if (z // 2) % 2 else 4] = True
    A[nz - 2, 10, :] = False
    rA = np.where(A, 0.8, 0.2)
    o, g = _both(mask, rA, 1.0 - rA, default_params(storage_bits=64))
    no, mo = o.trapped_volume(0, 0, nz)
    for _ in range(3):
        ng, mg = g.trapped_volume(0, 0, nz)
        assert ng == no == int(A.sum()) and mg == pytest.approx(mo, rel=1e-13)
    c = make_config(4, size=64)
    o, g = _both(c["mask"], c["rhoA"], c["rhoB"], c["params"])
    o.step(20)
    g.step(20)
    first = None
    for _ in range(3):
        r = g.trapped_volume(0, 0, 64), g.trapped_volume(1, 8, 56)
        first = first or r
        assert r == first                          # bit-identical: fixed-order reduction
    assert first[0][0] == o.trapped_volume(0, 0, 64)[0]
    assert first[1][0] == o.trapped_volume(1, 8, 56)[0]


def test_trapped_volume_full_size_against_library_labelling():
    """Config 4's 256^3 rock (4.3 M fluid nodes, fp32 production build) with a synthetic blob
    field: the GPU result against scipy.ndimage.label + a label-graph merge across the periodic
    x,y wrap (a library routine, neither the oracle's flood fill nor the CUDA union-find)."""
    from scipy import ndimage
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components
    c = make_config(4)
    mask = c["mask"]
    nz = mask.shape[0]
    f = _blobs(mask.shape, 77, 3.0)
    rA = np.where(f > 0.8, 0.9, 0.1).astype(np.float64)
    rB = 1.0 - rA
    g = Lbm(mask, c["params"])
    g.set_density(rA, rB)
    for comp in (0, 1):
        phase = (mask == 0) & ((rA > rB) if comp == 0 else ~(rA > rB))
        lab, nl = ndimage.label(phase)                      # 6-connected, not periodic
        pairs = []
        for a, b in ((lab[:, :, 0], lab[:, :, -1]), (lab[:, 0, :], lab[:, -1, :])):
            both = (a > 0) & (b > 0)
            pairs.append(np.stack([a[both], b[both]]))
        pr = np.concatenate(pairs, axis=1)
        graph = coo_matrix((np.ones(pr.shape[1]), (pr[0], pr[1])), shape=(nl + 1, nl + 1))
        _, root = connected_components(graph, directed=False)
        cl = root[lab]                                       # cluster id per voxel (0 = background's)
        touching = np.zeros(root.max() + 1, bool)
        touching[np.unique(cl[0][phase[0]])] = True
        touching[np.unique(cl[-1][phase[-1]])] = True
        trapped = phase & ~touching[cl]
        for z0, z1 in ((0, nz), (40, 200)):
            n, m = g.trapped_volume(comp, z0, z1)
            assert n == int(trapped[z0:z1].sum()), (comp, z0, z1)
            want = float((rA if comp == 0 else rB)[z0:z1][trapped[z0:z1]].sum())
            assert abs(m - want) <= 1e-6 * max(1.0, want)
        if comp == 0:
            assert int(trapped.sum()) > 1000                 # the case is not trivial
