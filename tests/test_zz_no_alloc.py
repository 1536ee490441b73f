"""lbm_trapped_volume_static: the trapped-volume query (reading R15) for callers
that cannot allocate -- its union-find scratch is a file-scope device array of the library
(include/lbm.h: at most LBM_STATIC_MAX_NODES = 2^20 fluid nodes; 8 MiB held per GPU).  Checked
against the existing lbm_trapped_volume (same kernels: node count and mass identical) on two calls
in a row, which share the array and see each other's leftovers.

This file is collected last on purpose (the suite runs with `pytest -x`)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

LBM_STATIC_MAX_NODES = 1 << 20


def _blobs(shape, seed, sigma):
    rng = np.random.Generator(np.random.PCG64(seed))
    f = rng.standard_normal(shape)
    k = [np.fft.fftfreq(n) for n in shape]
    kk = k[0][:, None, None] ** 2 + k[1][None, :, None] ** 2 + k[2][None, None, :] ** 2
    f = np.real(np.fft.ifftn(np.fft.fftn(f) * np.exp(-2 * (np.pi * sigma) ** 2 * kk)))
    return f / f.std()


def _case(shape, solid, seed, bits):
    from paper_2207_01534_b200 import Lbm
    from workloads import default_params
    rng = np.random.Generator(np.random.PCG64(seed))
    mask = (rng.uniform(size=shape) < solid).astype(np.uint8)
    f = _blobs(shape, seed + 1, 2.5)
    rA = np.where(f > 0.3, 0.9, 0.1) + 0.01 * rng.uniform(size=shape)
    g = Lbm(mask, default_params(storage_bits=bits))
    g.set_density(rA, 1.0 - rA)
    return g


def test_static_scratch_matches_allocating_path_on_consecutive_calls():
    import torch
    big = _case((64, 60, 70), 0.3, 5, 32)        # 188 k fluid nodes
    small = _case((20, 18, 22), 0.2, 9, 64)      # 6 k: runs inside the big case's leftovers
    nz = 64
    found = 0
    # two calls in a row (and more): different component, z-range, context, size -- every one
    # against the allocating path on the same state
    for g, comp, z0, z1 in ((big, 0, 0, nz), (big, 1, 0, nz), (small, 0, 0, 20), (big, 0, 16, 48),
                            (small, 1, 3, 17), (big, 1, nz - 1, nz)):
        want = g.trapped_volume(comp, z0, z1)
        got = g.trapped_volume_static(comp, z0, z1)
        again = g.trapped_volume_static(comp, z0, z1)     # straight after itself
        assert got == want and again == want, (comp, z0, z1, want, got, again)
        found += want[0]
    assert found > 0                              # the cases do contain trapped clusters
    # after some time steps the state is no longer the initial one; still identical
    big.step(5)
    for comp in (0, 1):
        assert big.trapped_volume_static(comp) == big.trapped_volume(comp)
    # no allocation: torch's caching allocator (the library's only source of device memory)
    # sees no request during the static call, and one during the allocating call
    torch.cuda.synchronize()
    n0 = torch.cuda.memory_stats()["allocation.all.allocated"]
    r0 = torch.cuda.memory_reserved()
    big.trapped_volume_static(0)
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == n0
    assert torch.cuda.memory_reserved() == r0
    big.trapped_volume(0)
    assert torch.cuda.memory_stats()["allocation.all.allocated"] > n0
    big.close()
    small.close()


def test_static_scratch_rejects_boxes_beyond_its_maximum():
    from paper_2207_01534_b200 import Lbm, LbmError
    from workloads import default_params
    shape = (66, 128, 128)                        # 1 081 344 fluid nodes > 2^20
    g = Lbm(np.zeros(shape, np.uint8), default_params())
    assert g.num_fluid > LBM_STATIC_MAX_NODES
    g.set_density(np.full(shape, 0.6), np.full(shape, 0.4))
    with pytest.raises(LbmError) as e:
        g.trapped_volume_static(0)
    assert e.value.code == -1 and "LBM_STATIC_MAX_NODES" in str(e.value) and "1048576" in str(e.value)
    assert g.trapped_volume(0)[0] == 0            # the allocating path serves it
    g.close()
    # exactly at the limit it works
    shape = (64, 128, 128)
    g = Lbm(np.zeros(shape, np.uint8), default_params())
    assert g.num_fluid == LBM_STATIC_MAX_NODES
    rA = np.full(shape, 0.2)
    rA[20:30, 40:60, 40:60] = 0.8                 # one blob of A away from both ends: trapped
    g.set_density(rA, 1.0 - rA)
    assert g.trapped_volume_static(0) == g.trapped_volume(0)
    assert g.trapped_volume_static(0)[0] == 10 * 20 * 20
    g.close()
