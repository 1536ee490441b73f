"""CPU-side tests of the z-slab sharding: the partition, the halo lists the
library builds (against a brute-force numpy restatement of the rule in geometry.hpp), their
agreement between neighbouring slabs, and the ring exchange choreography on two gloo ranks.
No compute entry point is called (no GPU here)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2207_01534_b200 import lbm_build_slab_halo
from paper_2207_01534_b200 import slab
from workloads import sphere_pack_mask

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

E = np.array([(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1),
              (1, 1, 0), (-1, 1, 0), (1, -1, 0), (-1, -1, 0), (1, 0, 1), (-1, 0, 1), (1, 0, -1),
              (-1, 0, -1), (0, 1, 1), (0, -1, 1), (0, 1, -1), (0, -1, -1)])
DOWN = [i for i in range(19) if E[i, 2] == -1]
UP = [i for i in range(19) if E[i, 2] == +1]


def _rock(n=24, seed=11):
    return sphere_pack_mask(n, seed, 3.0, 5.0)[0]


def test_partition_covers_and_balances():
    m = _rock(32)
    for parts in (1, 2, 3, 5, 8):
        r = slab.partition(m, parts)
        assert r[0][0] == 0 and r[-1][1] == 32
        assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
        assert all(z1 - z0 >= slab.GHOST for z0, z1 in r)
        counts = [int((m[z0:z1] == 0).sum()) for z0, z1 in r]
        assert sum(counts) == int((m == 0).sum())
        # balanced to within two planes' worth of fluid nodes
        assert max(counts) - min(counts) <= 2 * 32 * 32
    with pytest.raises(ValueError):
        slab.partition(m, 17)          # 32 planes cannot hold 17 slabs of 2 planes
    thin = slab.partition(m, 16)
    assert all(z1 - z0 == 2 for z0, z1 in thin)


def test_local_box_wraps_periodically():
    a = np.arange(10)[:, None, None] * np.ones((10, 2, 2))
    b = slab.local_box(a, 0, 4)
    assert list(b[:, 0, 0]) == [8, 9, 0, 1, 2, 3, 4, 5]
    b = slab.local_box(a, 7, 10)
    assert list(b[:, 0, 0]) == [5, 6, 7, 8, 9, 0, 1]


def _brute_lists(ml):
    """(pack, unpack) per face as lists of (dir, local voxel), straight from the rule: an entry for
    (direction crossing the cut, destination node x) iff x and x - e_i are both fluid."""
    nz, ny, nx = ml.shape
    G = slab.GHOST
    out = {"pack": [], "unpack": []}
    for face in (0, 1):
        z_halo, z_own = (G - 1, G) if face == 0 else (nz - G, nz - G - 1)
        leaving, arriving = (DOWN, UP) if face == 0 else (UP, DOWN)
        pk, up = [], []
        for i in leaving:
            for y in range(ny):
                for x in range(nx):
                    xs, ys = (x - E[i, 0]) % nx, (y - E[i, 1]) % ny
                    if ml[z_halo, y, x] == 0 and ml[z_own, ys, xs] == 0:
                        pk.append((i, x + nx * (y + ny * z_halo)))
        for i in arriving:
            for y in range(ny):
                for x in range(nx):
                    xs, ys = (x - E[i, 0]) % nx, (y - E[i, 1]) % ny
                    if ml[z_own, y, x] == 0 and ml[z_halo, ys, xs] == 0:
                        up.append((i, x + nx * (y + ny * z_own)))
        out["pack"].append(np.array(pk, np.int32).reshape(-1, 2))
        out["unpack"].append(np.array(up, np.int32).reshape(-1, 2))
    return out


def test_halo_lists_match_bruteforce_rule():
    m = _rock(20, seed=12)
    z0, z1 = 5, 12
    ml = slab.local_box(m, z0, z1)
    h = lbm_build_slab_halo(ml)
    ref = _brute_lists(ml)
    for face in (0, 1):
        assert np.array_equal(h["pack"][face], ref["pack"][face])
        assert np.array_equal(h["unpack"][face], ref["unpack"][face])
        assert len(h["pack"][face]) > 0
    G = slab.GHOST
    assert h["n_owned"] == int((ml[G:-G] == 0).sum())
    assert h["psi_send"] == (int((ml[G:2 * G] == 0).sum()), int((ml[-2 * G:-G] == 0).sum()))
    assert h["psi_recv"] == (int((ml[:G] == 0).sum()), int((ml[-G:] == 0).sum()))


def _to_global(entries, planes, nx, ny):
    """(dir, local voxel) -> (dir, global voxel)"""
    d, v = entries[:, 0].astype(np.int64), entries[:, 1].astype(np.int64)
    z = planes[v // (nx * ny)]
    return np.stack([d, v % (nx * ny) + nx * ny * z], axis=1)


def test_neighbouring_slabs_agree_on_every_message():
    """What slab r packs at its high face is, entry by entry, what slab r+1 unpacks at its low
    face (same direction, same global voxel, same order), and vice versa; psi counts agree."""
    m = _rock(24, seed=13)
    nz, ny, nx = m.shape
    for parts in (1, 2, 3):
        ranges = slab.partition(m, parts)
        hs = [lbm_build_slab_halo(slab.local_box(m, *r)) for r in ranges]
        pl = [slab.local_planes(nz, *r) for r in ranges]
        for r in range(parts):
            u = (r + 1) % parts
            a = _to_global(hs[r]["pack"][1], pl[r], nx, ny)
            b = _to_global(hs[u]["unpack"][0], pl[u], nx, ny)
            assert np.array_equal(a, b)
            a = _to_global(hs[u]["pack"][0], pl[u], nx, ny)
            b = _to_global(hs[r]["unpack"][1], pl[r], nx, ny)
            assert np.array_equal(a, b)
            assert hs[r]["psi_send"][1] == hs[u]["psi_recv"][0]
            assert hs[u]["psi_send"][0] == hs[r]["psi_recv"][1]
        assert sum(h["n_owned"] for h in hs) == int((m == 0).sum())


def test_open_box_slabs_agree_and_have_no_message_at_the_box_ends():
    from workloads import make_config
    m = make_config(3, size=32)["mask"]
    nz, ny, nx = m.shape
    for parts in (2, 3):
        ranges = slab.partition(m, parts)
        flags = [slab.halo_flags(r, parts, True) for r in range(parts)]
        assert flags[0] == (0, 1) and flags[-1] == (1, 0)
        hs = [lbm_build_slab_halo(slab.local_box(m, *ranges[r], flags[r]), 1, flags[r])
              for r in range(parts)]
        pl = [slab.local_planes(nz, *ranges[r], flags[r]) for r in range(parts)]
        assert len(hs[0]["pack"][0]) == len(hs[0]["unpack"][0]) == 0
        assert len(hs[-1]["pack"][1]) == len(hs[-1]["unpack"][1]) == 0
        assert hs[0]["psi_send"][0] == hs[0]["psi_recv"][0] == 0
        assert hs[-1]["psi_send"][1] == hs[-1]["psi_recv"][1] == 0
        for r in range(parts - 1):
            a = _to_global(hs[r]["pack"][1], pl[r], nx, ny)
            b = _to_global(hs[r + 1]["unpack"][0], pl[r + 1], nx, ny)
            assert len(a) > 0 and np.array_equal(a, b)
            a = _to_global(hs[r + 1]["pack"][0], pl[r + 1], nx, ny)
            b = _to_global(hs[r]["unpack"][1], pl[r], nx, ny)
            assert np.array_equal(a, b)
            assert hs[r]["psi_send"][1] == hs[r + 1]["psi_recv"][0]
            assert hs[r + 1]["psi_send"][0] == hs[r]["psi_recv"][1]
        assert sum(h["n_owned"] for h in hs) == int((m == 0).sum())


def test_slab_rejects_too_thin_box():
    from paper_2207_01534_b200.lbm import LbmError
    with pytest.raises(LbmError):
        lbm_build_slab_halo(np.zeros((5, 4, 4), np.uint8))   # 1 owned plane + 4 halo planes


# ---------------------------------------------------------------- two gloo ranks

def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2207_01534_b200 import lbm_build_slab_halo as build_halo
    from paper_2207_01534_b200 import slab as sl
    from workloads import sphere_pack_mask as spm
    m = spm(24, 13, 3.0, 5.0)[0]
    nz, ny, nx = m.shape
    ranges = sl.partition(m, world)
    planes = sl.local_planes(nz, *ranges[rank])
    h = build_halo(sl.local_box(m, *ranges[rank]))
    ring = sl.RingTransport(rank, world)
    ok = True
    # the population messages: ship (dir, global voxel) of every packed entry to the neighbours and
    # compare with what this rank would unpack -- sizes and order must agree or the recv fails
    g = lambda e: torch.from_numpy(np.ascontiguousarray(
        np.stack([e[:, 0].astype(np.int64),
                  e[:, 1].astype(np.int64) % (nx * ny) + nx * ny * planes[e[:, 1] // (nx * ny)]],
                 axis=1)))
    send_lo, send_hi = g(h["pack"][0]), g(h["pack"][1])
    want_lo, want_hi = g(h["unpack"][0]), g(h["unpack"][1])
    recv_lo, recv_hi = torch.zeros_like(want_lo), torch.zeros_like(want_hi)
    for _ in range(3):   # repeated exchanges keep their pairing
        ring.exchange(send_lo, send_hi, recv_lo, recv_hi)
        ok = ok and torch.equal(recv_lo, want_lo) and torch.equal(recv_hi, want_hi)
    # the psi messages: plane-tagged payloads of the agreed sizes
    z0, z1 = ranges[rank]
    s_lo = torch.full((h["psi_send"][0],), float(z0))
    s_hi = torch.full((h["psi_send"][1],), float(z1 - 1))
    r_lo, r_hi = torch.zeros(h["psi_recv"][0]), torch.zeros(h["psi_recv"][1])
    ring.exchange(s_lo, s_hi, r_lo, r_hi)
    ok = ok and bool((r_lo == float((z0 - 1) % nz)).all()) and bool((r_hi == float(z1 % nz)).all())
    # empty messages are skipped on both ends
    ring.exchange(None, s_hi, r_lo, None)
    ok = ok and bool((r_lo == float((z0 - 1) % nz)).all())
    dist.barrier()
    out.put((rank, ok, h["n_owned"]))
    dist.destroy_process_group()


def test_ring_exchange_world_size_2_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert all(ok for _, ok, _ in res)
    m = _rock(24, seed=13)
    assert sum(n for _, _, n in res) == int((m == 0).sum())
