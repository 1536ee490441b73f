"""z-slab sharding of the two-component D3Q19 step across GPUs (C ABI:
include/lbm.h "z-slab sharding").

The paper is single-GPU; its step has two grid-wide dependencies per time step
(Eq. 11/13: forces need the neighbours' rho(t); Eq. 15: a wall solid's rho~(t) needs its fluid
neighbours' rho(t)) and one transport across a cut (Eq. 1 LHS).  A box that is periodic in z is cut
into contiguous z-slabs balanced by fluid-node count; every slab is one `Lbm(slab=True)` context
with two halo planes per end, and a step is

    slab_density(0)  [boundary planes]   -> psi exchange starts
    slab_density(1)  [interior]          -> psi exchange completes
    slab_collide(0)  [wall pass, boundary tiles, pack] -> population exchange starts
    slab_collide(1)  [interior tiles]    -> population exchange completes
    slab_unpack

so that both exchanges run beside the interior work of the same pass.

All arithmetic runs in the library's kernels; this module only partitions the mask, slices the
initial state and moves the DEVICE exchange buffers between neighbours:

  * `RingTransport`   one slab per process / GPU; `torch.distributed.batch_isend_irecv` on the
                      buffers (NCCL send/recv over NVLink on GPUs; gloo in the CPU tests of the
                      choreography);
  * in-process copies when all slabs live on one GPU (`SlabLbm(..., world=None)`): the slabs run one
                      after another on one stream -- the single-GPU check that the sharded step
                      is bit-identical to the unsharded one, not a performance mode.
"""
import numpy as np

from .lbm import Lbm

GHOST = 2  # LBM_SLAB_GHOST


def partition(mask, parts):
    """Cut [0, nz) into `parts` contiguous z-ranges with nearly equal fluid-node counts, each at
    least GHOST planes thick.  Returns [(z0, z1), ...]."""
    nz = mask.shape[0]
    if parts < 1 or nz < GHOST * parts:
        raise ValueError(f"cannot cut {nz} planes into {parts} slabs of >= {GHOST} planes")
    per_plane = (np.asarray(mask).reshape(nz, -1) == 0).sum(axis=1).astype(np.int64)
    cum = np.concatenate([[0], np.cumsum(per_plane)])
    total = int(cum[-1])
    cuts = [0]
    for k in range(1, parts):
        z = int(np.searchsorted(cum, total * k / parts, side="left"))
        z = max(z, cuts[-1] + GHOST)                 # minimum thickness of the slab below
        z = min(z, nz - GHOST * (parts - k))         # leave room for the slabs above
        cuts.append(z)
    cuts.append(nz)
    return [(cuts[k], cuts[k + 1]) for k in range(parts)]


def local_planes(nz, z0, z1, halo=(1, 1)):
    """Global z index of every plane of the slab's local box: the owned planes [z0, z1) plus GHOST
    halo planes at each end that is a cut (they wrap periodically)."""
    return np.arange(z0 - GHOST * halo[0], z1 + GHOST * halo[1]) % nz


def local_box(a, z0, z1, halo=(1, 1)):
    """Slice a global [z, y, x] (or [q, z, y, x]) array to the slab's local box."""
    a = np.asarray(a)
    ax = a.ndim - 3
    return np.ascontiguousarray(np.take(a, local_planes(a.shape[ax], z0, z1, halo), axis=ax))


def halo_flags(r, parts, z_open):
    """(low, high): 1 = that end of slab r is a cut; 0 = the end of a z-open box."""
    return (0 if (z_open and r == 0) else 1, 0 if (z_open and r == parts - 1) else 1)


class _DeviceBytes:
    """A span of device memory owned by an lbm_ctx, exposed through __cuda_array_interface__ so
    that torch can alias it (no copy)."""

    def __init__(self, ptr, nbytes, keepalive):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1",
                                         "data": (ptr, False), "version": 2}
        self._keepalive = keepalive


def buffer_tensor(sim, which):
    """uint8 torch tensor aliasing exchange buffer `which` of a slab context (None if empty)."""
    import torch
    ptr, nbytes = sim.slab_buffer(which)
    if nbytes == 0:
        return None
    return torch.as_tensor(_DeviceBytes(ptr, nbytes, sim),
                           device=torch.device("cuda", torch.cuda.current_device()))


class RingTransport:
    """Neighbour exchange on the periodic ring of slabs, one slab per rank.  `exchange(send_lo,
    send_hi, recv_lo, recv_hi)`: my low-face message goes to rank-1 and lands in its high-face
    receive buffer, my high-face message goes to rank+1 and lands in its low-face buffer.  Posting
    order (send up, send down, receive from below, receive from above) keeps the two messages
    between the same pair of ranks (world size 2) matched.  A None tensor is an empty message; both
    ends see it empty (the sizes derive from the same mask planes)."""

    def __init__(self, rank, world, group=None, stage_host=None):
        self.rank, self.world, self.group = rank, world, group
        # NCCL moves device buffers directly.  Any other backend (gloo) gets the messages staged
        # through pinned host buffers: slower, but the same choreography -- it is what the
        # two-process test on one GPU runs, where NCCL refuses two ranks on one device.
        if stage_host is None and world > 1:
            import torch.distributed as dist
            stage_host = dist.get_backend(group) != "nccl"
        self.stage_host = bool(stage_host)
        self._pinned = {}

    def _host(self, t, key):
        import torch
        h = self._pinned.get(key)
        if h is None or h.shape != t.shape or h.dtype != t.dtype:
            h = torch.empty(t.shape, dtype=t.dtype, pin_memory=t.is_cuda)
            self._pinned[key] = h
        return h

    def exchange(self, send_lo, send_hi, recv_lo, recv_hi):
        self.finish(self.start(send_lo, send_hi, recv_lo, recv_hi))

    @staticmethod
    def finish(works):
        for w in works:
            if isinstance(w, tuple):      # staged receive: (work, host buffer, device buffer)
                w[0].wait()
                w[2].copy_(w[1], non_blocking=True)
            else:
                w.wait()   # NCCL: stream-ordered on CUDA tensors, no host block

    def start(self, send_lo, send_hi, recv_lo, recv_hi):
        """Post the four messages; returns the handles `finish` waits on.  On CUDA tensors the
        transfers run on NCCL's stream, after everything enqueued so far on the current stream and
        beside whatever is enqueued next."""
        if self.world == 1:
            if recv_lo is not None:
                recv_lo.copy_(send_hi)
            if recv_hi is not None:
                recv_hi.copy_(send_lo)
            return []
        import torch.distributed as dist
        up, down = (self.rank + 1) % self.world, (self.rank - 1) % self.world
        if self.stage_host:
            return self._start_staged(send_lo, send_hi, recv_lo, recv_hi, up, down)
        ops = []
        if send_hi is not None:
            ops.append(dist.P2POp(dist.isend, send_hi, up, self.group))
        if send_lo is not None:
            ops.append(dist.P2POp(dist.isend, send_lo, down, self.group))
        if recv_lo is not None:
            ops.append(dist.P2POp(dist.irecv, recv_lo, down, self.group))
        if recv_hi is not None:
            ops.append(dist.P2POp(dist.irecv, recv_hi, up, self.group))
        return dist.batch_isend_irecv(ops) if ops else []

    def _start_staged(self, send_lo, send_hi, recv_lo, recv_hi, up, down):
        import torch
        import torch.distributed as dist
        works = []
        hs_hi = hs_lo = None
        if send_hi is not None:
            hs_hi = self._host(send_hi, "s_hi")
            hs_hi.copy_(send_hi, non_blocking=True)
        if send_lo is not None:
            hs_lo = self._host(send_lo, "s_lo")
            hs_lo.copy_(send_lo, non_blocking=True)
        if (send_hi is not None and send_hi.is_cuda) or (send_lo is not None and send_lo.is_cuda):
            torch.cuda.current_stream().synchronize()   # the host copies must be complete
        if hs_hi is not None:
            works.append(dist.isend(hs_hi, up, group=self.group))
        if hs_lo is not None:
            works.append(dist.isend(hs_lo, down, group=self.group))
        if recv_lo is not None:
            h = self._host(recv_lo, "r_lo")
            works.append((dist.irecv(h, down, group=self.group), h, recv_lo))
        if recv_hi is not None:
            h = self._host(recv_hi, "r_hi")
            works.append((dist.irecv(h, up, group=self.group), h, recv_hi))
        return works


class SlabLbm:
    """A simulation cut into z-slabs (z periodic, or z open with the inlet plane on the first and
    the outlet plane on the last slab).

    world=None: all `parts` slabs are created in this process on the current GPU and stepped one
    after another (validation of the sharded path on one GPU).
    world=N, rank=r: this process owns slab r of N (one process per GPU); exchanges go through
    torch.distributed's default (or the given) process group.

    Global arrays are [z, y, x]; `get_macroscopic` returns the owned planes of this process
    (all planes when world is None)."""

    def __init__(self, mask, params, parts=None, rank=None, world=None, group=None, options=None,
                 native=None):
        mask = np.ascontiguousarray(mask, np.uint8)
        self.shape = mask.shape
        self.world = world
        self.z_open = int(params["z_open"]) != 0
        nparts = world if world is not None else (parts or 1)
        self.ranges = partition(mask, nparts)
        self.mine = [rank] if world is not None else list(range(nparts))
        self.halo = [halo_flags(r, nparts, self.z_open) for r in range(nparts)]
        self.sims = [Lbm(local_box(mask, *self.ranges[r], self.halo[r]), params, slab=True,
                         halo=self.halo[r], options=options) for r in self.mine]
        # fluid nodes per global plane (host copy of the mask statistics the queries weight with)
        self._plane_fluid = (mask.reshape(mask.shape[0], -1) == 0).sum(axis=1).astype(np.int64)
        self.num_fluid = sum(s.num_owned for s in self.sims)
        self._ring = RingTransport(rank, world, group) if world is not None else None
        self._buf = [[buffer_tensor(s, w) for w in range(12)] for s in self.sims]
        # native = the step and its exchanges run inside the library (lbm_slab_step: NCCL send /
        # recv on a side stream); default whenever every rank has its own GPU, i.e. with the NCCL
        # backend (or a single rank).  Otherwise the step is sequenced here, call by call, with the
        # exchanges through RingTransport (gloo: the CPU tests and several ranks on one GPU).
        if native is None:
            native = world is not None and (world == 1 or self._backend(group) == "nccl")
        self.native = bool(native) and world is not None
        if self.native:
            self.sims[0].slab_comm_init(self._comm_id(rank, world, group), rank, world)

    @staticmethod
    def _backend(group):
        import torch.distributed as dist
        return dist.get_backend(group) if dist.is_initialized() else None

    @staticmethod
    def _comm_id(rank, world, group):
        """The ring's rendezvous token: made on rank 0, broadcast through torch.distributed."""
        from .lbm import lbm_comm_unique_id
        if world == 1:
            return lbm_comm_unique_id()
        import torch
        import torch.distributed as dist
        dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
        t = torch.zeros(128, dtype=torch.uint8, device=dev)
        if rank == 0:
            t.copy_(torch.frombuffer(bytearray(lbm_comm_unique_id()), dtype=torch.uint8))
        dist.broadcast(t, src=0, group=group)
        return bytes(t.cpu().numpy().tobytes())

    def close(self):
        self._buf = []
        for s in self.sims:
            s.close()
        self.sims = []

    # -- exchanges: kind 0 = psi (buffers 0,1 -> 2,3), kind 1 = populations (4,5 -> 6,7),
    #    kind 2 = cluster flags of the trapped-volume query (8,9 -> 10,11)
    def _exchange_start(self, kind):
        b = 4 * kind
        if self.native:     # one grouped ncclSend/ncclRecv round inside the library, in stream order
            self.sims[0].slab_exchange(kind)
            return []
        if self._ring is not None:
            buf = self._buf[0]
            return self._ring.start(buf[b], buf[b + 1], buf[b + 2], buf[b + 3])
        n = len(self.sims)
        for r in range(n):
            lo, hi = self._buf[(r - 1) % n], self._buf[(r + 1) % n]
            if self._buf[r][b + 2] is not None:
                self._buf[r][b + 2].copy_(lo[b + 1])   # my low halo <- lower slab's high face
            if self._buf[r][b + 3] is not None:
                self._buf[r][b + 3].copy_(hi[b])       # my high halo <- upper slab's low face
        return []

    def _density_and_psi_halo(self):
        for s in self.sims:
            s.slab_density(0)
        works = self._exchange_start(0)
        for s in self.sims:
            s.slab_density(1)
        RingTransport.finish(works)

    def step(self, n=1):
        if self.native:
            self.sims[0].slab_step(int(n))
            return
        for _ in range(int(n)):
            self._density_and_psi_halo()
            for s in self.sims:
                s.slab_collide(0)
            works = self._exchange_start(1)
            for s in self.sims:
                s.slab_collide(1)
            RingTransport.finish(works)
            for s in self.sims:
                s.slab_unpack()

    def sync(self):
        for s in self.sims:
            s.sync()

    def set_density(self, rhoA, rhoB):
        for s, r in zip(self.sims, self.mine):
            z0, z1 = self.ranges[r]
            s.set_density(local_box(rhoA, z0, z1, self.halo[r]),
                          local_box(rhoB, z0, z1, self.halo[r]))

    def set_populations(self, comp, f):
        for s, r in zip(self.sims, self.mine):
            s.set_populations(comp, local_box(f, *self.ranges[r], self.halo[r]))

    def set_boundary(self, inlet_value, outlet_rho):
        for s in self.sims:
            s.set_boundary(inlet_value, outlet_rho)

    def _owned(self, a, r):
        lo, hi = self.halo[r]
        return a[..., GHOST * lo:a.shape[-3] - GHOST * hi, :, :]

    def get_populations(self, comp):
        return np.concatenate([self._owned(s.get_populations(comp), r)
                               for s, r in zip(self.sims, self.mine)], axis=1)

    def _weighted_mean(self, call, z0, z1):
        """sum over slabs of (plane-range mean x fluid nodes in it) / nodes: how a query over the
        global planes [z0, z1) is put together from the per-slab library queries (local planes)."""
        self._density_and_psi_halo()
        num, den = 0.0, 0
        for s, r in zip(self.sims, self.mine):
            a, b = max(z0, self.ranges[r][0]), min(z1, self.ranges[r][1])
            n = int(self._plane_fluid[a:b].sum()) if b > a else 0
            if n == 0:
                continue
            off = GHOST * self.halo[r][0] - self.ranges[r][0]
            num += call(s, a + off, b + off) * n
            den += n
        if self.world is not None and self.world > 1:
            import torch
            import torch.distributed as dist
            dev = "cuda" if dist.get_backend(self._ring.group) == "nccl" else "cpu"
            t = torch.tensor([num, float(den)], dtype=torch.float64, device=dev)
            dist.all_reduce(t, group=self._ring.group)
            num, den = float(t[0]), int(round(float(t[1])))
        if den == 0:
            raise ValueError("no fluid node in the z-range")
        return num / den

    def saturation(self, comp, z0=0, z1=None):
        z1 = self.shape[0] if z1 is None else z1
        return self._weighted_mean(lambda s, a, b: s.saturation(comp, a, b), z0, z1)

    def mean_pressure(self, z0=0, z1=None):
        z1 = self.shape[0] if z1 is None else z1
        return self._weighted_mean(lambda s, a, b: s.mean_pressure(a, b), z0, z1)

    def get_macroscopic(self, fields=("rhoA", "rhoB", "ux", "uy", "uz", "P")):
        self._density_and_psi_halo()   # the library's slab getter needs psi of the current state
        parts = [s.get_macroscopic(fields) for s in self.sims]
        return {k: np.concatenate([self._owned(p[k], r) for p, r in zip(parts, self.mine)], axis=0)
                for k in parts[0]}

    def _sum_over_ranks(self, values):
        if self.world is None or self.world == 1:
            return values
        import torch
        import torch.distributed as dist
        dev = "cuda" if dist.get_backend(self._ring.group) == "nccl" else "cpu"
        t = torch.tensor(values, dtype=torch.float64, device=dev)
        dist.all_reduce(t, group=self._ring.group)
        return [float(v) for v in t.cpu()]

    def trapped_volume(self, comp, z0=0, z1=None):
        """(nodes, mass) of the phase-`comp` clusters in the global planes [z0, z1) that reach
        neither z = 0 nor z = nz-1 (reading R15): per-slab connected components, then the
        end-connected flag is passed across the cuts until no slab changes (include/lbm.h
        lbm_slab_ccl_*).  Nothing connects across the periodic wrap."""
        nz = self.shape[0]
        z1 = nz if z1 is None else z1
        last = len(self.ranges) - 1
        self._density_and_psi_halo()
        for s, r in zip(self.sims, self.mine):
            s.slab_ccl_begin(comp, r == 0, r == last)
        while True:
            for s in self.sims:
                s.slab_ccl_export()
            RingTransport.finish(self._exchange_start(2))
            changed = sum(s.slab_ccl_import(r > 0, r < last) for s, r in zip(self.sims, self.mine))
            if self._sum_over_ranks([float(changed)])[0] == 0:
                break
        nodes, mass = 0, 0.0
        for s, r in zip(self.sims, self.mine):
            a, b = max(z0, self.ranges[r][0]), min(z1, self.ranges[r][1])
            if b <= a:
                a = b = self.ranges[r][0]          # empty range: the session still has to end
            off = GHOST * self.halo[r][0] - self.ranges[r][0]
            n, m = s.slab_ccl_finish(a + off, b + off)
            nodes += n
            mass += m
        nodes, mass = self._sum_over_ranks([float(nodes), mass])
        return int(round(nodes)), mass

    def diagnostics(self):
        """(mass[2], momentum[3]) over the owned nodes of this process; summed over all ranks when
        distributed (one all_reduce of 5 doubles)."""
        m, j = np.zeros(2), np.zeros(3)
        for s in self.sims:
            a, b = s.diagnostics()
            m += a
            j += b
        if self.world is not None and self.world > 1:
            import torch
            import torch.distributed as dist
            dev = "cuda" if dist.get_backend(self._ring.group) == "nccl" else "cpu"
            t = torch.tensor(np.concatenate([m, j]), dtype=torch.float64, device=dev)
            dist.all_reduce(t, group=self._ring.group)
            t = t.cpu().numpy()
            m, j = t[:2], t[2:]
        return m, j
