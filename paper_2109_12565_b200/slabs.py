"""Y-slab multi-GPU driver (host logic only; every lattice operation is a call of the C ABI, include/tlb.h "Y-SLABS").

One process per GPU owns a contiguous slab of rows of the nx x ny lattice (x stays periodic locally, the flat walls
live on the first / last slab).  Per time step and interior face, the 3 owned rows next to the face (all 27 planes)
travel to the neighbour's halo rows: `torch.distributed` point-to-point (NCCL over NVLink on GPUs, gloo in the CPU
tests of the host logic) on a side stream, overlapped with the fused kernel on the interior rows.  The population
buffers keep the 27 plane rows of a lattice row together, so those 3 rows are one contiguous block on both sides:
the transport reads the sender's state and writes the receiver's halo rows directly (tlb_halo_region, zero copy);
tlb_halo_pack / _unpack into separate buffers remain as the staged alternative (`zero_copy=False`).  Observables are six partial sums per slab, all-reduced and finished by tlb_observables_from_sums.
The multi-GPU path is the paper's stated future work.

This module holds none of the method's arithmetic and never imports anything under oracle/.
"""
import numpy as np

HALO = 3  # rows per interior face; must equal kHalo of csrc/tlb_internal.cuh (checked against tlb_slab_layout)


def partition(ny, world):
    """Contiguous, near-equal row ranges [(y0, y1)] of `world` slabs; the first ny % world slabs get one more row."""
    if world < 1 or ny < world:
        raise ValueError("cannot split %d rows into %d slabs" % (ny, world))
    base, extra = divmod(ny, world)
    out, y = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((y, y + n))
        y += n
    return out


def neighbours(rank, world, periodic_y):
    """(rank below, rank above) across the low / high face, None where the face is a flat wall."""
    lo = rank - 1 if rank > 0 else (world - 1 if periodic_y else None)
    hi = rank + 1 if rank < world - 1 else (0 if periodic_y else None)
    return lo, hi


def slab_layout(ny, y0, y1, periodic_y, halo=HALO):
    """Local lattice of the slab [y0, y1): the same numbers tlb_slab_layout reports."""
    halo_lo = 0 if (y0 == 0 and not periodic_y) else halo
    halo_hi = 0 if (y1 == ny and not periodic_y) else halo
    if (halo_lo or halo_hi) and y1 - y0 < halo:
        raise ValueError("a slab next to a halo face needs at least %d rows" % halo)
    return dict(ny_local=(y1 - y0) + halo_lo + halo_hi, own0=halo_lo, own1=halo_lo + (y1 - y0),
                y_off=y0 - halo_lo, halo_lo=halo_lo, halo_hi=halo_hi)


def local_rows(ny, y0, y1, periodic_y, halo=HALO):
    """Row of the whole lattice behind each local row (halo rows wrap when the lattice is periodic in y)."""
    lay = slab_layout(ny, y0, y1, periodic_y, halo)
    rows = lay["y_off"] + np.arange(lay["ny_local"])
    return rows % ny if periodic_y else rows


def face_rows(lay, face, halo=HALO):
    """(rows packed for `face`, halo rows unpacked beyond `face`) as local row indices; face 0 = low y, 1 = high."""
    if face == 0:
        return np.arange(lay["own0"], lay["own0"] + halo), np.arange(lay["own0"] - halo, lay["own0"])
    return np.arange(lay["own1"] - halo, lay["own1"]), np.arange(lay["own1"], lay["own1"] + halo)


def exchange(dist, send, recv, lo, hi, rank):
    """Move the packed faces: send[0] (my low rows) -> rank `lo`, send[1] (my high rows) -> rank `hi`; recv[0] <- what
    `lo` sent upwards, recv[1] <- what `hi` sent downwards.  When lo == hi (two slabs of a periodic lattice) both
    directions go to the same peer.  gloo tells them apart by the tags; NCCL ignores tags and pairs the k-th send to a
    peer with the k-th receive that peer posts for this rank, so the pairing then rests on the ORDER below -- send up,
    send down, receive the upward face, receive the downward face -- being the same on both ranks.  Keep it.  A face whose neighbour is this rank itself (one slab of a periodic lattice)
    is a local copy.  Returns when the receives have completed on the current stream / thread."""
    UP, DOWN = 0, 1
    ops = []
    if hi is not None:
        if hi == rank:
            recv[0].copy_(send[1])
        else:
            ops.append(dist.P2POp(dist.isend, send[1], hi, tag=UP))
    if lo is not None:
        if lo == rank:
            recv[1].copy_(send[0])
        else:
            ops.append(dist.P2POp(dist.isend, send[0], lo, tag=DOWN))
    if lo is not None and lo != rank:
        ops.append(dist.P2POp(dist.irecv, recv[0], lo, tag=UP))
    if hi is not None and hi != rank:
        ops.append(dist.P2POp(dist.irecv, recv[1], hi, tag=DOWN))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()


class Slab:
    """One y-slab of the lattice on one GPU: a binding.TLB slab handle plus its halo buffers.  Arrays handed to the
    set_* calls are those of the WHOLE lattice (numpy); the slab takes the rows it needs."""

    def __init__(self, nx, ny, rank, world, params=None, device="cuda:0", stream=None, **overrides):
        from . import binding
        self.rank, self.world = rank, world
        self.y0, self.y1 = partition(ny, world)[rank]
        self.t = binding.TLB(nx, ny, params=params, device=device, stream=stream, slab=(self.y0, self.y1), **overrides)
        self.periodic_y = bool(self.t.params.periodic_y)
        self.lo, self.hi = neighbours(rank, world, self.periodic_y)
        lay = slab_layout(ny, self.y0, self.y1, self.periodic_y)
        got = dict(ny_local=self.t.ny, own0=self.t.own0, own1=self.t.own1, y_off=self.t.y_off,
                   halo_lo=self.t.halo_lo, halo_hi=self.t.halo_hi)
        assert lay == got, (lay, got)  # this module and the library agree on the geometry
        self.rows = local_rows(ny, self.y0, self.y1, self.periodic_y)
        self.send = [self.t.halo_buffer() if nb is not None else None for nb in (self.lo, self.hi)]
        self.recv = [self.t.halo_buffer() if nb is not None else None for nb in (self.lo, self.hi)]

    # ---- state ------------------------------------------------------------------------------
    def _take(self, a):
        return np.ascontiguousarray(np.asarray(a)[..., self.rows, :])

    def set_solid(self, solid):
        self.t.set_solid(self._take(solid))

    def set_fields(self, rho_A, rho_B, T):
        self.t.set_fields(self._take(rho_A), self._take(rho_B), self._take(T))

    def set_populations(self, fA, fB, g):
        self.t.set_populations(self._take(fA), self._take(fB), self._take(g))

    def init(self, seed):
        self.t.init(seed)  # the seeded recipe is stated on the whole lattice: every slab fills its own rows and halos

    def owned(self, a):
        """Owned rows of a local array (fields, populations)."""
        return a[..., self.t.own0:self.t.own1, :]

    # ---- one time step in two halves, the exchange in between ---------------------------------
    zero_copy = True  # exchange straight out of / into the population buffers (tlb_halo_region)

    def regions(self):
        """(send, recv): per face the views of the rows to export and of the halo rows to fill, in the buffer this step writes."""
        send = [self.t.halo_region(f, 0) if nb is not None else None for f, nb in enumerate((self.lo, self.hi))]
        recv = [self.t.halo_region(f, 1) if nb is not None else None for f, nb in enumerate((self.lo, self.hi))]
        return send, recv

    def begin_step(self):
        self.t.slab_step_edges()
        if self.zero_copy:
            self.send, self.recv = self.regions()
        else:
            for face in (0, 1):
                if self.send[face] is not None:
                    self.t.halo_pack(face, self.send[face])
        self.t.slab_step_interior()

    def end_step(self):
        if not self.zero_copy:
            for face in (0, 1):
                if self.recv[face] is not None:
                    self.t.halo_unpack(face, self.recv[face])
        self.t.slab_step_finish()


def step_local(slabs, n=1):
    """Advance slabs that live in ONE process (one GPU, one stream) by n steps: the exchange is a device copy.
    This is the single-GPU stand-in used by the tests; kernels of different slabs never wait on one another."""
    world = len(slabs)
    for _ in range(n):
        for s in slabs:
            s.begin_step()
        for s in slabs:
            if s.hi is not None:
                slabs[s.hi].recv[0].copy_(s.send[1])
            if s.lo is not None:
                slabs[s.lo].recv[1].copy_(s.send[0])
        for s in slabs:
            s.end_step()
    return world


class DistributedSlab(Slab):
    """A slab whose neighbours are other ranks of a torch.distributed group (one process per GPU, NCCL)."""

    def __init__(self, nx, ny, params=None, device="cuda:0", **overrides):
        import torch
        import torch.distributed as dist
        self.torch, self.dist = torch, dist
        super().__init__(nx, ny, dist.get_rank(), dist.get_world_size(), params=params, device=device, **overrides)
        self.comm_stream = torch.cuda.Stream(device=self.t.device)
        self.packed, self.arrived = torch.cuda.Event(), torch.cuda.Event()
        # A gloo group cannot send device memory: the faces are then staged through host tensors (what a node without
        # GPU-direct transport would do, and what lets two ranks share ONE GPU in the tests).  NCCL reads and writes the
        # population buffers directly.
        self.host_staged = dist.get_backend() == "gloo"

    def _exchange(self):
        """Runs on the side stream, after the edge rows of this step: move the faces to / from the neighbours."""
        if not self.host_staged:
            exchange(self.dist, self.send, self.recv, self.lo, self.hi, self.rank)
            return
        send_h = [None if s is None else s.cpu() for s in self.send]          # synchronous copies on the side stream
        recv_h = [None if r is None else self.torch.empty_like(r, device="cpu") for r in self.recv]
        exchange(self.dist, send_h, recv_h, self.lo, self.hi, self.rank)
        for r, h in zip(self.recv, recv_h):
            if r is not None:
                r.copy_(h)

    def step(self, n=1):
        torch, main = self.torch, self.t.stream
        for _ in range(n):
            self.t.slab_step_edges()
            if self.zero_copy:
                self.send, self.recv = self.regions()
            else:
                for face in (0, 1):
                    if self.send[face] is not None:
                        self.t.halo_pack(face, self.send[face])
            self.packed.record(main)
            self.t.slab_step_interior()              # overlaps the exchange below
            with torch.cuda.stream(self.comm_stream):
                self.comm_stream.wait_event(self.packed)
                self._exchange()
                self.arrived.record(self.comm_stream)
            main.wait_event(self.arrived)
            self.end_step()

    def observables(self):
        """dict(mass_A, mass_B, E, Nu) of the whole lattice: all-reduce of the slabs' six sums."""
        sums = self.t.observable_sums()
        if self.world > 1:
            if self.host_staged:
                host = sums.cpu()
                self.dist.all_reduce(host, op=self.dist.ReduceOp.SUM)
                sums.copy_(host)
            else:
                self.dist.all_reduce(sums, op=self.dist.ReduceOp.SUM)
        return self.t.observables_from_sums(sums)
