"""Domain decomposition of one box over several idfx contexts (block decomposition, device-side
pack / unpack of the two-cell halos, exchange direction by direction x -> y -> z; dt over "the entire
integration volume").  Host orchestration only: every cell is computed by the kernels of libidfx.so; this module decides
who talks to whom and in which order, and moves the packed slabs.

Two links carry the slabs and the dt reduction:
  * LocalLink  -- all sub-boxes live in this process (contexts on the same device, or on several devices of one
                  process); a slab packed by one context is unpacked by its neighbour straight from the buffer.
                  This is how one GPU tests the whole scheme: the result must equal the undecomposed run bit for bit.
  * DistLink   -- one sub-box per torch.distributed rank (NCCL over NVLink on GPUs, gloo in the CPU tests): slabs travel
                  with batched isend / irecv, dt with all_reduce(MAX).

The sub-box objects are duck-typed (`Idfx`, or the numpy stand-in of tests/test_decomp_host.py): they need
nstages, cycle_begin, stage_flux, stage_update, cycle_end, set_state_finish, dt_word, halo_count, halo_pack, halo_unpack,
halo_fill and new_buffer(count).
"""


def cart_coords(rank, dims):
    """Coordinates (cx, cy, cz) of `rank` in a (px, py, pz) grid of sub-boxes, x fastest."""
    px, py, pz = dims
    return rank % px, (rank // px) % py, rank // (px * py)


def cart_rank(coords, dims):
    px, py, pz = dims
    return coords[0] + px * (coords[1] + py * coords[2])


def neighbour(rank, dims, d, side, periodic=True):
    """Rank of the sub-box next to `rank` along direction d on its lower (side 0) or upper (side 1) side; None at the
    edge of a box that is not periodic."""
    c = list(cart_coords(rank, dims))
    c[d] += 1 if side else -1
    if c[d] < 0 or c[d] >= dims[d]:
        if not periodic:
            return None
        c[d] %= dims[d]
    return cart_rank(c, dims)


def split_extent(n, parts):
    """[(first cell, cell count)] of `parts` consecutive pieces of n cells, the first n % parts one cell longer."""
    base, rem = divmod(n, parts)
    out, lo = [], 0
    for p in range(parts):
        cnt = base + (1 if p < rem else 0)
        out.append((lo, cnt))
        lo += cnt
    return out


def sub_box(rank, dims, shape):
    """((x0, nx), (y0, ny), (z0, nz)) of the sub-box of `rank`; shape = (nx, ny, nz) of the whole box."""
    c = cart_coords(rank, dims)
    return tuple(split_extent(shape[d], dims[d])[c[d]] for d in range(3))


def wall_sides(rank, dims):
    """Bit mask for IDFX_OPT_OUTFLOW_SIDES of a box with outflow boundaries: the sides of `rank` with no neighbour."""
    return sum(1 << (2 * d + side) for d in range(3) for side in (0, 1) if neighbour(rank, dims, d, side, False) is None)


def exchange_dirs(dims):
    """Bit mask for IDFX_OPT_EXCHANGE_DIRS: the directions split over more than one sub-box."""
    return sum(1 << d for d in range(3) if dims[d] > 1)


class LocalLink:
    """All sub-boxes in this process: boxes[rank]."""

    def __init__(self, boxes, dims, periodic=True, push=True):
        assert len(boxes) == dims[0] * dims[1] * dims[2]
        self.boxes, self.dims, self.periodic = boxes, dims, periodic
        self.ranks = list(range(len(boxes)))
        # contexts of one process can write each other's ghost layers directly (idfx_halo_push: one launch per slab,
        # peer stores over NVLink between devices); otherwise pack -> buffer -> unpack
        self.push = push and all(hasattr(b, "halo_push") for b in boxes)

    def local(self):
        return list(zip(self.ranks, self.boxes))

    def reduce_dt(self):
        words = [b.dt_word() for b in self.boxes]   # one-element float64 tensors (views of the workspaces)
        m = words[0].clone()
        for w in words[1:]:
            m = m.maximum(w.to(m.device))
        for w in words:
            w.copy_(m)

    def exchange(self, d):
        if self.push:
            # a push reads active layers (and ghost layers of the directions already exchanged) and writes ghost layers of
            # direction d only, so the pushes of one direction do not depend on one another
            for r, b in self.local():
                for side in (0, 1):
                    nb = neighbour(r, self.dims, d, side, self.periodic)
                    if nb is None:
                        b.halo_fill(d, side, True)
                    else:
                        b.halo_push(d, side, self.boxes[nb])
            return
        # pack every slab first (a box's upper and lower slabs come from disjoint layers, and nobody's ghosts are touched
        # until all are packed), then unpack
        packed = {}
        for r, b in self.local():
            for side in (0, 1):
                buf = b.new_buffer(b.halo_count(d))
                b.halo_pack(d, side, buf)
                packed[(r, side)] = buf
        for r, b in self.local():
            for side in (0, 1):
                nb = neighbour(r, self.dims, d, side, self.periodic)
                if nb is None:
                    b.halo_fill(d, side, True)
                else:                      # my lower ghosts are my lower neighbour's upper layers, and vice versa
                    b.halo_unpack(d, side, b.adopt(packed[(nb, 1 - side)]))


class DistLink:
    """One sub-box per torch.distributed rank."""

    def __init__(self, box, dims, periodic=True, group=None, tags=True):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.tags = tags          # False: every message with tag 0, i.e. matched by order alone as NCCL does (tests)
        self.box, self.dims, self.periodic = box, dims, periodic
        self.rank = dist.get_rank(group)
        assert dist.get_world_size(group) == dims[0] * dims[1] * dims[2]

    def local(self):
        return [(self.rank, self.box)]

    def reduce_dt(self):
        self.dist.all_reduce(self.box.dt_word(), op=self.dist.ReduceOp.MAX, group=self.group)

    def exchange(self, d):
        b, dist = self.box, self.dist
        nbs = [neighbour(self.rank, self.dims, d, side, self.periodic) for side in (0, 1)]
        send = [b.new_buffer(b.halo_count(d)) for _ in (0, 1)]
        recv = [b.new_buffer(b.halo_count(d)) for _ in (0, 1)]   # recv[side]: what goes into my ghost layers of that side
        ops = []
        # NCCL has no tags: between two ranks the k-th send matches the k-th receive.  Everybody sends its lower slab, then its
        # upper slab; the lower slab of my upper neighbour fills my upper ghosts, so receives are posted upper first.  (With
        # two ranks along a periodic direction both neighbours are the same peer, and only this order pairs them correctly;
        # gloo also honours the tags.)
        for side in (0, 1):
            if nbs[side] is None:
                continue
            b.halo_pack(d, side, send[side])
            ops.append(dist.P2POp(dist.isend, send[side], nbs[side], self.group, tag=(2 * d + side) if self.tags else 0))
        for side in (1, 0):
            if nbs[side] is not None:
                ops.append(dist.P2POp(dist.irecv, recv[side], nbs[side], self.group, tag=(2 * d + (1 - side)) if self.tags else 0))
        if ops:
            for w in dist.batch_isend_irecv(ops):
                w.wait()
        for side in (0, 1):
            if nbs[side] is None:
                b.halo_fill(d, side, True)
            else:
                b.halo_unpack(d, side, recv[side])


class Decomposition:
    """Drives the sub-boxes of a link through whole cycles (include/idfx.h, "The cycle in pieces")."""

    def __init__(self, link):
        self.link = link

    def fill_ghosts(self):
        """a1 of the whole box: x, then y, then z, so that edges and corners arrive."""
        for d in range(3):
            if self.link.dims[d] > 1:
                self.link.exchange(d)
            else:
                for _, b in self.link.local():
                    for side in (0, 1):
                        b.halo_fill(d, side, not self.link.periodic)

    def finish_set_state(self):
        """After every sub-box has copied its part of the state in (set_state): ghosts of the face field, Bc and the
        conserved variables, ghosts of the primitives."""
        self.fill_ghosts()
        for _, b in self.link.local():
            b.set_state_finish()
        self.fill_ghosts()

    def cycle(self, cfl, dt=0.0):
        boxes = [b for _, b in self.link.local()]
        for b in boxes:
            b.cycle_begin(dt, cfl)
        for s in range(boxes[0].nstages):
            for b in boxes:
                b.stage_flux(s)
            if s == 0 and not dt > 0.0:
                self.link.reduce_dt()
            for b in boxes:
                b.stage_update(s)
            self.fill_ghosts()
        for b in boxes:
            b.cycle_end()

    def advance(self, nsteps, cfl):
        for _ in range(nsteps):
            self.cycle(cfl)
