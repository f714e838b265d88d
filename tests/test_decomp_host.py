"""Host orchestration of the domain decomposition (paper_2304_13746_b200/decomp.py) without a GPU:
topology, the x -> y -> z exchange order, and the max-reduction of dt, with world_size 2 over gloo (DistLink) and with all
sub-boxes in one process (LocalLink).  The sub-boxes are numpy stand-ins that implement the slab layout of
idfx_halo_pack / unpack / fill (include/idfx.h) and a toy "scheme" whose result needs every ghost cell, corners included:
a decomposed run must reproduce the single periodic box bit for bit.  The real kernels take the same calls in
tests/test_gpu_decomp.py."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2304_13746_b200 import decomp  # noqa: E402

NG = 2


class HostBox:
    """Stand-in for an Idfx sub-box: `nf` fields with two ghost layers; one 'stage' replaces every cell by a weighted sum
    over its 5 x 5 x 5 neighbourhood times the globally reduced word."""
    nstages = 2

    def __init__(self, field):                       # field [nf][nz][ny][nx]: the active cells
        nf, nz, ny, nx = field.shape
        self.n = (nx, ny, nz)
        self.f = np.full((nf, nz + 2 * NG, ny + 2 * NG, nx + 2 * NG), np.nan)
        self.f[:, NG:-NG, NG:-NG, NG:-NG] = field
        self.word = torch.zeros(1, dtype=torch.float64)
        self.log = []

    def active(self):
        return self.f[:, NG:-NG, NG:-NG, NG:-NG]

    # ---- slab geometry of include/idfx.h: NG layers normal to d, whole padded extent below d, active cells above d ----
    def _slab(self, d, first):
        sl = []
        for q in range(3):                           # q = 0 (x) is the last array axis
            if q == d:
                sl.append(slice(first + NG, first + 2 * NG))
            elif q < d:
                sl.append(slice(0, self.n[q] + 2 * NG))
            else:
                sl.append(slice(NG, self.n[q] + NG))
        return (slice(None), sl[2], sl[1], sl[0])

    def halo_count(self, d):
        return int(np.prod(self.f[self._slab(d, 0)].shape))

    def new_buffer(self, count):
        return torch.empty(count, dtype=torch.float64)

    def adopt(self, buf):
        return buf

    def halo_pack(self, d, side, buf):
        self.log.append(("pack", d, side))
        buf.numpy()[:] = self.f[self._slab(d, self.n[d] - NG if side else 0)].ravel()

    def halo_unpack(self, d, side, buf):
        self.log.append(("unpack", d, side))
        sl = self._slab(d, self.n[d] if side else -NG)
        self.f[sl] = buf.numpy().reshape(self.f[sl].shape)

    def halo_fill(self, d, side, zero_gradient):
        self.log.append(("fill", d, side))
        dst = self._slab(d, self.n[d] if side else -NG)
        if zero_gradient:
            src = self._slab(d, self.n[d] - 1 if side else 0)
            one = list(src)
            ax = 3 - d
            one[ax] = slice(src[ax].start, src[ax].start + 1)
            self.f[dst] = np.repeat(self.f[tuple(one)], NG, axis=ax)
        else:
            self.f[dst] = self.f[self._slab(d, 0 if side else self.n[d] - NG)]

    # ---- the cycle in pieces ----
    def cycle_begin(self, dt, cfl):
        self.word[0] = 0.0

    def stage_flux(self, s):
        assert not np.isnan(self.f).any(), "a ghost cell was never filled"
        acc = np.zeros_like(self.active())
        nx, ny, nz = self.n
        for dz in range(-NG, NG + 1):
            for dy in range(-NG, NG + 1):
                for dx in range(-NG, NG + 1):
                    w = 1.0 / ((1 + abs(dx)) * (2 + abs(dy)) * (3 + abs(dz))) * (1 + 0.1 * dx + 0.01 * dy + 0.001 * dz)
                    acc += w * self.f[:, NG + dz:NG + dz + nz, NG + dy:NG + dy + ny, NG + dx:NG + dx + nx]
        self.next = acc
        if s == 0:
            self.word[0] = float(np.abs(self.active()).max())

    def stage_update(self, s):
        self.active()[...] = self.next / (1.0 + float(self.word[0]))
        self.f[:, :NG], self.f[:, -NG:] = np.nan, np.nan       # the update writes no ghost layer
        self.f[:, :, :NG], self.f[:, :, -NG:] = np.nan, np.nan
        self.f[:, :, :, :NG], self.f[:, :, :, -NG:] = np.nan, np.nan

    def cycle_end(self):
        pass

    def set_state_finish(self):
        pass

    def dt_word(self):
        return self.word


def whole_field(shape, seed=3):
    nx, ny, nz = shape
    return np.random.default_rng(seed).standard_normal((2, nz, ny, nx))


def run_local(field, dims, periodic, cycles=2):
    shape = field.shape[:0:-1]
    n = dims[0] * dims[1] * dims[2]
    boxes, slices = [], []
    for r in range(n):
        (x0, nx), (y0, ny), (z0, nz) = decomp.sub_box(r, dims, shape)
        sl = (slice(None), slice(z0, z0 + nz), slice(y0, y0 + ny), slice(x0, x0 + nx))
        boxes.append(HostBox(field[sl]))
        slices.append(sl)
    dec = decomp.Decomposition(decomp.LocalLink(boxes, dims, periodic))
    dec.finish_set_state()
    dec.advance(cycles, 0.3)
    out = np.empty_like(field)
    for b, sl in zip(boxes, slices):
        out[sl] = b.active()
    return out, boxes


def test_topology():
    dims = (3, 2, 2)
    assert [decomp.cart_coords(r, dims) for r in (0, 1, 3, 6, 11)] == [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (2, 1, 1)]
    for r in range(12):
        assert decomp.cart_rank(decomp.cart_coords(r, dims), dims) == r
        for d in range(3):
            up = decomp.neighbour(r, dims, d, 1)
            assert decomp.neighbour(up, dims, d, 0) == r              # neighbours are mutual
    assert decomp.neighbour(2, dims, 0, 1) == 0 and decomp.neighbour(2, dims, 0, 1, periodic=False) is None
    assert decomp.neighbour(0, dims, 2, 0) == 6 and decomp.neighbour(0, dims, 1, 0, periodic=False) is None
    assert decomp.split_extent(37, 3) == [(0, 13), (13, 12), (25, 12)]
    assert decomp.sub_box(11, dims, (37, 26, 19)) == ((25, 12), (13, 13), (10, 9))
    assert decomp.exchange_dirs((2, 1, 4)) == 0b101 and decomp.exchange_dirs((1, 1, 1)) == 0
    assert decomp.wall_sides(0, (2, 1, 1)) == 0b111101 and decomp.wall_sides(1, (2, 1, 1)) == 0b111110


@pytest.mark.parametrize("periodic", [True, False])
@pytest.mark.parametrize("dims", [(2, 1, 1), (1, 2, 1), (1, 1, 2), (2, 2, 2), (3, 2, 1)])
def test_local_link_reproduces_the_single_box(dims, periodic):
    field = whole_field((13, 10, 9))
    one, _ = run_local(field, (1, 1, 1), periodic)
    many, boxes = run_local(field, dims, periodic)
    assert np.array_equal(one, many)
    assert not np.array_equal(one, field)
    # every ghost fill went x, then y, then z
    for b in boxes:
        fills, cur = [], []
        for op in b.log:                              # a new ghost fill starts where the direction drops back to x
            if cur and op[1] < cur[-1]:
                fills.append(cur)
                cur = []
            cur.append(op[1])
        fills.append(cur)
        assert len(fills) == 2 + 2 * 2                # set_state: twice; two cycles of two stages
        for f in fills:
            assert sorted(set(f)) == [0, 1, 2] and f == sorted(f)


def _worker(rank, world, port, dims, periodic, path, tags=True):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    field = whole_field((13, 10, 9))
    shape = field.shape[:0:-1]
    (x0, nx), (y0, ny), (z0, nz) = decomp.sub_box(rank, dims, shape)
    sl = (slice(None), slice(z0, z0 + nz), slice(y0, y0 + ny), slice(x0, x0 + nx))
    box = HostBox(field[sl])
    dec = decomp.Decomposition(decomp.DistLink(box, dims, periodic, tags=tags))
    dec.finish_set_state()
    dec.advance(2, 0.3)
    np.save(path % rank, box.active())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("dims,periodic,port", [((2, 1, 1), True, 29541), ((1, 1, 2), True, 29542), ((1, 2, 1), False, 29543)])
def test_dist_link_over_gloo_world_size_2(tmp_path, dims, periodic, port):
    path = str(tmp_path / "rank%d.npy")
    mp.spawn(_worker, args=(2, port, dims, periodic, path), nprocs=2, join=True)
    field = whole_field((13, 10, 9))
    one, _ = run_local(field, (1, 1, 1), periodic)
    for rank in range(2):
        (x0, nx), (y0, ny), (z0, nz) = decomp.sub_box(rank, dims, field.shape[:0:-1])
        assert np.array_equal(np.load(path % rank), one[:, z0:z0 + nz, y0:y0 + ny, x0:x0 + nx])


def test_dist_link_pairs_messages_by_order_alone(tmp_path):
    """NCCL has no tags: between two ranks the k-th send meets the k-th receive.  With two ranks along a periodic direction
    both neighbours of a rank are the same peer, so only the right posting order delivers each slab to the right side.
    All tags equal makes gloo match by order too."""
    dims, periodic = (2, 1, 1), True
    path = str(tmp_path / "rank%d.npy")
    mp.spawn(_worker, args=(2, 29547, dims, periodic, path, False), nprocs=2, join=True)
    field = whole_field((13, 10, 9))
    one, _ = run_local(field, (1, 1, 1), periodic)
    for rank in range(2):
        (x0, nx), (y0, ny), (z0, nz) = decomp.sub_box(rank, dims, field.shape[:0:-1])
        assert np.array_equal(np.load(path % rank), one[:, z0:z0 + nz, y0:y0 + ny, x0:x0 + nx])
