"""Domain decomposition and outflow boundaries with a magnetic field (reading G23) on ONE GPU.

The sub-boxes of a decomposed run are separate contexts on the same device; their halo slabs travel as device buffers
(decomp.LocalLink) and dt is the maximum over the sub-boxes.  Nothing in the kernels depends on where a ghost cell came
from, so every cell of the decomposed run must equal the undecomposed run BIT FOR BIT -- which itself is compared with the
oracle in test_gpu_parity.py.  The host orchestration over real ranks is tested with gloo in test_decomp_host.py."""
import numpy as np
import pytest
import torch

from paper_2304_13746_b200 import decomp

pytestmark = pytest.mark.gpu
HLL, HLLC, HLLD, ROE = 0, 1, 2, 3
MINMOD, VANLEER, LIMO3 = 1, 2, 3
EMF_NONE, EMF_ARITH, EMF_UCT, EMF_UCT0 = 0, 1, 2, 3
G53 = 5.0 / 3.0
TOL, TOL_DT = 1e-10, 1e-12


@pytest.fixture(scope="module")
def idfx():
    from paper_2304_13746_b200 import idfx as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.lib()
    return m


def smooth(shape, seed, mhd):
    from test_gpu_parity import smooth_ic
    nx, ny, nz = shape
    prim, b, dx = smooth_ic(nx, ny, nz, seed, mhd)
    if b is not None:
        mean = np.array([0.4, -0.3, 0.2]).reshape(3, 1, 1, 1)
        b = mean + (b - mean) * (min(shape) / max(shape))
    return torch.from_numpy(prim).cuda(), (None if b is None else torch.from_numpy(b).cuda()), dx


def run_decomposed(idfx, shape, dims, dx, scheme, prim, b, cycles, cfl, periodic=True, nstages=2, push=True, force_open=0):
    solver, limiter, emf = scheme
    nranks = dims[0] * dims[1] * dims[2]
    boxes, slices = [], []
    for r in range(nranks):
        (x0, nx), (y0, ny), (z0, nz) = decomp.sub_box(r, dims, shape)
        sl = (slice(None), slice(z0, z0 + nz), slice(y0, y0 + ny), slice(x0, x0 + nx))
        # a decomposed outflow box: every direction is exchanged or walled; a sub-box knows which of its sides are walls
        sim = idfx.Idfx(nx, ny, nz, dx, G53, solver, limiter, emf, nstages=nstages,
                        exchange_dirs=(decomp.exchange_dirs(dims) | force_open) if periodic else 7,
                        outflow_sides=0 if periodic else decomp.wall_sides(r, dims))
        sim.set_state(prim[sl].contiguous(), None if b is None else b[sl].contiguous())
        boxes.append(sim)
        slices.append(sl)
    dec = decomp.Decomposition(decomp.LocalLink(boxes, dims, periodic, push=push))
    dec.finish_set_state()
    dec.advance(cycles, cfl)
    cons = torch.empty_like(prim)
    bf = None if b is None else torch.empty_like(b)
    for sim, sl in zip(boxes, slices):
        assert sim.status() == 0
        c, f = sim.get_conserved()
        cons[sl] = c
        if bf is not None:
            bf[sl] = f
    return cons, bf, boxes[0].last_dt()


CASES = [
    ((8, 8, 8), (2, 2, 2), (HLLD, VANLEER, EMF_UCT), 2),          # 4^3 sub-boxes: the minimum size, every tile partial
    ((9, 8, 13), (2, 1, 3), (HLLC, VANLEER, EMF_NONE), 3),
    ((40, 24, 16), (2, 1, 1), (HLLD, VANLEER, EMF_UCT), 2),
    ((40, 24, 16), (1, 2, 1), (HLLD, VANLEER, EMF_UCT), 2),
    ((40, 24, 16), (1, 1, 2), (HLLD, VANLEER, EMF_UCT), 2),
    ((37, 26, 19), (2, 2, 2), (HLLD, VANLEER, EMF_UCT), 2),
    ((37, 26, 19), (3, 2, 1), (ROE, MINMOD, EMF_ARITH), 3),
    ((40, 24, 16), (2, 2, 1), (HLL, LIMO3, EMF_UCT0), 2),
    ((37, 26, 19), (2, 2, 2), (HLLC, VANLEER, EMF_NONE), 2),
    ((40, 24, 16), (2, 1, 2), (ROE, MINMOD, EMF_NONE), 3),
]


@pytest.mark.parametrize("shape,dims,scheme,nstages", CASES)
def test_decomposed_run_equals_the_single_box_bit_for_bit(idfx, shape, dims, scheme, nstages):
    mhd = scheme[2] != EMF_NONE
    prim, b, dx = smooth(shape, 31, mhd)
    one = idfx.Idfx(shape[0], shape[1], shape[2], dx, G53, *scheme, nstages=nstages)
    one.set_state(prim, b)
    one.advance(3, 0.4)
    assert one.status() == 0
    c1, b1 = one.get_conserved()
    c2, b2, dt2 = run_decomposed(idfx, shape, dims, dx, scheme, prim, b, 3, 0.4, nstages=nstages)
    assert dt2 == one.last_dt()
    assert torch.equal(c1, c2)
    if mhd:
        assert torch.equal(b1, b2)
    assert float((c1 - prim.new_tensor(0.0)).abs().max()) > 0


def test_staged_calls_equal_advance_on_a_periodic_box(idfx):
    """idfx_cycle_begin / stage_flux / stage_update / cycle_end without exchanged directions are what idfx_advance runs."""
    shape = (33, 20, 12)
    prim, b, dx = smooth(shape, 5, True)
    sims = [idfx.Idfx(*shape, dx, G53, HLLD, VANLEER, EMF_UCT) for _ in range(2)]
    for s in sims:
        s.set_state(prim, b)
    sims[0].advance(2, 0.3)
    for _ in range(2):
        sims[1].cycle_begin(0.0, 0.3)
        for st in range(2):
            sims[1].stage_flux(st)
            sims[1].stage_update(st)
        sims[1].cycle_end()
    for x, y in zip(sims[0].get_conserved(), sims[1].get_conserved()):
        assert torch.equal(x, y)


OUTFLOW_CASES = [
    ((8, 9, 8), (2, 2, 2), (HLLD, MINMOD, EMF_UCT), 2),
    ((40, 24, 16), (2, 1, 1), (HLLD, VANLEER, EMF_UCT), 2),
    ((37, 26, 19), (2, 2, 2), (HLLD, VANLEER, EMF_UCT), 2),
    ((40, 24, 16), (1, 2, 2), (ROE, MINMOD, EMF_ARITH), 3),
    ((37, 26, 19), (2, 2, 1), (HLLC, VANLEER, EMF_NONE), 2),
]


@pytest.mark.parametrize("shape,dims,scheme,nstages", OUTFLOW_CASES)
def test_decomposed_outflow_box_equals_the_single_box(idfx, shape, dims, scheme, nstages):
    mhd = scheme[2] != EMF_NONE
    prim, b, dx = smooth(shape, 37, mhd)
    one = idfx.Idfx(shape[0], shape[1], shape[2], dx, G53, *scheme, nstages=nstages, boundary=idfx.BOUNDARY_OUTFLOW)
    one.set_state(prim, b)
    one.advance(3, 0.4)
    assert one.status() == 0
    c1, b1 = one.get_conserved()
    c2, b2, dt2 = run_decomposed(idfx, shape, dims, dx, scheme, prim, b, 3, 0.4, periodic=False, nstages=nstages)
    assert dt2 == one.last_dt()
    assert torch.equal(c1, c2)
    if mhd:
        assert torch.equal(b1, b2)


@pytest.mark.parametrize("scheme,nstages", [((HLLD, VANLEER, EMF_UCT), 2), ((ROE, MINMOD, EMF_ARITH), 3), ((HLLC, VANLEER, EMF_NONE), 2)])
def test_one_open_sub_box_equals_the_periodic_kernels(idfx, scheme, nstages):
    """One sub-box whose three directions are all declared exchanged: nothing wraps inside the kernels (the OPEN instantiation
    of k_mhd_stage, the lattice plane n, no ghost images), every ghost layer is the periodic copy of idfx_halo_fill -- and the
    result equals the periodic kernels' bit for bit."""
    shape = (37, 26, 19)
    mhd = scheme[2] != EMF_NONE
    prim, b, dx = smooth(shape, 53, mhd)
    one = idfx.Idfx(*shape, dx, G53, *scheme, nstages=nstages)
    one.set_state(prim, b)
    one.advance(3, 0.4)
    c1, b1 = one.get_conserved()
    c2, b2, dt2 = run_decomposed(idfx, shape, (1, 1, 1), dx, scheme, prim, b, 3, 0.4, nstages=nstages, force_open=7)
    assert dt2 == one.last_dt() and torch.equal(c1, c2)
    if mhd:
        assert torch.equal(b1, b2)


MHD_OUTFLOW = [((HLLD, VANLEER, EMF_UCT), 2), ((HLLD, MINMOD, EMF_ARITH), 2), ((ROE, VANLEER, EMF_UCT0), 2), ((HLL, LIMO3, EMF_UCT), 2),
               ((HLLD, LIMO3, EMF_UCT), 3), ((HLLD, VANLEER, EMF_UCT), 1)]


@pytest.mark.parametrize("scheme,nstages", MHD_OUTFLOW)
def test_mhd_outflow_against_the_oracle(idfx, R, scheme, nstages):
    """Outflow boundaries with a magnetic field (reading G23) element by element against the oracle on a ragged box whose
    flow crosses all six walls; dt, compute_dt and div B on the cells whose six faces belong to the state."""
    shape = (37, 21, 13)
    prim, b, dx = smooth(shape, 41, True)
    sim = idfx.Idfx(*shape, dx, G53, *scheme, nstages=nstages, boundary=idfx.BOUNDARY_OUTFLOW)
    sim.set_state(prim, b)
    ref = R.Oracle(*shape, dx, G53, *scheme, nstages=nstages, boundary=R.BOUNDARY_OUTFLOW)
    ref.set_state(prim.cpu().numpy(), b.cpu().numpy())
    from test_gpu_parity import assert_state_close
    for s in range(4):
        dt_g, dt_r = sim.compute_dt(0.4), ref.compute_dt(0.4)
        assert abs(dt_g - dt_r) <= TOL_DT * dt_r
        sim.advance(1, 0.4)
        ref.advance(1, 0.4)
        assert abs(sim.last_dt() - ref.last_dt()) <= TOL_DT * ref.last_dt()
        assert_state_close(sim, ref, TOL, "MHD outflow cycle %d" % s)
    assert sim.status() == 0 and ref.status() == 0
    bf = sim.get_conserved()[1]
    div = (bf[0][:-1, :-1, 1:] - bf[0][:-1, :-1, :-1]) + (bf[1][:-1, 1:, :-1] - bf[1][:-1, :-1, :-1]) + (bf[2][1:, :-1, :-1] - bf[2][:-1, :-1, :-1])
    assert float(div.abs().max() / bf.abs().max()) <= 1e-13


def test_hd_outflow_compute_dt_matches_advance(idfx, R):
    """ADVICE (round 1): idfx_compute_dt on an outflow box must be the dt idfx_advance takes (the upper boundary faces are
    solved from the ghost cells, not wrapped)."""
    shape = (37, 21, 13)
    prim, _, dx = smooth(shape, 43, False)
    prim[1] += 1.5     # a strong flow through the upper x wall
    sim = idfx.Idfx(*shape, dx, G53, HLLC, VANLEER, EMF_NONE, boundary=idfx.BOUNDARY_OUTFLOW)
    sim.set_state(prim, None)
    ref = R.Oracle(*shape, dx, G53, HLLC, VANLEER, EMF_NONE, boundary=R.BOUNDARY_OUTFLOW)
    ref.set_state(prim.cpu().numpy())
    for s in range(3):
        dt = sim.compute_dt(0.4)
        assert abs(dt - ref.compute_dt(0.4)) <= TOL_DT * dt
        sim.advance(1, 0.4)
        ref.advance(1, 0.4)
        assert sim.last_dt() == dt


@pytest.mark.parametrize("periodic", [True, False])
def test_pack_unpack_path_equals_the_push_path(idfx, periodic):
    """The slab exchange through buffers (idfx_halo_pack / unpack: what a transport between processes carries) and the
    direct push into the neighbour's ghost layers give the same bits."""
    shape, dims, scheme = (37, 26, 19), (2, 2, 2), (HLLD, VANLEER, EMF_UCT)
    prim, b, dx = smooth(shape, 47, True)
    res = [run_decomposed(idfx, shape, dims, dx, scheme, prim, b, 2, 0.4, periodic=periodic, push=p) for p in (True, False)]
    assert res[0][2] == res[1][2]
    assert torch.equal(res[0][0], res[1][0]) and torch.equal(res[0][1], res[1][1])
