"""Parity of the CUDA path against the oracle for the optional parts: Euler / RK3 (Tab. 1), the
LimO3 reconstruction, the vector-potential form of CT (Eq. 7-8), idfx_advance_to, and the paper's 3D Orszag-Tang run
(PAPER.md:346).  Same bar as tests/test_gpu_parity.py: 1e-10 relative on the conserved variables and the face field,
1e-12 on dt and on the time reached."""
import numpy as np
import pytest
import torch

from paper_2304_13746_b200 import inputs
from test_gpu_parity import (EMF_ARITH, EMF_NONE, EMF_UCT, EMF_UCT0, HLL, HLLC, HLLD, MINMOD, ROE, TOL, TOL_DT, VANLEER,
                             assert_state_close, idfx, smooth_ic)  # noqa: F401  (idfx is a fixture)

pytestmark = pytest.mark.gpu

LIMO3 = 3
PPM = 4
EMF_UCT_HLL = 4
EMF_UCT_HLLD = 5
G53 = 5.0 / 3.0


def pair(idfx, R, shape, dx, solver, limiter, emf, prim, b, nstages=2, ct_form=0):
    nx, ny, nz = shape
    sim = idfx.Idfx(nx, ny, nz, dx, G53, solver, limiter, emf, nstages=nstages, ct_form=ct_form)
    sim.set_state(torch.from_numpy(prim).cuda(), None if b is None else torch.from_numpy(b).cuda())
    ref = R.Oracle(nx, ny, nz, dx, G53, solver, limiter, emf, nstages=nstages, ct_form=ct_form)
    ref.set_state(prim, b)
    return sim, ref


OPTION_COMBOS = [
    # solver, limiter, emf, stages, CT form
    (HLLD, VANLEER, EMF_UCT, 3, 0), (HLLD, LIMO3, EMF_UCT, 3, 0), (HLLD, LIMO3, EMF_UCT, 2, 0), (ROE, LIMO3, EMF_ARITH, 3, 0),
    (HLL, LIMO3, EMF_UCT0, 1, 0), (HLLD, VANLEER, EMF_UCT, 1, 0), (HLLC, LIMO3, EMF_NONE, 3, 0), (HLL, MINMOD, EMF_NONE, 1, 0),
    (ROE, LIMO3, EMF_NONE, 2, 0),
    (HLLD, VANLEER, EMF_UCT, 2, 1), (HLLD, LIMO3, EMF_UCT, 3, 1), (ROE, VANLEER, EMF_ARITH, 1, 1), (HLL, MINMOD, EMF_UCT0, 3, 1),
    # PPM (five-cell stencils, evaluated by k_flux_face_ppm + k_rhs)
    (HLLD, PPM, EMF_UCT, 3, 0), (HLLD, PPM, EMF_UCT, 2, 0), (ROE, PPM, EMF_ARITH, 3, 0), (HLL, PPM, EMF_UCT0, 1, 1),
    (HLLC, PPM, EMF_NONE, 3, 0), (ROE, PPM, EMF_NONE, 2, 0),
    # 2D-HLL EMF
    (HLL, VANLEER, EMF_UCT_HLL, 2, 0), (HLLD, LIMO3, EMF_UCT_HLL, 3, 0), (HLL, MINMOD, EMF_UCT_HLL, 2, 1), (ROE, VANLEER, EMF_UCT_HLL, 1, 0),
    # 2D-HLLD EMF (reading G24)
    (HLLD, VANLEER, EMF_UCT_HLLD, 2, 0), (HLLD, LIMO3, EMF_UCT_HLLD, 3, 0), (HLLD, MINMOD, EMF_UCT_HLLD, 2, 1), (HLLD, VANLEER, EMF_UCT_HLLD, 1, 0),
]


@pytest.mark.parametrize("solver,limiter,emf,nstages,ct_form", OPTION_COMBOS)
def test_option_combinations_ragged_box(idfx, R, solver, limiter, emf, nstages, ct_form):
    nx, ny, nz = 37, 21, 13
    prim, b, dx = smooth_ic(nx, ny, nz, 23, emf != EMF_NONE)
    sim, ref = pair(idfx, R, (nx, ny, nz), dx, solver, limiter, emf, prim, b, nstages, ct_form)
    for s in range(4):
        sim.advance(1, 0.35)
        ref.advance(1, 0.35)
        assert abs(sim.last_dt() - ref.last_dt()) <= TOL_DT * ref.last_dt()
        assert_state_close(sim, ref, TOL, "step %d" % s)
    assert sim.status() == 0 and ref.status() == 0
    assert abs(sim.time() - ref.time()) <= TOL_DT * ref.time()
    if ct_form == 1:
        a_g, a_r = sim.get_potential().cpu().numpy(), ref.get_potential()
        assert np.abs(a_g - a_r).max() <= TOL * np.abs(a_r).max()


def test_limo3_on_steep_data(idfx, R):
    """Random-phase Mach-1 turbulence at 40^3 after a few cycles has cells on both sides of the LimO3 smoothness switch
    (eta = 1) and at its limited branches; the two implementations (theta form / division-free form) must agree."""
    prim, b, cfg = inputs.make("config3", n=40)
    sim, ref = pair(idfx, R, (40, 40, 40), cfg["dx"], HLLD, LIMO3, EMF_UCT, prim.numpy(), b.numpy(), 3, 0)
    sim.advance(6, 0.3)
    ref.advance(6, 0.3)
    assert_state_close(sim, ref, TOL, "config3 recipe, LimO3 + RK3")
    p = ref.get_state()[0]
    d = np.diff(p[0], axis=2)
    eta = (d[:, :, 1:] ** 2 + d[:, :, :-1] ** 2) / cfg["dx"] ** 2
    assert (eta > 1).any() and (eta < 1).any()      # both branches were exercised


def test_ppm_on_steep_data(idfx, R):
    """Random-phase Mach-1 turbulence at 40^3: after a few cycles the flow has smooth and non-smooth extrema, clipped
    interface values and overshooting parabolas, i.e. every branch of the PPM limiter (G22); the oracle follows the
    formulas as printed, the kernel shares the five interfaces of a stencil between its two parabolas."""
    prim, b, cfg = inputs.make("config3", n=40)
    sim, ref = pair(idfx, R, (40, 40, 40), cfg["dx"], HLLD, PPM, EMF_UCT, prim.numpy(), b.numpy(), 3, 0)
    for _ in range(3):
        sim.advance(2, 0.3)
        ref.advance(2, 0.3)
        assert abs(sim.last_dt() - ref.last_dt()) <= TOL_DT * ref.last_dt()
    assert_state_close(sim, ref, TOL, "config3 recipe, PPM + RK3")
    assert sim.status() == 0 and ref.status() == 0
    assert abs(sim.compute_dt(0.3) - ref.compute_dt(0.3)) <= TOL_DT * ref.compute_dt(0.3)   # standalone dt, PPM states
    # smallest box (the stencil wraps around the whole box) and hydrodynamics
    for shape, solver, emf in (((4, 4, 4), HLLD, EMF_UCT), ((5, 4, 7), HLLC, EMF_NONE)):
        prim, b, dx = smooth_ic(*shape, 3, emf != EMF_NONE)
        sim, ref = pair(idfx, R, shape, dx, solver, PPM, emf, prim, b, 3, 0)
        sim.advance(3, 0.3)
        ref.advance(3, 0.3)
        assert_state_close(sim, ref, TOL, "PPM %s" % (shape,))


def test_ppm_refused_where_not_implemented(idfx):
    with pytest.raises(Exception):
        idfx.Idfx(8, 8, 8, 0.125, G53, HLL, PPM, EMF_UCT_HLL)
    with pytest.raises(idfx.IdfxError) as e:
        idfx.Idfx(8, 8, 8, 0.125, G53, HLLC, PPM, EMF_NONE, boundary=idfx.BOUNDARY_OUTFLOW)
    assert e.value.code == idfx.ERR_UNSUPPORTED


@pytest.mark.parametrize("ct_form", [0, 1])
def test_advance_to_matches_the_oracle(idfx, R, ct_form):
    nx, ny, nz = 24, 20, 16
    prim, b, dx = smooth_ic(nx, ny, nz, 5)
    sim, ref = pair(idfx, R, (nx, ny, nz), dx, HLLD, VANLEER, EMF_UCT, prim, b, 2, ct_form)
    t_end = 7.3 * ref.compute_dt(0.3)
    n_g, t_g = sim.advance_to(t_end, 0.3)
    rc, n_r = ref.advance_to(t_end, 0.3)
    assert rc == 0 and n_g == n_r and t_g == t_end == ref.time() == sim.time()
    assert_state_close(sim, ref, TOL, "advance_to")
    # already there: nothing happens; max_steps stops early
    before = [x.clone() for x in sim.get_conserved()]
    assert sim.advance_to(t_end, 0.3) == (0, t_end)
    for x, y in zip(before, sim.get_conserved()):
        assert torch.equal(x, y)
    sim.set_state(torch.from_numpy(prim).cuda(), torch.from_numpy(b).cuda())
    n, t = sim.advance_to(t_end, 0.3, max_steps=3)
    assert n == 3 and 0.0 < t < t_end


@pytest.mark.parametrize("nstages", [2, 3])
def test_cycles_enqueued_past_t_end_change_nothing(idfx, nstages, monkeypatch):
    """idfx_advance_to enqueues batches; a cycle that starts at t_end must hand the state on bit for bit.
    IDFX_ADVANCE_BATCH=8 (read at bind) makes the batches overshoot: 3 real cycles, then idle ones."""
    nx, ny, nz = 20, 12, 8
    prim, b, dx = smooth_ic(nx, ny, nz, 9)
    outs = []
    for batch in (None, "8"):
        if batch:
            monkeypatch.setenv("IDFX_ADVANCE_BATCH", batch)
        sim = idfx.Idfx(nx, ny, nz, dx, G53, HLLD, VANLEER, EMF_UCT, nstages=nstages)
        sim.set_state(torch.from_numpy(prim).cuda(), torch.from_numpy(b).cuda())
        t_end = 2.5 * sim.compute_dt(0.3)
        n, t = sim.advance_to(t_end, 0.3)
        assert n == 3 and t == t_end
        outs.append([x.clone() for x in sim.get_conserved()] + [sim.get_state()[0]])
    for x, y in zip(*outs):
        assert torch.equal(x, y)


def test_vector_potential_divb_on_device(idfx):
    """After many cycles the divergence of B_ref + curl A is still one rounding of the face values."""
    n = 24
    prim, b, dx = smooth_ic(n, n, n, 3)
    res = {}
    for form in (0, 1):
        sim = idfx.Idfx(n, n, n, dx, G53, HLLD, VANLEER, EMF_UCT, ct_form=form)
        sim.set_state(torch.from_numpy(prim).cuda(), torch.from_numpy(b).cuda())
        sim.advance(300, 0.3)
        assert sim.status() == 0
        bf = sim.get_conserved()[1]
        div = (torch.roll(bf[0], -1, 2) - bf[0]) + (torch.roll(bf[1], -1, 1) - bf[1]) + (torch.roll(bf[2], -1, 0) - bf[2])
        res[form] = float(div.abs().max() / bf.abs().max())
    print("div B / |B| after 300 cycles: face form %.2e, potential form %.2e" % (res[0], res[1]))
    assert res[1] <= 8 * 2.2e-16 and res[0] < 1e-13


def test_orszag_tang_3d_run(idfx, R):
    """The paper's performance workload (3D Orszag-Tang, HLLD + PLM + E^c + RK2) at 32^3 to t = 0.1 on both
    sides: same number of cycles, same final time, fields within the bar."""
    n = 32
    prim, b = inputs.orszag_tang_3d(n)
    sim, ref = pair(idfx, R, (n, n, n), 1.0 / n, HLLD, VANLEER, EMF_UCT, prim.numpy(), b.numpy().copy())
    n_g, t_g = sim.advance_to(0.1, 0.3)
    rc, n_r = ref.advance_to(0.1, 0.3)
    assert rc == 0 and sim.status() == 0 and n_g == n_r and t_g == 0.1
    assert_state_close(sim, ref, TOL, "3D OT to t = 0.1 (%d cycles)" % n_g)
    bf = sim.get_conserved()[1]
    div = (torch.roll(bf[0], -1, 2) - bf[0]) + (torch.roll(bf[1], -1, 1) - bf[1]) + (torch.roll(bf[2], -1, 0) - bf[2])
    assert float(div.abs().max() / bf.abs().max()) < 1e-13


def test_pressure_floor_matches_the_oracle(idfx, R):
    """3D Orszag-Tang at 32^3 with a floor placed inside the range the flow reaches (p_min ~ 0.016 by t = 0.25), so
    that it acts on many cells: same cells floored, same fields."""
    n, floor = 32, 0.03
    prim, b = inputs.orszag_tang_3d(n)
    nx = ny = nz = n
    sim = idfx.Idfx(nx, ny, nz, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT, pressure_floor=floor)
    sim.set_state(prim.contiguous().cuda(), b.contiguous().cuda())
    ref = R.Oracle(nx, ny, nz, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT, pressure_floor=floor)
    ref.set_state(prim.numpy(), b.numpy().copy())
    n_g, _ = sim.advance_to(0.25, 0.3)
    rc, n_r = ref.advance_to(0.25, 0.3)
    assert rc == 0 and sim.status() == 0 and n_g == n_r
    assert_state_close(sim, ref, TOL, "floored run")
    assert ref.floor_count() > 100 and abs(sim.floor_count() - ref.floor_count()) <= 2
    assert float(sim.get_state()[0][4].min()) == floor
    # off by default: the same run without the floor is flagged or stays above it
    sim0 = idfx.Idfx(nx, ny, nz, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT)
    sim0.set_state(prim.contiguous().cuda(), b.contiguous().cuda())
    sim0.advance_to(0.25, 0.3)
    assert sim0.floor_count() == 0 and float(sim0.get_state()[0][4].min()) < floor


def test_floor_count_does_not_depend_on_the_batch_size(idfx, monkeypatch):
    """Cycles enqueued past t_end (IDFX_ADVANCE_BATCH=16 forces them) meet the already floored cells again: they must not
    be floored or counted a second time, so the count is the same as with batches that do not overshoot."""
    n, floor = 32, 0.03
    prim, b = inputs.orszag_tang_3d(n)
    counts, states = [], []
    for batch in (None, "16"):
        if batch:
            monkeypatch.setenv("IDFX_ADVANCE_BATCH", batch)
        sim = idfx.Idfx(n, n, n, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT, pressure_floor=floor)
        sim.set_state(prim.contiguous().cuda(), b.contiguous().cuda())
        sim.advance_to(0.25, 0.3)
        counts.append(sim.floor_count())
        states.append(sim.get_conserved()[0].clone())
    assert counts[0] == counts[1] > 100, counts
    assert torch.equal(states[0], states[1])


def test_sedov_blast_parity_and_radius(idfx, R):
    """The paper's Cartesian Sedov test (HLL + PLM + RK2, periodic): parity with the oracle at 32^3, and at
    128^3 the shock radius against the self-similar solution r = 1.152 (E t^2 / rho)^(1/5)."""
    n = 32
    prim, _ = inputs.sedov(n)
    sim = idfx.Idfx(n, n, n, 1.0 / n, G53, HLL, VANLEER, EMF_NONE)
    sim.set_state(prim.cuda())
    ref = R.Oracle(n, n, n, 1.0 / n, G53, HLL, VANLEER, EMF_NONE)
    ref.set_state(prim.numpy())
    n_g, t_g = sim.advance_to(0.01, 0.3)
    rc, n_r = ref.advance_to(0.01, 0.3)
    assert rc == 0 and n_g == n_r and t_g == 0.01
    assert_state_close(sim, ref, TOL, "Sedov 32^3")
    n = 128
    prim, _ = inputs.sedov(n, device="cuda")
    sim = idfx.Idfx(n, n, n, 1.0 / n, G53, HLL, VANLEER, EMF_NONE)
    sim.set_state(prim)
    sim.advance_to(0.05, 0.3)
    assert sim.status() == 0
    rho = sim.get_state()[0][0]
    r_exact = 1.152 * (0.05 ** 2) ** 0.2
    c = n // 2
    for line in (rho[c, c, c:], rho[c, c:, c], rho[c:, c, c]):
        r_num = (int(torch.argmax(line)) + 0.5) / n
        assert abs(r_num - r_exact) <= 2.0 / n, (r_num, r_exact)
    assert float(rho.max()) > 2.5


def test_outflow_boundaries_hd(idfx, R):
    """Zero-gradient ghosts (HD): the paper's Sod tube with outflow ends along each axis, and a 3D blast reaching
    the walls, against the oracle."""
    for axis in range(3):
        shape = [6, 5, 4]
        shape[2 - axis] = 64
        nz, ny, nx = shape
        bc = [1, 1, 1]
        bc[2 - axis] = 64
        left = ((np.arange(64) + 0.5) / 64 < 0.5).reshape(bc)
        prim = np.zeros([5] + shape)
        prim[0] = np.where(left, 1.0, 0.125)
        prim[4] = np.where(left, 1.0, 0.1)
        sim = idfx.Idfx(nx, ny, nz, 1.0 / 64, 1.4, ROE, VANLEER, EMF_NONE, boundary=idfx.BOUNDARY_OUTFLOW)
        sim.set_state(torch.from_numpy(prim).cuda())
        ref = R.Oracle(nx, ny, nz, 1.0 / 64, 1.4, ROE, VANLEER, EMF_NONE, boundary=R.BOUNDARY_OUTFLOW)
        ref.set_state(prim)
        n_g, _ = sim.advance_to(0.2, 0.4)
        rc, n_r = ref.advance_to(0.2, 0.4)
        assert rc == 0 and n_g == n_r
        assert_state_close(sim, ref, TOL, "Sod, outflow, axis %d" % axis)
    n = 24
    prim, _ = inputs.sedov(n)
    sim = idfx.Idfx(n, n, n, 1.0 / n, G53, HLL, VANLEER, EMF_NONE, boundary=idfx.BOUNDARY_OUTFLOW, nstages=3)
    sim.set_state(prim.cuda())
    ref = R.Oracle(n, n, n, 1.0 / n, G53, HLL, VANLEER, EMF_NONE, boundary=R.BOUNDARY_OUTFLOW, nstages=3)
    ref.set_state(prim.numpy())
    sim.advance_to(0.2, 0.3)       # the shock (r = 0.61 at t = 0.2) has left through the walls
    ref.advance_to(0.2, 0.3)
    assert_state_close(sim, ref, TOL, "blast through outflow walls")
    assert float(sim.get_conserved()[0][4].sum()) / n ** 3 < 0.9     # energy left the box
    # with a magnetic field (tests/test_gpu_decomp.py): face-flux EMFs and the face form of CT only
    with pytest.raises(idfx.IdfxError):
        idfx.Idfx(8, 8, 8, 0.125, G53, HLLD, VANLEER, EMF_UCT_HLL, boundary=idfx.BOUNDARY_OUTFLOW)
    with pytest.raises(idfx.IdfxError):
        idfx.Idfx(8, 8, 8, 0.125, G53, HLLD, VANLEER, EMF_UCT, ct_form=1, boundary=idfx.BOUNDARY_OUTFLOW)


def test_all_options_together_medium_box(idfx, R):
    """RK3 + LimO3 + 2D-HLL EMF + vector potential + a floor on a box that spans many tiles in every direction and has
    ragged tails (96 x 80 x 72): two cycles against the oracle."""
    nx, ny, nz = 96, 80, 72
    prim, b, dx = smooth_ic(nx, ny, nz, 31)
    sim, ref = None, None
    sim = idfx.Idfx(nx, ny, nz, dx, G53, HLLD, LIMO3, EMF_UCT_HLL, nstages=3, ct_form=1, pressure_floor=1e-8)
    sim.set_state(torch.from_numpy(prim).cuda(), torch.from_numpy(b).cuda())
    ref = R.Oracle(nx, ny, nz, dx, G53, HLLD, LIMO3, EMF_UCT_HLL, nstages=3, ct_form=1, pressure_floor=1e-8)
    ref.set_state(prim, b)
    sim.advance(2, 0.3)
    ref.advance(2, 0.3)
    assert abs(sim.last_dt() - ref.last_dt()) <= TOL_DT * ref.last_dt()
    assert_state_close(sim, ref, TOL, "all options, 96 x 80 x 72")
    assert sim.floor_count() == 0 == ref.floor_count()


def test_hd_fused_kernel_ragged_and_chunked(idfx, R):
    """The one-kernel HD stage on a box whose sizes are not multiples of its 31 x 7 tiles and whose z extent splits into
    several chunks, RK3 + LimO3 + HLLC, against the oracle and against the three-sweep path."""
    nx, ny, nz = 70, 45, 150
    prim, _, dx = smooth_ic(nx, ny, nz, 17, mhd=False)
    sim = idfx.Idfx(nx, ny, nz, dx, G53, HLLC, LIMO3, EMF_NONE, nstages=3)
    sim.set_state(torch.from_numpy(prim).cuda())
    ref = R.Oracle(nx, ny, nz, dx, G53, HLLC, LIMO3, EMF_NONE, nstages=3)
    ref.set_state(prim)
    sim.advance(2, 0.4)
    ref.advance(2, 0.4)
    assert abs(sim.last_dt() - ref.last_dt()) <= TOL_DT * ref.last_dt()
    assert_state_close(sim, ref, TOL, "fused HD stage, 70 x 45 x 150")


def test_emf_hlld2d_on_turbulence_all_fan_regions(idfx, R):
    """Mach-1 turbulence at 40^3 after a few cycles puts faces into every region of the HLLD fan (supersonic, starred and
    double-starred on both sides): the 2D-HLLD EMF of the CUDA path (unified response form) against the oracle's region by
    region coefficients."""
    prim, b, cfg = inputs.make("config3", n=40)
    sim, ref = pair(idfx, R, (40, 40, 40), cfg["dx"], HLLD, VANLEER, EMF_UCT_HLLD, prim.numpy(), b.numpy(), 2, 0)
    sim.advance(6, 0.3)
    ref.advance(6, 0.3)
    assert sim.status() == 0 and ref.status() == 0
    assert abs(sim.last_dt() - ref.last_dt()) <= TOL_DT * ref.last_dt()
    assert_state_close(sim, ref, TOL, "2D-HLLD EMF, 40^3 turbulence")
    bf = sim.get_conserved()[1]
    div = (torch.roll(bf[0], -1, 2) - bf[0]) + (torch.roll(bf[1], -1, 1) - bf[1]) + (torch.roll(bf[2], -1, 0) - bf[2])
    assert float(div.abs().max() / bf.abs().max()) <= 1e-13


@pytest.mark.parametrize("solver,limiter", [(HLLC, VANLEER), (ROE, MINMOD), (HLL, LIMO3)])
def test_hd_cycles_fed_with_the_conserved_fields(idfx, R, solver, limiter):
    """Hydrodynamic RK2 cycles on a periodic box read the conserved fields and never write the primitive buffers
    (csrc/hd_stage_u.cuh), except the first cycle after set_state, which reconstructs from the caller's primitives as given.
    Every way in and out of that mode against the oracle: graph replay and single steps, compute_dt and get_state in
    between, a switch to RK3 and back, fixed steps, and a second set_state.  The box
    spans several 31 x 7 tiles, partial ones and three z chunks."""
    nx, ny, nz = 70, 45, 50
    prim, _, dx = smooth_ic(nx, ny, nz, 29, mhd=False)
    sim = idfx.Idfx(nx, ny, nz, dx, G53, solver, limiter, EMF_NONE)
    ref = R.Oracle(nx, ny, nz, dx, G53, solver, limiter, EMF_NONE)
    sim.set_state(torch.from_numpy(prim).cuda())
    ref.set_state(prim)

    def both(what, *args):
        getattr(sim, what)(*args)
        getattr(ref, what)(*args)

    def check(tag):
        assert abs(sim.last_dt() - ref.last_dt()) <= TOL_DT * ref.last_dt(), tag
        assert_state_close(sim, ref, TOL, tag)
        dg, dr = sim.compute_dt(0.4), ref.compute_dt(0.4)
        assert abs(dg - dr) <= TOL_DT * dr, tag + ": compute_dt"

    both("advance", 4, 0.4)                      # one cycle from the given primitives, three from the conserved fields
    check("4 cycles")
    both("advance", 1, 0.4)                      # compute_dt and get_state in between must not have disturbed anything
    check("5 cycles")
    dt = 0.5 * ref.last_dt()
    both("step", dt)                             # outside the graphs
    both("step", dt)
    check("fixed steps")
    sim.set_integrator(3)                        # RK3 needs the primitive buffers again ...
    assert ref.L.idfxref_set_option(ref.h, 0, 3) == 0
    both("advance", 2, 0.4)
    check("RK3")
    sim.set_integrator(2)                        # ... and RK2 drops them again, with the conserved buffers swapped or not
    assert ref.L.idfxref_set_option(ref.h, 0, 2) == 0
    both("advance", 3, 0.4)
    check("RK2 again")
    for _ in range(2):                           # the same cycles through the staged calls (include/idfx.h)
        sim.cycle_begin(0.0, 0.4)
        for stage in range(2):
            sim.stage_flux(stage)
            sim.stage_update(stage)
        sim.cycle_end()
    ref.advance(2, 0.4)
    check("staged calls")
    # a halo slab is cut from the primitive buffer, which those cycles left behind: the call brings it up to date first
    buf = sim.new_buffer(sim.halo_count(0))
    sim.halo_pack(0, 0, buf)
    slab = buf.view(5, nz, ny, 2)
    assert torch.equal(slab, sim.get_state()[0][:, :, :, 0:2]), "lower x slab of the primitives"
    both("advance", 1, 0.4)
    check("after a halo call")
    sim.set_state(torch.from_numpy(prim).cuda())
    ref.set_state(prim)
    both("advance", 3, 0.4)
    check("after a second set_state")
    assert sim.status() == 0 and ref.status() == 0
    cons_g = sim.get_conserved()[0].cpu().numpy()
    cons_r = ref.get_conserved()[0]
    assert np.abs(cons_g - cons_r).max() <= TOL * np.abs(cons_r).max()
