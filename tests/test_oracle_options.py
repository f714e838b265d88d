"""Pins for the oracle's optional parts: the Euler / RK2 / RK3 weights of Tab. 1,
the LimO3 reconstruction, the vector-potential form of CT (Eq. 7-8) and the
run-to-a-time driver.  Expected values are closed forms (stability polynomials, point values of a parabola),
convergence orders, or the equivalence the paper states ("mathematically equivalent to the original CT")."""
import math

import numpy as np
import pytest

from test_oracle_scheme import (EMF_ARITH, EMF_NONE, EMF_UCT, FLAT, G53, HLL, HLLD, VANLEER, curl_np, divb,
                                linear_wave_mode, smooth_mhd_ic)

LIMO3 = 3


# =================================================================================================
# Tab. 1: the stability polynomial of each integrator on a linear problem
# =================================================================================================
@pytest.mark.parametrize("nstages", [1, 2, 3])
def test_rk_amplification_polynomials(R, nstages):
    """Supersonic uniform flow + flat reconstruction + HLL = first-order upwind advection of rho (linear).  One
    cycle multiplies Fourier mode m by sum_{q<=s} z^q/q!, z = -(u dt/dx)(1 - exp(-i k dx)): Euler 1 + z, RK2
    + z^2/2, RK3 + z^3/6 (Gottlieb & Shu 1998, the schemes Tab. 1 encodes)."""
    n = 16
    dx = 1.0 / n
    x = (np.arange(n) + 0.5) * dx
    prim = np.zeros((5, 1, 1, n))
    prim[0, 0, 0] = 1.0 + 0.1 * np.cos(2 * np.pi * x) + 0.05 * np.sin(4 * np.pi * x)
    prim[1] = 3.0
    prim[4] = 0.1
    o = R.Oracle(n, 1, 1, dx, 1.4, HLL, FLAT, EMF_NONE, nstages=nstages)
    o.set_state(prim)
    dt = 0.37 * dx / 3.0
    o.step(dt)
    f0, f1 = np.fft.fft(prim[0].ravel()), np.fft.fft(o.get_state()[0][0].ravel())
    for m in (1, 2):
        z = -(3.0 * dt / dx) * (1 - np.exp(-2j * np.pi * m / n))
        poly = sum(z ** q / math.factorial(q) for q in range(nstages + 1))
        assert f1[m] / f0[m] == pytest.approx(poly, abs=1e-13)
    assert o.time() == dt


def nonlinear_1d_ic(n, amp=0.05):
    dx = 1.0 / n
    c = np.cos(2 * np.pi * (np.arange(n) + 0.5) * dx)
    s = np.sin(2 * np.pi * (np.arange(n) + 0.5) * dx)
    prim = np.empty((5, 1, 1, n))
    prim[0, 0, 0] = 1 + amp * c
    prim[1, 0, 0] = amp * s
    prim[2, 0, 0] = 0.5 * amp * c
    prim[3, 0, 0] = -0.3 * amp * s
    prim[4, 0, 0] = 0.6 + amp * 0.4 * c
    bf = np.empty((3, 1, 1, n))
    bf[0], bf[1, 0, 0], bf[2, 0, 0] = 1.0, 1.5 + amp * s, amp * 0.5 * c
    return prim, bf


@pytest.mark.parametrize("nstages", [1, 2, 3])
def test_temporal_order_of_the_integrators(R, nstages):
    """Fixed grid, smooth nonlinear MHD flow, time step halved: the difference to a finely stepped run falls as
    dt^s for the s-stage scheme, for the cell variables and for the face field alike."""
    n, T = 32, 0.02
    prim, bf = nonlinear_1d_ic(n)

    def run(nsteps):
        o = R.Oracle(n, 1, 1, 1.0 / n, G53, HLL, LIMO3, EMF_UCT, nstages=nstages)
        o.set_state(prim, bf)
        for _ in range(nsteps):
            assert o.step(T / nsteps) == 0
        u, b = o.get_conserved()
        return np.concatenate([u.ravel(), b.ravel()])

    ref = run(1024 if nstages == 1 else 256)
    e = [np.abs(run(k) - ref).max() for k in (4, 8, 16)]
    for a, b in zip(e[:-1], e[1:]):
        assert math.log2(a / b) == pytest.approx(nstages, abs=0.25), (nstages, e)


# =================================================================================================
# LimO3
# =================================================================================================
def test_limo3_reproduces_a_parabola_where_the_data_are_smooth(R):
    """Cell averages of q(x) = a + b x + c x^2 on a uniform grid: the unlimited weight (2 + theta)/3 returns the point
    values of q at both faces exactly (third order); dx = 0.1 and small coefficients keep eta < 1."""
    a, b, c, dx = 0.7, 0.31, -0.23, 0.1
    avg = lambda xc: a + b * xc + c * (xc * xc + dx * dx / 12.0)
    q = lambda x: a + b * x + c * x * x
    for xc in (-0.35, 0.0, 0.2, 1.05):
        lo, hi = R.reconstruct(LIMO3, avg(xc - dx), avg(xc), avg(xc + dx), dx)
        assert lo == pytest.approx(q(xc - dx / 2), abs=2e-16 * 8)
        assert hi == pytest.approx(q(xc + dx / 2), abs=2e-16 * 8)


def test_limo3_limited_branch_values(R):
    """Steep data (eta > 1): phi = max(0, min((2+theta)/3, max(-theta/2, min(2 theta, (2+theta)/3, 1.6)))).  Linear data keep
    phi = 1; a monotone kink is capped by 2 theta on one side and by 1.6 on the other; extrema with theta in (-2, 0)
    keep a reduced, non-zero increment (the scheme does not clip extrema) and theta <= -2 gives zero."""
    dx = 1e-3
    # (qm, q0, qp) -> expected phi(theta) for the upper face and phi(1/theta) for the lower one
    cases = [((0.0, 1.0, 2.0), 1.0, 1.0),            # theta = 1
             ((0.0, 10.0, 11.0), 1.6, 0.2),          # theta = 10: cap 1.6;   1/theta = 0.1: 2 theta
             ((0.0, 1.0, 5.0), 0.5, 1.6),            # theta = 1/4: 2 theta;  1/theta = 4: min(phat = 2, 1.6)
             ((0.0, 1.0, 0.0), 1.0 / 3.0, 1.0 / 3.0),  # theta = -1: min(1/3, 1/2)
             ((0.0, 3.0, 2.0), 0.0, 0.5 / 3.0),      # theta = -3 -> 0;  1/theta = -1/3: min(5/9, 1/6)
             ((0.0, 1.0, 1.0), 0.0, 0.0)]            # d+ = 0
    for (qm, q0, qp), phi_up, phi_lo in cases:
        lo, hi = R.reconstruct(LIMO3, qm, q0, qp, dx)
        assert hi == pytest.approx(q0 + 0.5 * phi_up * (qp - q0), abs=1e-15)
        assert lo == pytest.approx(q0 - 0.5 * phi_lo * (q0 - qm), abs=1e-15)


def test_limo3_symmetries_and_bounds(R):
    rng = np.random.default_rng(5)
    for _ in range(2000):
        qm, q0, qp = rng.normal(size=3) * 10.0 ** rng.integers(-3, 2)
        dx = 10.0 ** rng.integers(-4, 1)
        lo, hi = R.reconstruct(LIMO3, qm, q0, qp, dx)
        lo_r, hi_r = R.reconstruct(LIMO3, qp, q0, qm, dx)      # mirror image
        assert (lo, hi) == (hi_r, lo_r)
        lo_n, hi_n = R.reconstruct(LIMO3, -qm, -q0, -qp, dx)   # odd in the data
        assert (lo_n, hi_n) == (-lo, -hi)                   # exactly: every operation is odd
        lo_s, hi_s = R.reconstruct(LIMO3, qm + 1.0, q0 + 1.0, qp + 1.0, dx)
        assert lo_s == pytest.approx(lo + 1.0, abs=1e-12 * max(1.0, abs(q0))) and hi_s == pytest.approx(hi + 1.0, abs=1e-12 * max(1.0, abs(q0)))
        if (qm - q0) ** 2 + (qp - q0) ** 2 > 1.01 * dx * dx:   # limited: 0 <= phi <= 1.6, and monotone data stay bounded
            slack = 4e-16 * max(abs(q0), abs(qp)) * abs(qp - q0)   # hi is rounded at the size of q0
            assert -slack <= (hi - q0) * (qp - q0) <= 0.8 * (qp - q0) ** 2 + slack
            if (q0 - qm) * (qp - q0) > 0:
                assert min(q0, qp) <= hi <= max(q0, qp) and min(qm, q0) <= lo <= max(qm, q0)


def run_wave_1d(R, n, limiter, nstages, kind="fast", cfl=0.4, eps=1e-6):
    speed, r = linear_wave_mode(kind)
    dx = 1.0 / n
    c = np.cos(2 * np.pi * (np.arange(n) + 0.5) * dx).reshape(1, 1, n)
    prim = np.empty((5, 1, 1, n))
    prim[0] = 1 + eps * r[0] * c
    prim[1], prim[2], prim[3] = eps * r[1] * c, eps * r[2] * c, eps * r[3] * c
    prim[4] = 0.6 + eps * r[4] * c
    bf = np.empty((3, 1, 1, n))
    bf[0], bf[1], bf[2] = 1.0, 1.5 + eps * r[5] * c, eps * r[6] * c
    o = R.Oracle(n, 1, 1, dx, G53, HLLD, limiter, EMF_UCT, nstages=nstages)
    o.set_state(prim, bf)
    period = 1.0 / speed
    nsteps = int(math.ceil(period / o.compute_dt(cfl)))
    for _ in range(nsteps):
        assert o.step(period / nsteps) == 0
    p1, b1 = o.get_state()
    tot = [np.abs(p1[v] - prim[v]).mean() for v in range(5)] + [np.abs(b1[d] - bf[d]).mean() for d in range(3)]
    return math.sqrt(sum(t * t for t in tot)) / eps


@pytest.mark.parametrize("kind", ["fast", "alfven"])
def test_rk3_limo3_linear_wave_is_third_order(R, kind):
    """The paper's most accurate combination short of PPM (Fig. 7): third-order convergence, and an
    error well below the second-order scheme's at the same resolution."""
    errs = [run_wave_1d(R, n, LIMO3, 3, kind) for n in (32, 64)]
    assert math.log2(errs[0] / errs[1]) >= 2.8, errs
    assert errs[1] < 0.2 * run_wave_1d(R, 64, VANLEER, 2, kind)


# =================================================================================================
# Eq. 7-8: vector-potential form of CT
# =================================================================================================
@pytest.mark.parametrize("nstages,emf", [(2, EMF_UCT), (3, EMF_ARITH), (1, EMF_UCT)])
def test_vector_potential_form_equals_face_form(R, nstages, emf):
    """"mathematically equivalent to the original CT algorithm": same run in both forms, differences at
    rounding level only; and the potential is what Eq. 7 says, checked on one Euler step against the stored EMFs."""
    n = 12
    prim, b = smooth_mhd_ic(n, seed=11)
    outs = []
    for form in (R.CT_FACE, R.CT_POTENTIAL):
        o = R.Oracle(n, n, n, 1.0 / n, G53, HLLD, VANLEER, emf, nstages=nstages, ct_form=form)
        o.set_state(prim, b)
        assert o.advance(6, 0.3) == 0
        outs.append(o.get_conserved())
    for x, y in zip(outs[0], outs[1]):
        assert np.abs(x - y).max() <= 2e-14 * np.abs(x).max()
    o = R.Oracle(n, n, n, 1.0 / n, G53, HLLD, VANLEER, emf, nstages=1, ct_form=R.CT_POTENTIAL)
    o.set_state(prim, b)
    dt = 0.5 * o.compute_dt(0.3)
    o.step(dt)
    np.testing.assert_array_equal(o.get_potential(), -dt * o.get_emf())
    a = o.get_potential()
    bnew = o.get_conserved()[1]
    np.testing.assert_allclose(bnew, b + curl_np(a[0], a[1], a[2], 1.0 / n), rtol=0, atol=1e-15)


def test_vector_potential_divb_does_not_accumulate(R):
    """"prevents roundoff errors from accumulating in div B": after many cycles the divergence of the
    potential form is still one rounding of the face values, while the face form has drifted above it."""
    n = 8
    prim, b = smooth_mhd_ic(n, seed=3)
    res = {}
    for form in (R.CT_FACE, R.CT_POTENTIAL):
        o = R.Oracle(n, n, n, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT, ct_form=form)
        o.set_state(prim, b)
        assert o.advance(150, 0.3) == 0
        bf = o.get_conserved()[1]
        res[form] = np.abs(divb(bf)).max() / np.abs(bf).max()
    assert res[R.CT_POTENTIAL] <= 8 * 2.2e-16      # sum of six face values, each rounded once
    assert res[R.CT_FACE] > res[R.CT_POTENTIAL]


# =================================================================================================
# run to a given time (the paper's runs are "to t = ...")
# =================================================================================================
def test_advance_to_lands_on_t_end(R):
    n = 8
    prim, b = smooth_mhd_ic(n, seed=7)
    o = R.Oracle(n, n, n, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT)
    o.set_state(prim, b)
    t_end = 3.6 * o.compute_dt(0.3)
    rc, nsteps = o.advance_to(t_end, 0.3)
    assert rc == 0 and o.time() == t_end and 4 <= nsteps <= 5
    # the same by hand: CFL steps, the last one shortened
    o2 = R.Oracle(n, n, n, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT)
    o2.set_state(prim, b)
    t = 0.0
    for _ in range(nsteps):
        dt = min(o2.compute_dt(0.3), t_end - t)
        o2.step(dt)
        t += dt
    for x, y in zip(o.get_conserved(), o2.get_conserved()):
        np.testing.assert_array_equal(x, y)
    # max_steps stops early
    o.set_state(prim, b)
    rc, k = o.advance_to(t_end, 0.3, max_steps=2)
    assert k == 2 and 0.0 < o.time() < t_end


# =================================================================================================
# optional pressure floor (reading G20; off by default, G13)
# =================================================================================================
def test_pressure_floor_closed_form_and_inert_when_not_needed(R):
    """A uniform moving magnetised state below the floor: the first stage raises every cell to the floor and rewrites
    E = p_floor/(gamma-1) + rho v^2/2 + B^2/2; nothing else changes (uniform states have no flux divergence) and the
    cells are not counted twice.  With pressures above the floor the option changes no bit."""
    n, floor = 6, 1e-4
    prim = np.zeros((5, n, n, n))
    prim[0], prim[1], prim[2], prim[4] = 1.3, 0.3, -0.2, 1e-7
    b = np.zeros((3, n, n, n))
    b[0], b[1], b[2] = 0.5, -0.25, 0.1
    o = R.Oracle(n, n, n, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT, pressure_floor=floor)
    o.set_state(prim, b)
    assert o.get_state()[0][4].min() == floor and o.floor_count() == n ** 3
    o.set_state(prim, b)
    assert o.step(1e-3) == 0
    u, bf = o.get_conserved()
    e_want = floor / (G53 - 1) + 0.5 * 1.3 * (0.09 + 0.04) + 0.5 * (0.25 + 0.0625 + 0.01)
    assert np.abs(u[4] - e_want).max() <= 4e-16 and o.floor_count() == n ** 3
    np.testing.assert_array_equal(bf, b)
    np.testing.assert_allclose(o.get_state()[0][4], floor, rtol=1e-9)
    prim2, b2 = smooth_mhd_ic(8, seed=2)
    outs = []
    for fl in (0.0, 1e-6):
        o = R.Oracle(8, 8, 8, 0.125, G53, HLLD, VANLEER, EMF_UCT, pressure_floor=fl)
        o.set_state(prim2, b2)
        assert o.advance(3, 0.3) == 0 and o.floor_count() == 0
        outs.append(o.get_conserved())
    for x, y in zip(*outs):
        np.testing.assert_array_equal(x, y)


# =================================================================================================
# Sedov-Taylor blast, HD path
# =================================================================================================
def test_sedov_blast_radius_and_symmetry(R):
    """E = 1 in rho = 1: the shock sits at r = xi0 (E t^2 / rho)^(1/5) with xi0 = 1.152 for gamma = 5/3 (Sedov 1946,
    Taylor 1950; textbook value).  40^3 cells, HLL + van Leer + RK2 as in the paper, to t = 0.02 (r = 0.241 = 9.6 cells):
    the density maximum along the axes lies within 1.5 cells of it, the eight octants are mirror images to round-off,
    and total energy is conserved (the deposited E plus the ambient p/(gamma-1))."""
    from paper_2304_13746_b200 import inputs
    n = 40
    prim, n_in = inputs.sedov(n)
    prim = prim.numpy()
    o = R.Oracle(n, n, n, 1.0 / n, G53, HLL, VANLEER, EMF_NONE)
    o.set_state(prim)
    e0 = o.get_conserved()[0][4].sum() / n ** 3
    assert e0 == pytest.approx(1.0 + 1e-2 / (G53 - 1) * (1 - n_in / n ** 3), rel=1e-13)
    rc, steps = o.advance_to(0.02, 0.3)
    assert rc == 0 and steps > 50
    u = o.get_conserved()[0]
    assert u[4].sum() / n ** 3 == pytest.approx(e0, rel=1e-12)
    rho = u[0]
    for ax in range(3):      # mirror symmetry about the centre, every axis
        np.testing.assert_allclose(rho, np.flip(rho, ax), rtol=1e-11)
    r_exact = 1.152 * (1.0 * 0.02 ** 2 / 1.0) ** 0.2
    c = n // 2
    for line in (rho[c, c, c:], rho[c, c:, c], rho[c:, c, c]):
        r_num = (np.argmax(line) + 0.5) / n
        assert abs(r_num - r_exact) <= 1.5 / n, (r_num, r_exact)
    assert rho.max() > 1.8      # a strong shock, smeared over ~3 cells by HLL at this resolution (limit (gamma+1)/(gamma-1) = 4)


# =================================================================================================
# 2D-HLL EMF ("2D HLL ... following the method of Mignone & Del Zanna (2021)"; reading G21)
# =================================================================================================
EMF_UCT_HLL = 4


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("limiter", [VANLEER, LIMO3])
def test_emf_hll2d_plane_parallel_identity(R, axis, limiter):
    """Plane-parallel flow along a grid axis with uniform transverse velocity: the edge EMF of the 2D-HLL scheme must be
    the EMF of the 1D HLL flux, E_t2 = -F_n[B_t1] and E_t1 = +F_n[B_t2] (the consistency requirement that fixes its
    weights alpha+-/(alpha+ + alpha-), its dissipation alpha+ alpha-/(alpha+ + alpha-) and the HLL-weighted face velocity)."""
    from test_oracle_scheme import HLL as HLL_
    n = 32
    dx = 1.0 / n
    x = (np.arange(n) + 0.5) * dx
    shape = [4, 4, 4]
    shape[2 - axis] = n
    bc = [1, 1, 1]
    bc[2 - axis] = n
    X = x.reshape(bc)
    a, b_, e = axis, (axis + 1) % 3, (axis + 2) % 3
    prim = np.empty([5] + shape)
    prim[0] = 1.0 + 0.3 * np.sin(2 * np.pi * X)
    prim[1 + a] = 0.4 * np.cos(2 * np.pi * X)
    prim[1 + b_] = 0.35
    prim[1 + e] = -0.25
    prim[4] = 1.0 + 0.2 * np.cos(4 * np.pi * X)
    bf = np.empty([3] + shape)
    bf[a] = 0.7
    bf[b_] = 0.5 + 0.3 * np.sin(2 * np.pi * X)
    bf[e] = -0.4 + 0.2 * np.cos(2 * np.pi * X)
    dims = shape[::-1]
    o = R.Oracle(dims[0], dims[1], dims[2], dx, G53, HLL_, limiter, EMF_UCT_HLL)
    o.set_state(prim, bf)
    o.step(o.compute_dt(0.4))
    E = o.get_emf()
    F, _ = o.get_flux(axis)
    np.testing.assert_allclose(E[e], -F[5], rtol=0, atol=1e-13)   # E_t2 = -F_n[B_t1]
    np.testing.assert_allclose(E[b_], F[6], rtol=0, atol=1e-13)   # E_t1 = +F_n[B_t2]
    assert np.abs(E[a]).max() > 0.01                               # the third component is the transverse -(v x B), not zero


def test_emf_hll2d_uniform_state_conservation_divb_and_symmetry(R):
    from test_oracle_scheme import HLL as HLL_, rot_prim, rot_vector
    n = 8
    prim = np.empty((5, n, n, n))
    for v, val in enumerate((1.3, 0.4, -0.7, 0.2, 0.8)):
        prim[v] = val
    b = np.empty((3, n, n, n))
    for d, val in enumerate((0.5, -0.3, 0.9)):
        b[d] = val
    o = R.Oracle(n, n, n, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT_HLL)
    o.set_state(prim, b)
    o.advance(2, 0.5)
    assert np.array_equal(o.get_conserved()[1], b)
    np.testing.assert_allclose(o.get_emf()[:, 0, 0, 0], -np.cross([0.4, -0.7, 0.2], [0.5, -0.3, 0.9]), rtol=1e-14)
    # smooth 3D data: conservation, div B, cyclic relabelling of the axes
    n = 12
    prim, b = smooth_mhd_ic(n, 7)
    o = R.Oracle(n, n, n, 1.0 / n, G53, HLL_, VANLEER, EMF_UCT_HLL)
    o.set_state(prim, b)
    c0, b0 = o.get_conserved()
    assert o.advance(3, 0.4) == 0
    c1, b1 = o.get_conserved()
    for v in range(5):
        assert abs(c1[v].sum() - c0[v].sum()) <= 1e-13 * max(np.abs(c0[v]).sum(), 1.0)
    for d in range(3):
        assert abs(b1[d].sum() - b0[d].sum()) <= 1e-13 * np.abs(b0[d]).sum()
    assert np.abs(divb(b1)).max() <= 1e-13 * np.abs(b1).max() * 6
    o2 = R.Oracle(n, n, n, 1.0 / n, G53, HLL_, VANLEER, EMF_UCT_HLL)
    o2.set_state(rot_prim(prim), rot_vector(b))
    o2.advance(3, 0.4)
    p2, b2 = o2.get_state()
    p1, _ = o.get_state()
    np.testing.assert_allclose(p2, rot_prim(p1), rtol=0, atol=1e-13)
    np.testing.assert_allclose(b2, rot_vector(b1), rtol=0, atol=1e-13)


def test_emf_hll2d_linear_wave_second_order(R):
    """Inclined fast wave, HLL fluxes + 2D-HLL EMF: the same convergence the other EMFs show (pre-asymptotic 16 -> 32)."""
    from test_oracle_scheme import HLL as HLL_, run_linear_wave
    errs = [run_linear_wave(R, n, "fast", HLL_, EMF_UCT_HLL) for n in (16, 32)]
    assert errs[0] < 0.1 and math.log2(errs[0] / errs[1]) >= 1.25, errs


# =================================================================================================
# outflow (zero-gradient) boundaries, hydrodynamics (PAPER.md:239 Sod tube, 253)
# =================================================================================================
def run_tube_outflow(R, n, axis, solver=3, t_end=0.2, cfl=0.4):
    """The paper's Sod tube as it is usually set up: one discontinuity in the middle of [0, 1], outflow at both ends."""
    g = 1.4
    dx = 1.0 / n
    x = (np.arange(n) + 0.5) * dx
    shape = [4, 4, 4]
    shape[2 - axis] = n
    bc = [1, 1, 1]
    bc[2 - axis] = n
    left = (x < 0.5).reshape(bc)
    prim = np.zeros([5] + shape)
    prim[0] = np.where(left, 1.0, 0.125)
    prim[4] = np.where(left, 1.0, 0.1)
    dims = shape[::-1]
    o = R.Oracle(dims[0], dims[1], dims[2], dx, g, solver, VANLEER, EMF_NONE, boundary=R.BOUNDARY_OUTFLOW)
    o.set_state(prim)
    rc, _ = o.advance_to(t_end, cfl)
    assert rc == 0
    out, _ = o.get_state()
    sl = [0, 0, 0]
    sl[2 - axis] = slice(None)
    line = out[(slice(None),) + tuple(sl)]
    assert np.all(out == np.broadcast_to(line.reshape([5] + bc), out.shape))
    return x, line


def test_sod_tube_with_outflow_boundaries(R):
    """Roe + linear reconstruction + RK2 as in the paper's Fig. 2, against the exact solution; the
    waves have not reached the ends at t = 0.2, so the L1 error converges at the usual first order of a shocked flow, and
    the result along y and z equals the one along x."""
    from test_oracle_scheme import sod_exact
    _, sample = sod_exact()
    errs = []
    for n in (100, 200):
        x, line = run_tube_outflow(R, n, 0)
        exact = np.array([sample((xx - 0.5) / 0.2) for xx in x]).T      # rho, u, p
        errs.append(np.abs(line[0] - exact[0]).mean() + np.abs(line[1] - exact[1]).mean() + np.abs(line[4] - exact[2]).mean())
    assert errs[0] < 0.02 and errs[1] < 0.62 * errs[0], errs
    xr, ref = run_tube_outflow(R, 100, 0)
    for axis in (1, 2):
        _, line = run_tube_outflow(R, 100, axis)
        perm = {1: [0, 3, 1, 2, 4], 2: [0, 2, 3, 1, 4]}[axis]        # the velocity components rotate with the axis
        np.testing.assert_allclose(line[[0, 1 + axis, 4]], ref[[0, 1, 4]], rtol=0, atol=1e-13)


def test_outflow_lets_a_uniform_flow_and_a_pulse_leave(R):
    """A uniform supersonic flow is a fixed point with zero-gradient ghosts; a density pulse advected out of the box
    leaves it without a reflection (the box returns to the uniform state)."""
    n = 32
    prim = np.zeros((5, 4, 4, n))
    prim[0], prim[1], prim[4] = 1.0, 2.0, 0.6
    o = R.Oracle(n, 4, 4, 1.0 / n, 1.4, HLL, VANLEER, EMF_NONE, boundary=R.BOUNDARY_OUTFLOW)
    o.set_state(prim)
    o.advance(5, 0.4)
    np.testing.assert_allclose(o.get_state()[0], prim, rtol=1e-14, atol=0)
    x = (np.arange(n) + 0.5) / n
    prim[0] = 1.0 + 0.3 * np.exp(-((x - 0.5) / 0.08) ** 2)
    o.set_state(prim)
    rc, _ = o.advance_to(1.0, 0.4)       # the pulse travels two box lengths
    assert rc == 0
    out = o.get_state()[0]
    assert np.abs(out[0] - 1.0).max() < 1e-6 and np.abs(out[1] - 2.0).max() < 1e-6
    with pytest.raises(ValueError):
        R.Oracle(8, 8, 8, 0.125, G53, HLLD, VANLEER, EMF_UCT_HLL, boundary=R.BOUNDARY_OUTFLOW)
    with pytest.raises(ValueError):
        R.Oracle(8, 8, 8, 0.125, G53, HLLD, VANLEER, EMF_UCT, ct_form=1, boundary=R.BOUNDARY_OUTFLOW)


# =================================================================================================
# outflow boundaries with a magnetic field (reading G23: zero-gradient staggered field)
# =================================================================================================
def brio_wu(n, axis, ntrans=4):
    """Brio & Wu (1988) tube along `axis`: rho = 1 | 0.125, p = 1 | 0.1, B_n = 0.75, B_t1 = 1 | -1, gamma = 2."""
    x = (np.arange(n) + 0.5) / n
    shape = [ntrans, ntrans, ntrans]
    shape[2 - axis] = n
    bc = [1, 1, 1]
    bc[2 - axis] = n
    left = (x < 0.5).reshape(bc)
    prim = np.zeros([5] + shape)
    prim[0] = np.where(left, 1.0, 0.125)
    prim[4] = np.where(left, 1.0, 0.1)
    b = np.zeros([3] + shape)
    b[axis] = 0.75
    b[(axis + 1) % 3] = np.where(left, 1.0, -1.0)      # cell-wise constant along the tube: a face value of its own cell
    return prim, b


def run_brio_wu(R, n, axis, boundary, cycles, dt, emf=EMF_UCT, length=1):
    """`length` = 2: the periodic double tube (the tube followed by its mirror image) as the reference."""
    prim, b = brio_wu(n, axis)
    if length == 2:
        prim = np.concatenate([prim, np.flip(prim, 3 - axis)], axis=3 - axis)
        b = np.concatenate([b, np.flip(b, 3 - axis)], axis=3 - axis)
    dims = prim.shape[1:][::-1]
    o = R.Oracle(dims[0], dims[1], dims[2], 1.0 / n, 2.0, HLLD, VANLEER, emf, boundary=boundary)
    o.set_state(prim, b)
    for _ in range(cycles):
        assert o.step(dt) == 0
    return o.get_state()


@pytest.mark.parametrize("emf", [EMF_UCT, EMF_ARITH])
def test_brio_wu_tube_with_outflow_stays_1d_and_matches_the_periodic_double_tube(R, emf):
    """With zero-gradient ghosts the tube stays exactly one-dimensional, B_n stays exactly uniform, and wherever the
    boundaries cannot have been felt (4 cells per RK2 cycle) the run is bit-identical to the periodic double tube, i.e. to
    the scheme already pinned; along y and z it equals the run along x."""
    n, cycles, dt = 64, 6, 0.1 / 64
    ref_line = None
    for axis in range(3):
        p, b = run_brio_wu(R, n, axis, R.BOUNDARY_OUTFLOW, cycles, dt, emf)
        sl = [0, 0, 0]
        sl[2 - axis] = slice(None)
        line_p, line_b = p[(slice(None),) + tuple(sl)], b[(slice(None),) + tuple(sl)]
        bc = [1, 1, 1]
        bc[2 - axis] = n
        assert np.all(p == np.broadcast_to(line_p.reshape([5] + bc), p.shape))          # transverse uniformity, to the bit
        assert np.all(b == np.broadcast_to(line_b.reshape([3] + bc), b.shape))
        assert np.all(line_b[axis] == 0.75) and np.abs(line_b[(axis + 2) % 3]).max() < 1e-14   # planar: B_t2 stays at round-off
        pp, bp = run_brio_wu(R, n, axis, R.BOUNDARY_PERIODIC, cycles, dt, emf, length=2)
        slp = list(sl)
        slp[2 - axis] = slice(0, n)
        per_p, per_b = pp[(slice(None),) + tuple(slp)], bp[(slice(None),) + tuple(slp)]
        m = 4 * cycles + 2
        assert np.array_equal(line_p[:, m:n - m], per_p[:, m:n - m]) and np.array_equal(line_b[:, m:n - m], per_b[:, m:n - m])
        assert np.abs(line_p[0, m:n - m] - np.where(np.arange(m, n - m) < n // 2, 1.0, 0.125)).max() > 0.05   # waves did form
        # rotate the components back to the frame of the x tube
        vel = line_p[[1 + axis, 1 + (axis + 1) % 3, 1 + (axis + 2) % 3]]
        mag = line_b[[axis, (axis + 1) % 3, (axis + 2) % 3]]
        cur = np.concatenate([line_p[[0]], vel, line_p[[4]], mag])
        if ref_line is None:
            ref_line = cur
        else:
            np.testing.assert_allclose(cur, ref_line, rtol=0, atol=1e-13)


def test_mhd_outflow_fixed_point_divb_and_a_pulse_leaving(R):
    """A uniform magnetised flow through the box is a fixed point; a blast reaching all six walls keeps div B at
    round-off on every cell whose six faces belong to the state; a fast pulse carried out of the box leaves the uniform
    state behind."""
    n = 16
    prim = np.zeros((5, n, n, n))
    prim[0], prim[1], prim[2], prim[3], prim[4] = 1.0, 0.9, -0.4, 0.3, 0.7
    b = np.zeros((3, n, n, n))
    b[0], b[1], b[2] = 0.5, -0.3, 0.2
    o = R.Oracle(n, n, n, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT, boundary=R.BOUNDARY_OUTFLOW)
    o.set_state(prim, b)
    assert o.advance(4, 0.3) == 0
    p1, b1 = o.get_state()
    np.testing.assert_allclose(p1, prim, rtol=1e-14, atol=1e-15)
    np.testing.assert_allclose(b1, b, rtol=1e-14, atol=0)
    # blast: over-pressured ball in a uniform oblique field, run until the fast shock has left through the walls
    z, y, x = np.meshgrid(*[(np.arange(n) + 0.5) / n - 0.5] * 3, indexing="ij")
    prim[1:4] = 0.0
    prim[4] = np.where(x * x + y * y + z * z < 0.15 ** 2, 10.0, 0.5)
    o = R.Oracle(n, n, n, 1.0 / n, G53, HLL, VANLEER, EMF_UCT, boundary=R.BOUNDARY_OUTFLOW)
    o.set_state(prim, b)
    rc, _ = o.advance_to(0.25, 0.3)
    assert rc == 0
    p2, b2 = o.get_state()
    assert np.abs(p2[1:4, :, :, 0]).max() > 0.05            # the flow did reach the wall
    div = (b2[0][:-1, :-1, 1:] - b2[0][:-1, :-1, :-1]) + (b2[1][:-1, 1:, :-1] - b2[1][:-1, :-1, :-1]) + \
          (b2[2][1:, :-1, :-1] - b2[2][:-1, :-1, :-1])
    assert np.abs(div).max() <= 1e-13 * np.abs(b2).max()
    # a fast-mode pulse on a super-fast flow along x is carried out: the uniform state remains
    prim[:] = 0.0
    xs = (np.arange(n * 2) + 0.5) / (2 * n)
    prim = np.zeros((5, 4, 4, 2 * n))
    prim[0] = 1.0 + 0.2 * np.exp(-((xs - 0.5) / 0.08) ** 2)
    prim[1], prim[4] = 4.0, 0.6
    bb = np.zeros((3, 4, 4, 2 * n))
    bb[0], bb[1] = 0.5, 0.4
    o = R.Oracle(2 * n, 4, 4, 1.0 / (2 * n), G53, HLLD, VANLEER, EMF_UCT, boundary=R.BOUNDARY_OUTFLOW)
    o.set_state(prim, bb)
    rc, _ = o.advance_to(0.5, 0.4)        # two box lengths at u = 4
    assert rc == 0
    p3, b3 = o.get_state()
    assert np.abs(p3[0] - 1.0).max() < 1e-6 and np.abs(p3[1] - 4.0).max() < 1e-6 and np.abs(b3[1] - 0.4).max() < 1e-6


# =================================================================================================
# PPM with the extremum-preserving limiter (Colella & Woodward 1984; Colella & Sekora 2008; reading G22)
# =================================================================================================
PPM = 4


def _cell_averages(F, xc, dx):
    """exact cell averages from the antiderivative F"""
    return np.array([(F(x + 0.5 * dx) - F(x - 0.5 * dx)) / dx for x in xc])


def test_ppm_is_exact_for_cell_averages_of_a_monotone_cubic(R):
    """The interface formula 7/12, -1/12 reproduces the point values of a cubic from its cell averages, and where the
    data are smooth and monotone no limiter acts (fourth order on regular grids)."""
    f = lambda x: 2.0 + x + 0.3 * x ** 2 + 0.1 * x ** 3
    F = lambda x: 2.0 * x + x ** 2 / 2 + 0.1 * x ** 3 + 0.025 * x ** 4
    for dx in (0.2, 0.05):
        for x0 in (0.3, 1.0, -0.2):
            xc = x0 + dx * np.arange(-2, 3)
            lo, hi = R.ppm_faces(_cell_averages(F, xc, dx))
            # the averages are differences of the antiderivative divided by dx: their own rounding is ~ 1e-16 |F| / dx
            assert abs(lo - f(x0 - 0.5 * dx)) <= 2e-13 and abs(hi - f(x0 + 0.5 * dx)) <= 2e-13
    a = 3.0 - 0.7 * np.arange(5.0)            # linear and constant data come back exactly
    lo, hi = R.ppm_faces(a)
    assert abs(lo - (a[2] + 0.35)) <= 1e-15 and abs(hi - (a[2] - 0.35)) <= 1e-15
    assert R.ppm_faces(np.full(5, 1.25)) == (1.25, 1.25)


def test_ppm_keeps_a_smooth_extremum_and_flattens_a_rough_one(R):
    """What 'extremum-preserving' means (Colella & Sekora 2008): the cell holding the maximum of a parabola keeps the exact
    edge values (the 1984 limiter would set both to the cell value); an isolated spike is flattened."""
    for dx in (0.1, 0.01):
        F = lambda x: x - x ** 3 / 3                      # f = 1 - x^2, maximum inside cell j
        for shift in (0.0, 0.2 * dx, -0.3 * dx):
            xc = shift + dx * np.arange(-2, 3)
            a = _cell_averages(F, xc, dx)
            lo, hi = R.ppm_faces(a)
            assert abs(lo - (1 - (shift - 0.5 * dx) ** 2)) <= 2e-13 and abs(hi - (1 - (shift + 0.5 * dx) ** 2)) <= 2e-13
            assert max(lo, hi) < a[2] or shift != 0.0     # not flattened
    assert R.ppm_faces(np.array([0.0, 0.0, 1.0, 0.0, 0.0])) == (1.0, 1.0)
    assert R.ppm_faces(np.array([1.0, 1.0, 0.0, 1.0, 1.0])) == (0.0, 0.0)
    # a smooth extremum whose neighbouring second differences are much smaller is limited to 1.25 times them
    a = np.array([-0.01, 0.0, 1.0, 0.0, -0.01])           # D2C = -2, D2L = D2R = 1.01: signs differ -> flat
    assert R.ppm_faces(a) == (1.0, 1.0)


def test_ppm_is_monotone_at_discontinuities_and_symmetric(R):
    rng = np.random.default_rng(5)
    step = np.array([0.0, 0.0, 0.0, 1.0, 1.0, 1.0, 1.0])
    for j in range(2, 5):                                   # every cell of a step keeps its faces inside [0, 1]
        lo, hi = R.ppm_faces(step[j - 2:j + 3])
        assert 0.0 <= lo <= 1.0 and 0.0 <= hi <= 1.0 and lo <= hi
    for _ in range(3000):
        a = rng.normal(size=5) * rng.choice([1e-3, 1.0, 30.0])
        lo, hi = R.ppm_faces(a)
        lo_r, hi_r = R.ppm_faces(a[::-1].copy())            # mirror image
        tol = 8e-16 * np.abs(a).max()                      # sums are formed in a fixed order: symmetric up to rounding
        assert abs(lo_r - hi) <= tol and abs(hi_r - lo) <= tol
        lo_n, hi_n = R.ppm_faces(-a)                        # odd in the data
        assert (lo_n, hi_n) == (-lo, -hi)                   # exactly: every operation is odd
        if (a[3] - a[2]) * (a[2] - a[1]) > 0 and (a[2] - a[1]) * (a[1] - a[0]) > 0 and (a[4] - a[3]) * (a[3] - a[2]) > 0:
            # monotone data: the parabola is monotone (no new extremum inside the cell) and stays between the neighbours
            assert min(a[1], a[2]) - 1e-15 <= lo <= max(a[1], a[2]) + 1e-15
            assert min(a[2], a[3]) - 1e-15 <= hi <= max(a[2], a[3]) + 1e-15
            assert abs(hi - a[2]) <= 2 * abs(a[2] - lo) + 1e-15 and abs(a[2] - lo) <= 2 * abs(hi - a[2]) + 1e-15
        else:   # next to an extremum an edge value may leave the range of its two cells (that is the point of the 2008
            # limiter: the extremum of the underlying function lies between the cell values) but only by a bounded amount
            span = a.max() - a.min()
            assert abs(lo - a[2]) <= span and abs(hi - a[2]) <= span


def test_ppm_face_values_converge_at_fourth_order(R):
    errs = []
    for n in (16, 32, 64):
        dx = 1.0 / n
        F = lambda x: -np.cos(2 * np.pi * x) / (2 * np.pi) + 2 * x     # f = sin(2 pi x) + 2
        x0 = 0.1
        xc = x0 + dx * np.arange(-2, 3)
        lo, hi = R.ppm_faces(_cell_averages(F, xc, dx))
        errs.append(abs(hi - (np.sin(2 * np.pi * (x0 + 0.5 * dx)) + 2)))
    assert math.log2(errs[0] / errs[1]) > 3.7 and math.log2(errs[1] / errs[2]) > 3.7, errs


@pytest.mark.parametrize("kind", ["fast", "alfven"])
def test_rk3_ppm_linear_wave_converges_like_the_integrator(R, kind):
    """PPM with RK3 (Fig. 8): third-order convergence at moderate resolution and an error well below the
    second-order scheme's."""
    errs = [run_wave_1d(R, n, PPM, 3, kind) for n in (32, 64)]
    assert math.log2(errs[0] / errs[1]) >= 2.8, errs
    assert errs[1] < 0.2 * run_wave_1d(R, 64, VANLEER, 2, kind)


def test_ppm_scheme_conserves_and_keeps_divb(R):
    from paper_2304_13746_b200 import inputs
    prim, bface, cfg = inputs.make("config3", n=12)
    o = R.Oracle(12, 12, 12, cfg["dx"], cfg["gamma"], HLLD, PPM, EMF_UCT, nstages=3)
    o.set_state(prim.numpy(), bface.numpy())
    c0, b0 = o.get_conserved()
    o.advance(6, 0.3)
    c1, b1 = o.get_conserved()
    for v in range(5):
        assert abs(c1[v].sum() - c0[v].sum()) <= 1e-13 * max(np.abs(c0[v]).sum(), 1.0)
    for d in range(3):
        assert abs(b1[d].sum() - b0[d].sum()) <= 1e-13 * np.abs(b0).sum()
    div = sum(np.roll(b1[d], -1, axis=2 - d) - b1[d] for d in range(3)) / cfg["dx"]
    assert np.abs(div).max() * cfg["dx"] <= 1e-13 * np.abs(b1).max()
    # a uniform state is a fixed point, bit for bit
    prim[:] = prim[:, :1, :1, :1]
    bface[:] = 0.3
    o.set_state(prim.numpy(), bface.numpy())
    o.advance(2, 0.3)
    p2, b2 = o.get_state()
    assert (p2 == p2[:, :1, :1, :1]).all() and (b2 == 0.3).all()
    # refused with the 2D-HLL EMF (3-cell edge reconstruction only)
    with pytest.raises(Exception):
        R.Oracle(12, 12, 12, cfg["dx"], cfg["gamma"], HLL, PPM, 4)
