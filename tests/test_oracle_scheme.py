"""Pins for the grid-level scheme of the oracle (SURVEY.md §8(c) "Pins" table): exact Sod solution, direction
symmetry, uniform states, conservation, div B, the E^c plane-parallel identity, the RK2 amplification factor,
closed-form dt, and second-order convergence of linear MHD waves (Eq. 14).  Expected values
are closed forms, exact solutions computed here by an independent textbook routine, or numbers the paper prints."""
import math
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

HLL, HLLC, HLLD, ROE, RUSANOV = 0, 1, 2, 3, 4
FLAT, MINMOD, VANLEER = 0, 1, 2
EMF_NONE, EMF_ARITH, EMF_UCT, EMF_UCT0 = 0, 1, 2, 3
G53 = 5.0 / 3.0
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def read_golden(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            out[k] = float(v)
    return out


# cyclic relabelling x->y->z->x of arrays laid out [z][y][x]: s'(x',y',z') = s(y', z', x')
def rot_scalar(s):
    return np.ascontiguousarray(np.transpose(s, (1, 2, 0)))


def rot_vector(v):
    return np.stack([rot_scalar(v[2]), rot_scalar(v[0]), rot_scalar(v[1])])


def rot_prim(p):
    return np.concatenate([rot_scalar(p[0])[None], rot_vector(p[1:4]), rot_scalar(p[4])[None]])


def divb(b):
    return (np.roll(b[0], -1, 2) - b[0]) + (np.roll(b[1], -1, 1) - b[1]) + (np.roll(b[2], -1, 0) - b[2])


def curl_np(ax, ay, az, dx):
    up = lambda a, d: np.roll(a, -1, d)
    return np.stack([((up(az, 1) - az) - (up(ay, 0) - ay)) / dx,
                     ((up(ax, 0) - ax) - (up(az, 2) - az)) / dx,
                     ((up(ay, 2) - ay) - (up(ax, 1) - ax)) / dx])


# =================================================================================================
# Sod tube against the exact Riemann solution (reading G4: P_L = 1)
# =================================================================================================
def sod_exact(g=1.4, L=(1.0, 0.0, 1.0), Rr=(0.125, 0.0, 0.1)):
    """Textbook exact Riemann solver (left rarefaction, right shock).  Returns a sampler xi -> (rho,u,p)."""
    rl, ul, pl = L
    rr, ur, pr = Rr
    al, ar = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)

    def fk(p, rk, pk, ak):
        if p > pk:
            A, B = 2.0 / ((g + 1) * rk), (g - 1) / (g + 1) * pk
            return (p - pk) * math.sqrt(A / (p + B))
        return 2 * ak / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1)

    lo, hi = 1e-8, 10.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if fk(mid, rl, pl, al) + fk(mid, rr, pr, ar) + (ur - ul) > 0:
            hi = mid
        else:
            lo = mid
    ps = 0.5 * (lo + hi)
    us = 0.5 * (ul + ur) + 0.5 * (fk(ps, rr, pr, ar) - fk(ps, rl, pl, al))
    rsl = rl * (ps / pl) ** (1 / g)
    q = (g - 1) / (g + 1)
    rsr = rr * (ps / pr + q) / (q * ps / pr + 1)
    shock = ur + ar * math.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))
    asl = al * (ps / pl) ** ((g - 1) / (2 * g))
    head, tail = ul - al, us - asl

    def sample(xi):
        xi = np.asarray(xi, dtype=float)
        rho = np.where(xi < head, rl, 0.0)
        u = np.where(xi < head, ul, 0.0)
        p = np.where(xi < head, pl, 0.0)
        fan = (xi >= head) & (xi < tail)
        c = 2 / (g + 1) + q / al * (ul - xi)
        rho = np.where(fan, rl * c ** (2 / (g - 1)), rho)
        u = np.where(fan, 2 / (g + 1) * (al + (g - 1) / 2 * ul + xi), u)
        p = np.where(fan, pl * c ** (2 * g / (g - 1)), p)
        m = (xi >= tail) & (xi < us)
        rho, u, p = np.where(m, rsl, rho), np.where(m, us, u), np.where(m, ps, p)
        m = (xi >= us) & (xi < shock)
        rho, u, p = np.where(m, rsr, rho), np.where(m, us, u), np.where(m, ps, p)
        m = xi >= shock
        rho, u, p = np.where(m, rr, rho), np.where(m, ur, u), np.where(m, pr, p)
        return rho, u, p

    return dict(p_star=ps, u_star=us, rho_star_L=rsl, rho_star_R=rsr, shock_speed=shock, head=head, tail=tail), sample


def test_sod_exact_solver_matches_golden():
    vals, _ = sod_exact()
    for k, v in read_golden("sod_exact.txt").items():
        assert vals[k] == pytest.approx(v, abs=2e-6)


def run_double_tube(R, n, axis, solver, limiter=VANLEER, t_end=0.2, cfl=0.4):
    """Periodic double Sod tube of length 2 along `axis` (n x 4 x 4 cells): high state on [0.5,1.5)."""
    g = 1.4
    dx = 2.0 / n
    x = (np.arange(n) + 0.5) * dx
    hi = (x >= 0.5) & (x < 1.5)
    shape = [4, 4, 4]
    shape[2 - axis] = n                       # arrays are [z][y][x]
    bc = [1, 1, 1]
    bc[2 - axis] = n
    prof = hi.reshape(bc)
    prim = np.zeros([5] + shape)
    prim[0] = np.where(prof, 1.0, 0.125)
    prim[4] = np.where(prof, 1.0, 0.1)
    dims = shape[::-1]
    o = R.Oracle(dims[0], dims[1], dims[2], dx, g, solver, limiter, EMF_NONE)
    o.set_state(prim)
    t = 0.0
    while t < t_end - 1e-14:
        dt = min(o.compute_dt(cfl), t_end - t)
        assert o.step(dt) == 0
        t += dt
    out, _ = o.get_state()
    sl = [0, 0, 0]
    sl[2 - axis] = slice(None)
    line = out[(slice(None),) + tuple(sl)]    # [5][n]
    # transverse uniformity (exact: identical arithmetic in every pencil)
    assert np.all(out == np.broadcast_to(line.reshape([5] + bc), out.shape))
    return x, line


@pytest.mark.parametrize("solver", [ROE, HLLC, HLL, RUSANOV])
def test_sod_plateaus_and_convergence(R, solver):
    vals, sample = sod_exact()
    t = 0.2
    errs = []
    for n in (100, 200, 400):
        x, q = run_double_tube(R, n, 0, solver)
        rho, u, p = q[0], q[1], q[4]
        right = x >= 1.0
        ex_r = sample((x[right] - 1.5) / t)
        ex_l = sample(-(x[~right] - 0.5) / t)
        rho_ex = np.concatenate([ex_l[0], ex_r[0]])
        errs.append(np.abs(rho - rho_ex).mean())
    # plateaus at the finest resolution, right half: between tail and contact, and between contact and shock
    xt, xc, xs = 1.5 + vals["tail"] * t, 1.5 + vals["u_star"] * t, 1.5 + vals["shock_speed"] * t
    mL = (x > xt + 0.25 * (xc - xt)) & (x < xc - 0.25 * (xc - xt))
    mR = (x > xc + 0.25 * (xs - xc)) & (x < xs - 0.25 * (xs - xc))
    assert mL.sum() > 5 and mR.sum() > 5
    tol = 1e-3 if solver not in (HLL, RUSANOV) else 3e-3
    assert np.abs(rho[mL].mean() - vals["rho_star_L"]) < tol
    assert np.abs(rho[mR].mean() - vals["rho_star_R"]) < tol
    for m in (mL, mR):
        assert np.abs(u[m].mean() - vals["u_star"]) < tol
        assert np.abs(p[m].mean() - vals["p_star"]) < tol
    # mirrored half is the mirror image
    assert np.allclose(rho[: x.size // 2], rho[x.size // 2:][::-1], atol=1e-12)
    assert np.allclose(u[: x.size // 2], -u[x.size // 2:][::-1], atol=1e-12)
    o1 = math.log2(errs[0] / errs[1])
    o2 = math.log2(errs[1] / errs[2])
    assert 0.55 < o1 < 1.25 and 0.55 < o2 < 1.25, (errs, o1, o2)


@pytest.mark.parametrize("solver", [ROE, HLLC])
def test_sod_along_y_and_z_equals_x(R, solver):
    x, qx = run_double_tube(R, 100, 0, solver)
    _, qy = run_double_tube(R, 100, 1, solver)
    _, qz = run_double_tube(R, 100, 2, solver)
    # normal velocity is component 1+axis
    for q, ax in ((qy, 1), (qz, 2)):
        np.testing.assert_allclose(q[0], qx[0], rtol=0, atol=1e-13)
        np.testing.assert_allclose(q[4], qx[4], rtol=0, atol=1e-13)
        np.testing.assert_allclose(q[1 + ax], qx[1], rtol=0, atol=1e-13)
        others = [c for c in (1, 2, 3) if c != 1 + ax]
        assert np.all(q[others] == 0.0)


# =================================================================================================
# Whole-scheme invariants on 3D data
# =================================================================================================
def smooth_mhd_ic(n, seed, amp=0.2):
    """Smooth periodic 3D fields, B = curl A (discretely solenoidal).  Test-local, not a BASELINE config."""
    rng = np.random.default_rng(seed)
    dx = 1.0 / n
    c = (np.arange(n) + 0.5) * dx
    e = np.arange(n) * dx
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")

    def wave(Xa, Ya, Za):
        k = rng.integers(1, 3, size=3)
        ph = rng.uniform(0, 2 * np.pi)
        return np.sin(2 * np.pi * (k[0] * Xa + k[1] * Ya + k[2] * Za) + ph)
    prim = np.empty((5, n, n, n))
    prim[0] = 1.0 + amp * wave(X, Y, Z)
    for d in range(3):
        prim[1 + d] = 0.5 * wave(X, Y, Z) + 0.3 * wave(X, Y, Z)
    prim[4] = 1.0 + amp * wave(X, Y, Z)
    Ze, Ye, Xe = np.meshgrid(e, e, e, indexing="ij")
    ax = 0.1 * wave(X, Ye, Ze)
    ay = 0.1 * wave(Xe, Y, Ze)
    az = 0.1 * wave(Xe, Ye, Z)
    b = curl_np(ax, ay, az, dx)
    b[0] += 0.3
    b[1] -= 0.2
    b[2] += 0.1
    return prim, b


MHD_COMBOS = [(HLLD, VANLEER, EMF_UCT0), (RUSANOV, VANLEER, EMF_UCT), (HLL, VANLEER, EMF_ARITH), (HLLD, VANLEER, EMF_UCT), (HLLD, MINMOD, EMF_ARITH),
              (ROE, VANLEER, EMF_UCT), (ROE, FLAT, EMF_ARITH)]


@pytest.mark.parametrize("solver,limiter,emf", MHD_COMBOS)
def test_mhd_conservation_and_divb(R, solver, limiter, emf):
    """Sum of rho, m, E and of each face-B component constant to round-off; div B at round-off (north_star;
    PAPER.md:97, 294)."""
    n = 16
    prim, b = smooth_mhd_ic(n, 5)
    assert np.abs(divb(b)).max() < 1e-13
    o = R.Oracle(n, n, n, 1.0 / n, G53, solver, limiter, emf)
    o.set_state(prim, b)
    c0, b0 = o.get_conserved()
    nsteps = 8
    assert o.advance(nsteps, 0.4) == 0
    c1, b1 = o.get_conserved()
    for v in range(5):
        scale = max(np.abs(c0[v]).sum(), 1.0)
        assert abs(c1[v].sum() - c0[v].sum()) <= 1e-13 * scale
    for d in range(3):
        assert abs(b1[d].sum() - b0[d].sum()) <= 1e-13 * np.abs(b0[d]).sum() + 1e-13
    assert np.abs(divb(b1)).max() / np.abs(b1).max() <= 1e-13
    assert np.abs(c1 - c0).max() > 1e-3          # it did evolve
    assert o.roe_fallbacks() == 0


@pytest.mark.parametrize("solver,limiter", [(HLL, VANLEER), (HLLC, MINMOD), (ROE, VANLEER)])
def test_hd_conservation(R, solver, limiter):
    n = 16
    prim, _ = smooth_mhd_ic(n, 6)
    o = R.Oracle(n, n, n, 1.0 / n, G53, solver, limiter, EMF_NONE)
    o.set_state(prim)
    c0, _ = o.get_conserved()
    assert o.advance(8, 0.4) == 0
    c1, _ = o.get_conserved()
    for v in range(5):
        assert abs(c1[v].sum() - c0[v].sum()) <= 1e-13 * max(np.abs(c0[v]).sum(), 1.0)


@pytest.mark.parametrize("solver,emf", [(HLL, EMF_ARITH), (HLLD, EMF_UCT), (HLLD, EMF_UCT0), (ROE, EMF_ARITH), (HLLC, EMF_NONE)])
def test_uniform_state_stays_uniform(R, solver, emf):
    """Any uniform (rho, v, p, B) is a fixed point: U unchanged, bit-identical across cells (north_star)."""
    n = 8
    prim = np.empty((5, n, n, n))
    for v, val in enumerate((1.3, 0.4, -0.7, 0.2, 0.8)):
        prim[v] = val
    b = None
    if emf != EMF_NONE:
        b = np.empty((3, n, n, n))
        for d, val in enumerate((0.5, -0.3, 0.9)):
            b[d] = val
    o = R.Oracle(n, n, n, 1.0 / n, G53, solver, VANLEER, emf)
    o.set_state(prim, b)
    c0, _ = o.get_conserved()
    o.advance(3, 0.5)
    c1, b1 = o.get_conserved()
    for v in range(5):
        assert np.all(c1[v] == c1[v].flat[0])
        assert c1[v].flat[0] == pytest.approx(c0[v].flat[0], rel=1e-14, abs=1e-15)
    if b is not None:
        assert np.array_equal(b1, b)
        # arithmetic / E^c EMF of a uniform state is exactly -v x B
        E = o.get_emf()
        vv, BB = np.array([0.4, -0.7, 0.2]), np.array([0.5, -0.3, 0.9])
        np.testing.assert_allclose(E[:, 0, 0, 0], -np.cross(vv, BB), rtol=1e-14)


@pytest.mark.parametrize("solver,limiter,emf", [(HLLD, VANLEER, EMF_UCT), (ROE, VANLEER, EMF_ARITH), (HLL, MINMOD, EMF_UCT)])
def test_direction_symmetry_mhd(R, solver, limiter, emf):
    """An initial condition cyclically relabelled x->y->z gives the cyclically relabelled result."""
    n = 12
    prim, b = smooth_mhd_ic(n, 7)
    o = R.Oracle(n, n, n, 1.0 / n, G53, solver, limiter, emf)
    o.set_state(prim, b)
    o.advance(3, 0.4)
    p1, b1 = o.get_state()
    o2 = R.Oracle(n, n, n, 1.0 / n, G53, solver, limiter, emf)
    o2.set_state(rot_prim(prim), rot_vector(b))
    o2.advance(3, 0.4)
    p2, b2 = o2.get_state()
    assert o.last_dt() == pytest.approx(o2.last_dt(), rel=1e-14)
    np.testing.assert_allclose(p2, rot_prim(p1), rtol=0, atol=1e-13)
    np.testing.assert_allclose(b2, rot_vector(b1), rtol=0, atol=1e-13)


def test_direction_symmetry_hd(R):
    n = 12
    prim, _ = smooth_mhd_ic(n, 8)
    res = []
    for pr in (prim, rot_prim(prim)):
        o = R.Oracle(n, n, n, 1.0 / n, G53, HLLC, MINMOD, EMF_NONE)
        o.set_state(pr)
        o.advance(3, 0.4)
        res.append(o.get_state()[0])
    np.testing.assert_allclose(res[1], rot_prim(res[0]), rtol=0, atol=1e-13)


def test_emf_uct_plane_parallel_identity(R):
    """Grid-aligned plane-parallel flow (1D in x, run in 3D, uniform v_y, v_z): with the E^c scheme the edge
    EMF equals the 1D Riemann-flux EMF, E_z,edge(i-1/2) = -F_x[B_y](i-1/2) and E_y,edge = +F_x[B_z], so CT
    reproduces the 1D flux-divergence update of B_t (Gardiner & Stone 2005 design requirement).  The arithmetic
    average does NOT have this property, which also checks the mode switch."""
    nx, ny, nz = 32, 4, 4
    dx = 1.0 / nx
    x = (np.arange(nx) + 0.5) * dx
    prim = np.empty((5, nz, ny, nx))
    prim[0] = 1.0 + 0.3 * np.sin(2 * np.pi * x)
    prim[1] = 0.4 * np.cos(2 * np.pi * x)
    prim[2] = 0.35
    prim[3] = -0.25
    prim[4] = 1.0 + 0.2 * np.cos(4 * np.pi * x)
    b = np.empty((3, nz, ny, nx))
    b[0] = 0.7
    b[1] = 0.5 + 0.3 * np.sin(2 * np.pi * x)
    b[2] = -0.4 + 0.2 * np.cos(2 * np.pi * x)
    out = {}
    for emf in (EMF_UCT, EMF_UCT0, EMF_ARITH):
        o = R.Oracle(nx, ny, nz, dx, G53, HLLD, VANLEER, emf)
        o.set_state(prim, b)
        dt = o.compute_dt(0.4)
        o.step(dt)                      # after the step the stored fluxes/EMFs are those of stage 2
        E = o.get_emf()
        Fx, _ = o.get_flux(0)
        out[emf] = (E, Fx)
    for mode in (EMF_UCT, EMF_UCT0):                                  # both Gardiner-Stone schemes have the property
        E, Fx = out[mode]
        np.testing.assert_allclose(E[2], -Fx[5], rtol=0, atol=1e-13)  # E_z = -F_x[B_y]
        np.testing.assert_allclose(E[1], Fx[6], rtol=0, atol=1e-13)   # E_y = +F_x[B_z]
    E, Fx = out[EMF_ARITH]
    assert np.abs(E[2] + Fx[5]).max() > 1e-4 and np.abs(E[1] - Fx[6]).max() > 1e-4


def test_emf_e0_closed_form(R):
    """E^0 (Gardiner & Stone 2005) = (1/2) sum of the four face EMFs - (1/4) sum of the four cell-centred -(v x B):
    rebuilt here from the oracle's own face fluxes and primitives of the second stage."""
    n = 10
    prim, b = smooth_mhd_ic(n, 17)
    o = R.Oracle(n, n, n, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT0)
    o.set_state(prim, b)
    dt = o.compute_dt(0.3)
    # make stage 2 of this cycle start from a state we can also get: run one Euler-like probe with tiny dt so that
    # the stage-2 input equals the initial state to 1e-12 and the stored fluxes are those of the initial state
    o.step(1e-14)
    E = o.get_emf()
    Fx, _ = o.get_flux(0)
    Fy, _ = o.get_flux(1)
    p0, b0 = prim, b
    bc = np.stack([0.5 * (b0[d] + np.roll(b0[d], -1, 2 - d)) for d in range(3)])
    v = p0[1:4]
    Ecz = v[1] * bc[0] - v[0] * bc[1]
    Ezx, Ezy = -Fx[5], Fy[6]                                            # E_z on x-faces and on y-faces
    dn = lambda a, ax: np.roll(a, 1, ax)                               # value one cell down along array axis ax
    ref = 0.5 * (Ezx + dn(Ezx, 1) + Ezy + dn(Ezy, 2)) - 0.25 * (Ecz + dn(Ecz, 2) + dn(Ecz, 1) + dn(dn(Ecz, 1), 2))
    np.testing.assert_allclose(E[2], ref, rtol=0, atol=1e-11)
    assert dt > 0


def test_arithmetic_emf_is_second_order_average(R):
    """For smooth data the arithmetic edge EMF equals -v x B at the edge to O(dx^2)."""
    errs = []
    for n in (16, 32):
        dx = 1.0 / n
        c = (np.arange(n) + 0.5) * dx
        e = np.arange(n) * dx
        Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
        prim = np.empty((5, n, n, n))
        prim[0], prim[4] = 1.0, 1.0
        vx = lambda x, y, z: 0.3 * np.sin(2 * np.pi * y)
        vy = lambda x, y, z: 0.2 * np.cos(2 * np.pi * x)
        prim[1], prim[2], prim[3] = vx(X, Y, Z), vy(X, Y, Z), 0.0
        bxf = lambda x, y, z: 0.5 + 0.1 * np.sin(2 * np.pi * y)      # independent of x: solenoidal
        byf = lambda x, y, z: 0.4 + 0.1 * np.cos(2 * np.pi * x)
        b = np.empty((3, n, n, n))
        Zf, Yf, Xf = np.meshgrid(c, c, e, indexing="ij")
        b[0] = bxf(Xf, Yf, Zf)
        Zf, Yf, Xf = np.meshgrid(c, e, c, indexing="ij")
        b[1] = byf(Xf, Yf, Zf)
        b[2] = 0.0
        o = R.Oracle(n, n, n, dx, G53, HLLD, VANLEER, EMF_ARITH)
        o.set_state(prim, b)
        o.step(1e-9)                                                  # state unchanged to 1e-9
        Ez = o.get_emf()[2]
        Ze, Ye, Xe = np.meshgrid(c, e, e, indexing="ij")
        exact = vy(Xe, Ye, Ze) * bxf(Xe, Ye, Ze) - vx(Xe, Ye, Ze) * byf(Xe, Ye, Ze)
        errs.append(np.abs(Ez - exact).max())
    assert errs[0] < 2e-2 and math.log2(errs[0] / errs[1]) > 1.7


def test_rk2_amplification_factor(R):
    """Supersonic uniform flow + flat reconstruction + HLL is exactly first-order upwind advection of rho, which
    is linear; one RK2 step multiplies the Fourier mode by 1 + z + z^2/2, z = -(u dt/dx)(1 - exp(-i k dx))
    (Eq. 9 with Tab. 1)."""
    n = 16
    dx = 1.0 / n
    x = (np.arange(n) + 0.5) * dx
    for axis in range(3):
        shape = [1, 1, 1]
        shape[2 - axis] = n
        prim = np.zeros([5] + shape)
        prim[0] = (1.0 + 0.1 * np.cos(2 * np.pi * x) + 0.05 * np.sin(4 * np.pi * x)).reshape(shape)
        prim[1 + axis] = 3.0
        prim[4] = 0.1
        dims = shape[::-1]
        o = R.Oracle(dims[0], dims[1], dims[2], dx, 1.4, HLL, FLAT, EMF_NONE)
        o.set_state(prim)
        dt = 0.37 * dx / 3.0
        o.step(dt)
        rho1 = o.get_state()[0][0].ravel()
        f0, f1 = np.fft.fft(prim[0].ravel()), np.fft.fft(rho1)
        for m in (1, 2):
            z = -(3.0 * dt / dx) * (1 - np.exp(-2j * np.pi * m / n))
            assert f1[m] / f0[m] == pytest.approx(1 + z + z * z / 2, abs=1e-13)
        assert f1[0] == pytest.approx(f0[0], rel=1e-15)


def test_dt_closed_forms(R):
    """Eq. 10 without eta: dt = cfl dx / sum_d (|v_d| + c_f,d) for a uniform state."""
    n, dx, cfl = 6, 0.01, 0.3
    v = np.array([0.3, -1.1, 0.6])
    B = np.array([0.5, -0.2, 0.8])
    rho, p = 1.7, 0.9
    prim = np.empty((5, n, n, n))
    prim[0], prim[4] = rho, p
    for d in range(3):
        prim[1 + d] = v[d]
    b = np.empty((3, n, n, n))
    for d in range(3):
        b[d] = B[d]
    a2, b2 = G53 * p / rho, B @ B / rho
    tot = 0.0
    for d in range(3):
        cf = math.sqrt(0.5 * (a2 + b2 + math.sqrt((a2 + b2) ** 2 - 4 * a2 * B[d] ** 2 / rho)))
        tot += abs(v[d]) + cf
    o = R.Oracle(n, n, n, dx, G53, HLLD, VANLEER, EMF_UCT)
    o.set_state(prim, b)
    assert o.compute_dt(cfl) == pytest.approx(cfl * dx / tot, rel=1e-14)
    # at rest, hydrodynamics: cfl dx / (3 a)
    prim[1:4] = 0.0
    o = R.Oracle(n, n, n, dx, G53, HLLC, MINMOD, EMF_NONE)
    o.set_state(prim)
    assert o.compute_dt(cfl) == pytest.approx(cfl * dx / (3 * math.sqrt(a2)), rel=1e-14)
    # advance() uses exactly compute_dt on the current state (G9)
    o.advance(1, cfl)
    assert o.last_dt() == pytest.approx(cfl * dx / (3 * math.sqrt(a2)), rel=1e-14)


def test_dt_takes_global_max_over_cells_and_faces(R):
    """One hot cell sets dt; the face->cell mapping (G8) uses the larger of the two faces of each cell."""
    n, dx = 8, 1.0 / 8
    prim = np.empty((5, n, n, n))
    prim[0], prim[4] = 1.0, 0.6
    prim[1:4] = 0.0
    o = R.Oracle(n, n, n, dx, G53, HLL, FLAT, EMF_NONE)
    o.set_state(prim)
    dt0 = o.compute_dt(0.5)
    prim[4, 3, 4, 5] = 6.0          # 10x the pressure in one cell
    o.set_state(prim)
    dt1 = o.compute_dt(0.5)
    a_hot, a = math.sqrt(G53 * 6.0), math.sqrt(G53 * 0.6)
    assert dt0 == pytest.approx(0.5 * dx / (3 * a), rel=1e-14)
    # flat reconstruction: every face of the hot cell sees c = a_hot -> all three directions
    assert dt1 == pytest.approx(0.5 * dx / (3 * a_hot), rel=1e-14)


def test_rejects_bad_arguments(R):
    with pytest.raises(ValueError):
        R.Oracle(8, 8, 8, 0.1, G53, HLLC, VANLEER, EMF_UCT)       # HLLC is HD-only
    with pytest.raises(ValueError):
        R.Oracle(8, 8, 8, 0.1, G53, HLLD, VANLEER, EMF_NONE)      # HLLD is MHD-only
    with pytest.raises(ValueError):
        R.Oracle(8, 8, 8, -0.1, G53, HLL, VANLEER, EMF_NONE)
    o = R.Oracle(4, 4, 4, 0.1, G53, HLL, VANLEER, EMF_NONE)
    with pytest.raises(ValueError):
        o.compute_dt(1.5)                                          # sigma_CFL < 1
    prim = np.ones((5, 4, 4, 4))
    prim[4, 1, 1, 1] = -1.0
    assert o.set_state(prim) == 0 and o.status() == -5             # unphysical flag, no floors (G13)


# =================================================================================================
# Linear MHD wave convergence (Eq. 14), cubic grids 16^3 -> 32^3 -> 64^3 (north_star)
# =================================================================================================
def primitive_jacobian(rho, p, B1, B2, B3, g):
    """Linearised ideal MHD about a state at rest, W = (rho, v1, v2, v3, p, B2, B3), textbook form."""
    A = np.zeros((7, 7))
    A[0, 1] = rho
    A[1, 4] = 1 / rho
    A[1, 5] = B2 / rho
    A[1, 6] = B3 / rho
    A[2, 5] = -B1 / rho
    A[3, 6] = -B1 / rho
    A[4, 1] = g * p
    A[5, 1] = B2
    A[5, 2] = -B1
    A[6, 1] = B3
    A[6, 3] = -B1
    return A


def linear_wave_mode(kind):
    gold = read_golden("linear_wave_speeds.txt")
    A = primitive_jacobian(1.0, 0.6, 1.0, 1.5, 0.0, G53)
    lam, vec = np.linalg.eig(A)
    target = {"fast": gold["c_fast"], "alfven": gold["c_alfven"], "slow": gold["c_slow"]}[kind]
    k = int(np.argmin(np.abs(lam.real - target)))
    assert abs(lam[k].real - target) < 1e-12 and abs(lam[k].imag) < 1e-12   # the paper's speeds
    r = vec[:, k].real
    r = r / np.abs(r).max()
    return target, r


def linear_wave_ic(n, r, eps):
    """Background rho=1, P=3/5, B1=1, B2=3/2 in the frame e1=(1,1,1)/sqrt3, e2=(1,-1,0)/sqrt2, e3=e1 x e2;
    phase 2 pi (x+y+z); perturbation eps cos(phase) r.  B from a vector potential sampled on edges."""
    dx = 1.0 / n
    e1 = np.array([1, 1, 1]) / math.sqrt(3)
    e2 = np.array([1, -1, 0]) / math.sqrt(2)
    e3 = np.cross(e1, e2)
    c = (np.arange(n) + 0.5) * dx
    e = np.arange(n) * dx
    kk = 2 * math.pi * math.sqrt(3)                      # phase = kk * x1
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    cosph = np.cos(2 * np.pi * (X + Y + Z))
    prim = np.empty((5, n, n, n))
    prim[0] = 1.0 + eps * r[0] * cosph
    dv = r[1] * e1[:, None, None, None] + r[2] * e2[:, None, None, None] + r[3] * e3[:, None, None, None]
    prim[1:4] = eps * dv * cosph
    prim[4] = 0.6 + eps * r[4] * cosph
    # A = (sin(phase)/kk) (dB3 e2 - dB2 e3)  =>  curl A = cos(phase) (dB2 e2 + dB3 e3)
    avec = eps * (r[6] * e2 - r[5] * e3) / kk
    Ze, Ye, Xc = np.meshgrid(e, e, c, indexing="ij")
    ax = avec[0] * np.sin(2 * np.pi * (Xc + Ye + Ze))
    Ze, Yc, Xe = np.meshgrid(e, c, e, indexing="ij")
    ay = avec[1] * np.sin(2 * np.pi * (Xe + Yc + Ze))
    Zc, Ye, Xe = np.meshgrid(c, e, e, indexing="ij")
    az = avec[2] * np.sin(2 * np.pi * (Xe + Ye + Zc))
    b = curl_np(ax, ay, az, dx)
    b0 = 1.0 * e1 + 1.5 * e2
    for d in range(3):
        b[d] += b0[d]
    return prim, b, b0


def run_linear_wave(R, n, kind, solver, emf, cfl=0.6, eps=1e-6):
    speed, r = linear_wave_mode(kind)
    prim, b, b0 = linear_wave_ic(n, r, eps)
    o = R.Oracle(n, n, n, 1.0 / n, G53, solver, VANLEER, emf)
    o.set_state(prim, b)
    period = (1.0 / math.sqrt(3)) / speed
    nsteps = int(math.ceil(period / o.compute_dt(cfl)))
    dt = period / nsteps
    for _ in range(nsteps):
        assert o.step(dt) == 0
    p1, b1 = o.get_state()
    # Eq. 14: per-component L1 error normalised by eps N^3 N_components, summed in quadrature
    bg = [1.0, 0.0, 0.0, 0.0, 0.6]
    comps = [(prim[v] - bg[v], p1[v] - bg[v]) for v in range(5)] + [(b[d] - b0[d], b1[d] - b0[d]) for d in range(3)]
    nz_comp = sum(1 for a, _ in comps if np.abs(a).max() > 1e-3 * eps)
    err = math.sqrt(sum((np.abs(a - c).sum() / (eps * n ** 3 * nz_comp)) ** 2 for a, c in comps))
    return err


WAVE_CASES = [("fast", HLLD, EMF_UCT, (16, 32, 64)), ("fast", HLL, EMF_ARITH, (16, 32)), ("fast", ROE, EMF_UCT, (16, 32)),
              ("fast", HLLD, EMF_ARITH, (16, 32)), ("alfven", HLLD, EMF_UCT, (16, 32)), ("alfven", ROE, EMF_ARITH, (16, 32)),
              ("alfven", HLL, EMF_UCT, (16, 32)), ("fast", HLLD, EMF_UCT0, (16, 32))]


@pytest.fixture(scope="module")
def wave_errors(R):
    """All runs at once in threads (ctypes releases the GIL; every oracle context is independent)."""
    jobs = [(kind, solver, emf, n) for kind, solver, emf, ns in WAVE_CASES for n in ns]
    jobs.sort(key=lambda j: -j[3])
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        res = list(ex.map(lambda j: run_linear_wave(R, j[3], j[0], j[1], j[2]), jobs))
    return dict(zip(jobs, res))


@pytest.mark.parametrize("kind,solver,emf,ns", WAVE_CASES)
def test_linear_wave_convergence_3d(wave_errors, kind, solver, emf, ns):
    """Wave inclined to all three axes, 16 cells per wavelength along each axis at 16^3.  The van Leer limiter
    clips the extrema, so 16^3 -> 32^3 is pre-asymptotic (observed 1.3-1.5, the same as the 1D runs below at
    the same resolution); 32^3 -> 64^3 must show second order (paper Fig. 7)."""
    errs = [wave_errors[(kind, solver, emf, n)] for n in ns]
    assert errs[0] < 0.1                                 # the wave survived one period at 16^3
    orders = [math.log2(a / b) for a, b in zip(errs[:-1], errs[1:])]
    assert orders[0] >= 1.25, (kind, solver, emf, errs)
    if len(orders) > 1:
        assert orders[1] >= 1.8, (kind, solver, emf, errs)


def run_linear_wave_1d(R, n, kind, solver, axis, cfl=0.6, eps=1e-6):
    """Same eigenmode, wave vector along a grid axis (n x 1 x 1 cells): cheap enough to reach the asymptotic range."""
    speed, r = linear_wave_mode(kind)
    dx = 1.0 / n
    c = np.cos(2 * np.pi * (np.arange(n) + 0.5) * dx)
    shape = [1, 1, 1]
    shape[2 - axis] = n
    c = c.reshape(shape)
    a, b_, e = axis, (axis + 1) % 3, (axis + 2) % 3
    prim = np.empty([5] + shape)
    prim[0] = 1 + eps * r[0] * c
    prim[1 + a], prim[1 + b_], prim[1 + e] = eps * r[1] * c, eps * r[2] * c, eps * r[3] * c
    prim[4] = 0.6 + eps * r[4] * c
    bf = np.empty([3] + shape)
    bf[a], bf[b_], bf[e] = 1.0, 1.5 + eps * r[5] * c, eps * r[6] * c     # transverse B does not vary across its own faces
    dims = shape[::-1]
    o = R.Oracle(dims[0], dims[1], dims[2], dx, G53, solver, VANLEER, EMF_UCT)
    o.set_state(prim, bf)
    period = 1.0 / speed
    nsteps = int(math.ceil(period / o.compute_dt(cfl)))
    for _ in range(nsteps):
        assert o.step(period / nsteps) == 0
    p1, b1 = o.get_state()
    tot = [np.abs(p1[v] - prim[v]).mean() for v in range(5)] + [np.abs(b1[d] - bf[d]).mean() for d in range(3)]
    return math.sqrt(sum(t * t for t in tot)) / eps


@pytest.mark.parametrize("kind", ["fast", "alfven", "slow"])
@pytest.mark.parametrize("solver", [HLL, HLLD, ROE])
def test_linear_wave_second_order_1d(R, kind, solver):
    errs = [run_linear_wave_1d(R, n, kind, solver, 0) for n in (64, 128)]
    assert math.log2(errs[0] / errs[1]) >= 1.9, (kind, solver, errs)


def test_linear_wave_1d_direction_symmetry(R):
    ref = run_linear_wave_1d(R, 64, "fast", HLLD, 0)
    for axis in (1, 2):
        assert run_linear_wave_1d(R, 64, "fast", HLLD, axis) == pytest.approx(ref, rel=1e-5)
