"""Pins of the UPWIND-SIDE rule of the upwind-contact EMF E^c ("E^c ... upwind-contact", Gardiner & Stone
2005; reading G10 of DESIGN.md: the transverse EMF derivative at a face is taken from the cell the face mass flux comes
FROM; an exactly vanishing mass flux takes the mean of the two candidates).

The plane-parallel identity (test_oracle_scheme.py) cannot see that rule: there the two candidates are equal.  Every
test here depends on WHICH side is taken and none retypes the oracle's edge formula:

 (a) domain of dependence: in a uniform, fully supersonic flow (flat reconstruction + HLL = pure donor-cell fluxes) a
     one-edge bump of the vector potential must leave the edge diagonally UPSTREAM of it unchanged to the bit and must
     change the other eight edges of its 3 x 3 neighbourhood -- for all four sign quadrants of the in-plane velocity and
     for each of the three edge families;
 (b) closed form of the same situation: with every face flux coming from its donor cell the E^c construction
     collapses to a fixed combination of donor-cell values, evaluated here straight from the input arrays;
 (c) field-loop advection along the diagonal (Gardiner & Stone 2005, sect. 3.2 test problem): the magnetic energy never
     grows over 250 cycles (the wrong side is anti-diffusive and grows it);
 (d) the `== 0 => mean` branch: in a fluid at rest with uniform density every face mass flux is exactly zero, and then
     E^c must coincide with E^0 (the same construction with averaged instead of upwinded derivatives, pinned by its own
     closed form in test_oracle_scheme.py);
 (e) the vector-potential update of (a): A_new = -dt E after one Euler step, so the untouched upstream edge keeps A = 0
     difference to the bit as well (checks the claim through idfxref_get_potential, i.e. what CT actually applies).
"""
import itertools

import numpy as np
import pytest

HLL, HLLD = 0, 2
FLAT, VANLEER = 0, 2
EMF_ARITH, EMF_UCT, EMF_UCT0 = 1, 2, 3
G53 = 5.0 / 3.0


def perm_axes(arr, comp):
    """Array [k][j][i] of a problem written for the z edge family -> the same problem relabelled so that the edge
    family is `comp` (cyclic relabelling x->y->z->x applied (comp - 2) mod 3 times ... done on the index triple)."""
    # written for (a, b, c) = (x, y, z); target (a, b, c) = cyclic with c = comp
    a, b, c = (comp + 1) % 3, (comp + 2) % 3, comp
    # source array axes are (z, y, x) = (c_src, b_src, a_src); the target wants axis order (z, y, x) of the new labels
    src_axis_of = {a: 2, b: 1, c: 0}            # where the data of new direction d sits in the source array
    return np.ascontiguousarray(np.transpose(arr, (src_axis_of[2], src_axis_of[1], src_axis_of[0])))


def build_problem(n, nc, va, vb, vc, bump_edge, amp, comp):
    """Uniform flow (v_a, v_b, v_c) in the local frame (a, b, c) of edge family `comp`, rho = 1, p = 0.1, and the
    face field curl(A_c) of a one-edge bump A_c(I-1/2, J-1/2, all c) = amp on top of a uniform field.  Returns
    prim [5][nz][ny][nx], bface [3][nz][ny][nx] in global labels, plus the local-frame arrays for the closed form."""
    I, J = bump_edge
    dx = 1.0 / n
    A = np.zeros((nc, n, n))                    # local layout [c][b][a]; A[., J, I] sits at (I-1/2, J-1/2)
    A[:, J, I] = amp
    # discrete curl, periodic: B_a(i-1/2, j) = [A(i-1/2, j+1/2) - A(i-1/2, j-1/2)]/dx ; B_b(i, j-1/2) = -[A(i+1/2, .) - A(i-1/2, .)]/dx
    Ba = (np.roll(A, -1, axis=1) - A) / dx + 0.03
    Bb = -(np.roll(A, -1, axis=2) - A) / dx - 0.02
    Bc = np.full_like(A, 0.05)
    loc_v = {"a": va, "b": vb, "c": vc}
    a, b, c = (comp + 1) % 3, (comp + 2) % 3, comp
    prim = np.empty((5,) + perm_axes(A, comp).shape)
    prim[0] = 1.0
    prim[4] = 0.1
    prim[1 + a], prim[1 + b], prim[1 + c] = va, vb, vc
    bface = np.empty((3,) + prim.shape[1:])
    bface[a], bface[b], bface[c] = perm_axes(Ba, comp), perm_axes(Bb, comp), perm_axes(Bc, comp)
    return prim, bface, (Ba, Bb, loc_v)


def edge_field(R, prim, bface, comp, dt=1e-3, want_potential=False):
    """E_comp on the edge lattice after ONE Euler stage (flat + HLL + E^c), back in the local layout [c][b][a]."""
    nz, ny, nx = prim.shape[1:]
    o = R.Oracle(nx, ny, nz, 1.0 / max(nx, ny, nz), G53, HLL, FLAT, EMF_UCT, nstages=1,
                 ct_form=R.CT_POTENTIAL if want_potential else R.CT_FACE)
    o.set_state(prim, bface)
    assert o.step(dt) == 0
    E = o.get_potential()[comp] if want_potential else o.get_emf()[comp]
    a, b, c = (comp + 1) % 3, (comp + 2) % 3, comp
    glob_axis_of = {2: 0, 1: 1, 0: 2}           # global direction d -> axis of a [z][y][x] array
    return np.ascontiguousarray(np.transpose(E, (glob_axis_of[c], glob_axis_of[b], glob_axis_of[a])))


QUADRANTS = list(itertools.product((+1, -1), (+1, -1)))


@pytest.mark.parametrize("comp", [0, 1, 2])
@pytest.mark.parametrize("sa,sb", QUADRANTS)
def test_uct_domain_of_dependence(R, comp, sa, sb):
    """(a): the edge diagonally upstream of the bump is bit-identical with and without the bump; the other eight edges of
    the 3 x 3 block around it change; nothing outside the block changes."""
    n, nc, I, J = 12, 4, 6, 5
    va, vb = 2.0 * sa, 1.7 * sb                 # Mach ~ 5 and ~ 4 against a = sqrt(gamma p / rho) = 0.41: fully one-sided fans
    p0, b0, _ = build_problem(n, nc, va, vb, 0.3, (I, J), 0.0, comp)
    p1, b1, _ = build_problem(n, nc, va, vb, 0.3, (I, J), 1e-3 / n, comp)
    E0, E1 = edge_field(R, p0, b0, comp), edge_field(R, p1, b1, comp)
    changed = E0 != E1                           # [c][b][a]
    assert (changed == changed[0]).all()         # the problem is uniform along c
    got = {(i, j) for j, i in zip(*np.nonzero(changed[0]))}
    block = {(I + di, J + dj) for di in (-1, 0, 1) for dj in (-1, 0, 1)}
    upstream_corner = (I - sa, J - sb)           # v_a > 0: the flow arrives from lower a, the untouched edge is at I - 1
    assert upstream_corner not in got, "the edge diagonally upstream of the bump saw it: wrong upwind side"
    assert got == block - {upstream_corner}


@pytest.mark.parametrize("comp", [0, 1, 2])
@pytest.mark.parametrize("sa,sb", QUADRANTS)
def test_uct_potential_update_keeps_upstream_edge(R, comp, sa, sb):
    """(e): the same statement on what constrained transport applies: after one Euler step of the vector-potential
    form A = -dt E, the upstream corner edge carries bit-identical potential with and without the bump."""
    n, nc, I, J = 10, 4, 4, 6
    va, vb = 1.9 * sa, 2.1 * sb
    p0, b0, _ = build_problem(n, nc, va, vb, -0.4, (I, J), 0.0, comp)
    p1, b1, _ = build_problem(n, nc, va, vb, -0.4, (I, J), 2e-3 / n, comp)
    A0 = edge_field(R, p0, b0, comp, want_potential=True)
    A1 = edge_field(R, p1, b1, comp, want_potential=True)
    assert A0[0, J - sb, I - sa] == A1[0, J - sb, I - sa]
    assert A0[0, J + sb, I + sa] != A1[0, J + sb, I + sa]
    assert A0[0, J, I] != A1[0, J, I]


@pytest.mark.parametrize("comp", [0, 1, 2])
@pytest.mark.parametrize("sa,sb", QUADRANTS)
def test_uct_donor_cell_closed_form(R, comp, sa, sb):
    """(b): closed form for a fully supersonic uniform flow.  Every face value is its donor cell's (flat reconstruction,
    one-sided HLL fan): E_c^(a)(i-1/2, j) = -(v_a Bc_b - v_b B_a,face)(donor in a), E_c^(b)(i, j-1/2) = +(v_b Bc_a - v_a B_b,face)
    (donor in b), and the upwinded derivatives all come from the donor side, so with (iu, ju) the donor indices of the edge
    (i-1/2, j-1/2) and (iL, iR) = (i-1, i), (jL, jR) = (j-1, j):
        E = 1/4 [E^a(jL) + E^a(jR) + E^b(iL) + E^b(iR)]
          + 1/4 [2 E^b(iu) - Ec(iu, jL) - Ec(iu, jR)] + 1/4 [2 E^a(ju) - Ec(iL, ju) - Ec(iR, ju)]."""
    n, nc = 10, 4
    rng = np.random.default_rng(40 + comp)
    va, vb, vc = 2.2 * sa, 1.8 * sb, 0.25
    # a smooth random potential A_c(a, b) instead of one bump: every edge is tested at once
    dx = 1.0 / n
    A = np.zeros((nc, n, n))
    A[:] = 1e-2 * dx * rng.standard_normal((n, n))[None]
    Ba = (np.roll(A, -1, axis=1) - A) / dx + 0.03      # on a-faces (i-1/2, j)
    Bb = -(np.roll(A, -1, axis=2) - A) / dx - 0.02     # on b-faces (i, j-1/2)
    a, b, c = (comp + 1) % 3, (comp + 2) % 3, comp
    shape = perm_axes(A, comp).shape
    prim = np.empty((5,) + shape)
    prim[0], prim[4] = 1.0, 0.1
    prim[1 + a], prim[1 + b], prim[1 + c] = va, vb, vc
    bface = np.empty((3,) + shape)
    bface[a], bface[b], bface[c] = perm_axes(Ba, comp), perm_axes(Bb, comp), perm_axes(np.full_like(A, 0.05), comp)
    E = edge_field(R, prim, bface, comp)[0]            # [b][a]
    Ba, Bb = Ba[0], Bb[0]
    Bca = 0.5 * (Ba + np.roll(Ba, -1, axis=1))         # cell-centred: mean of the two bounding faces (G1)
    Bcb = 0.5 * (Bb + np.roll(Bb, -1, axis=0))
    Ecc = vb * Bca - va * Bcb                          # -(v x B)_c at cell centres
    def cell(arr, i, j):
        return arr[j % n, i % n]
    worst = 0.0
    for j in range(n):
        for i in range(n):
            iL, iR, jL, jR = i - 1, i, j - 1, j
            iu, ju = (iL if va > 0 else iR), (jL if vb > 0 else jR)
            Ea = {jj: -(va * cell(Bcb, iu, jj) - vb * cell(Ba, i, jj)) for jj in (jL, jR)}   # a-faces (i-1/2, jj), donor iu
            Eb = {ii: +(vb * cell(Bca, ii, ju) - va * cell(Bb, ii, j)) for ii in (iL, iR)}   # b-faces (ii, j-1/2), donor ju
            want = (0.25 * (Ea[jL] + Ea[jR] + Eb[iL] + Eb[iR])
                    + 0.25 * (2.0 * Eb[iu] - cell(Ecc, iu, jL) - cell(Ecc, iu, jR))
                    + 0.25 * (2.0 * Ea[ju] - cell(Ecc, iL, ju) - cell(Ecc, iR, ju)))
            worst = max(worst, abs(E[j, i] - want))
    assert worst <= 1e-14 * np.abs(E).max()


def field_loop(n, nz, A0=1e-3, radius=0.3):
    """Gardiner & Stone (2005) field loop on the unit square: A_z = A0 max(radius - r, 0) sampled at the z edges,
    B = curl A, rho = p = 1, advected along the diagonal."""
    dx = 1.0 / n
    e = np.arange(n) * dx - 0.5                   # edge positions (i - 1/2) dx on [-1/2, 1/2)
    X, Y = np.meshgrid(e, e, indexing="xy")       # [j][i]
    A = A0 * np.maximum(radius - np.hypot(X, Y), 0.0)
    bx = (np.roll(A, -1, axis=0) - A) / dx
    by = -(np.roll(A, -1, axis=1) - A) / dx
    prim = np.empty((5, nz, n, n))
    prim[0], prim[4] = 1.0, 1.0
    prim[1], prim[2], prim[3] = 1.0, 1.0, 0.0
    b = np.zeros((3, nz, n, n))
    b[0], b[1] = bx[None], by[None]
    return prim, b


def test_field_loop_magnetic_energy_never_grows(R):
    """(c): 250 RK2 cycles (0.6 crossings of the diagonal) of the field loop on 16 x 16 x 4 with HLLD + van Leer + E^c:
    the magnetic energy of the face field is non-increasing cycle by cycle and has decayed at the end; the run stays
    physical and divergence-free.  Taking the derivative from the wrong side is anti-diffusive and fails this."""
    n, nz = 16, 4
    prim, b = field_loop(n, nz)
    o = R.Oracle(n, n, nz, 1.0 / n, G53, HLLD, VANLEER, EMF_UCT)
    o.set_state(prim, b)
    def energy():
        _, bf = o.get_conserved()
        return 0.5 * float((bf ** 2).sum())
    e_prev = e0 = energy()
    for cycle in range(25):
        assert o.advance(10, 0.4) == 0
        e = energy()
        assert e <= e_prev * (1.0 + 1e-12), (cycle, e / e_prev)
        e_prev = e
    assert 0.3 * e0 < e_prev < 0.95 * e0
    _, bf = o.get_conserved()
    div = (np.roll(bf[0], -1, axis=2) - bf[0]) + (np.roll(bf[1], -1, axis=1) - bf[1]) + (np.roll(bf[2], -1, axis=0) - bf[2])
    assert np.abs(div).max() <= 1e-13 * np.abs(bf).max()


def test_zero_mass_flux_takes_the_mean(R):
    """(d): fluid at rest, uniform density, non-uniform pressure and field: every face mass flux of the first stage is
    exactly zero (HLL: F[rho] = [S_R 0 - S_L 0 + S_L S_R (rho_R - rho_L)]/(S_R - S_L) = 0; HLLD would not do, its contact
    speed S_M follows the total-pressure jump), so every upwinded derivative is the
    mean of its two candidates and E^c equals E^0 edge by edge.  (With v = 0 the candidates are -2 E_face of two
    different faces, so any one-sided choice at zero differs at the level of the EMF itself.)"""
    n = 8
    rng = np.random.default_rng(11)
    dx = 1.0 / n
    Apot = 0.05 * dx * rng.standard_normal((3, n, n, n))
    ax, ay, az = Apot
    b = np.empty((3, n, n, n))                    # [z][y][x]; discrete curl of edge-centred A, periodic
    b[0] = (np.roll(az, -1, axis=1) - az) / dx - (np.roll(ay, -1, axis=0) - ay) / dx + 0.3
    b[1] = (np.roll(ax, -1, axis=0) - ax) / dx - (np.roll(az, -1, axis=2) - az) / dx - 0.2
    b[2] = (np.roll(ay, -1, axis=2) - ay) / dx - (np.roll(ax, -1, axis=1) - ax) / dx + 0.1
    prim = np.zeros((5, n, n, n))
    prim[0] = 1.0
    prim[4] = 1.0 + 0.2 * rng.random((n, n, n))
    E = {}
    for emf in (EMF_UCT, EMF_UCT0):
        o = R.Oracle(n, n, n, dx, G53, HLL, VANLEER, emf, nstages=1)
        o.set_state(prim, b)
        assert o.step(1e-3) == 0
        for d in range(3):
            F, _ = o.get_flux(d)
            assert not F[0].any(), "the mass flux of a fluid at rest with uniform density must vanish exactly"
        E[emf] = o.get_emf()
    scale = np.abs(E[EMF_UCT0]).max()
    assert scale > 1e-4
    np.testing.assert_allclose(E[EMF_UCT], E[EMF_UCT0], rtol=0, atol=2e-15 * scale + 1e-18)
