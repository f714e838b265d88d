"""Pins for the point-wise parts of the oracle (SURVEY.md §8(c) "Pins" table): flux functions, Riemann
solvers, Roe eigen-system, limiters.  Nothing here compares the oracle with itself: every expected value
is a closed form, an identity of the mathematics, a textbook routine retyped here independently, or a
number the paper prints."""
import os

import numpy as np
import pytest

HLL, HLLC, HLLD, ROE, RUSANOV = 0, 1, 2, 3, 4
FLAT, MINMOD, VANLEER = 0, 1, 2
G = 5.0 / 3.0
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def read_golden(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            out[k] = float(v)
    return out


def rand_state(rng, mhd=True):
    W = np.zeros(7)
    W[0] = rng.uniform(0.2, 3.0)
    W[1:4] = rng.uniform(-2.0, 2.0, 3)
    W[4] = rng.uniform(0.1, 3.0)
    if mhd:
        W[5:7] = rng.uniform(-2.0, 2.0, 2)
    return W


# ---- independent restatement of the ideal-MHD flux (Eq. 1-4) -------------------
def flux_np(W, Bn, g):
    rho, u, v, w, p, By, Bz = W
    B2 = Bn * Bn + By * By + Bz * Bz
    E = p / (g - 1) + 0.5 * rho * (u * u + v * v + w * w) + 0.5 * B2
    pT = p + 0.5 * B2
    vB = u * Bn + v * By + w * Bz
    return np.array([rho * u, rho * u * u + pT - Bn * Bn, rho * u * v - Bn * By, rho * u * w - Bn * Bz,
                     (E + pT) * u - Bn * vB, u * By - v * Bn, u * Bz - w * Bn])


def cons_np(W, Bn, g):
    rho, u, v, w, p, By, Bz = W
    E = p / (g - 1) + 0.5 * rho * (u * u + v * v + w * w) + 0.5 * (Bn * Bn + By * By + Bz * Bz)
    return np.array([rho, rho * u, rho * v, rho * w, E, By, Bz])


def test_phys_flux_matches_equations(R):
    rng = np.random.default_rng(1)
    for _ in range(200):
        W, Bn = rand_state(rng), rng.uniform(-2, 2)
        np.testing.assert_allclose(R.phys_flux(G, W, Bn), flux_np(W, Bn, G), rtol=1e-14, atol=1e-14)
        np.testing.assert_allclose(R.cons_from_prim(G, W, Bn), cons_np(W, Bn, G), rtol=1e-15)


@pytest.mark.parametrize("solver,mhd", [(HLL, False), (HLLC, False), (ROE, False), (RUSANOV, False), (HLL, True),
                                        (HLLD, True), (ROE, True), (RUSANOV, True)])
def test_flux_consistency(R, solver, mhd):
    """F_solver(U, U) = F(U) (north_star pin)."""
    rng = np.random.default_rng(2)
    for _ in range(300):
        W = rand_state(rng, mhd)
        Bn = rng.uniform(-2, 2) if mhd else 0.0
        F, c, fb = R.riemann(solver, G, W, W, Bn)
        ref = flux_np(W, Bn, G)
        assert fb == 0
        assert np.abs(F - ref).max() <= 1e-14 * max(1.0, np.abs(ref).max())


def test_wave_speeds_davis_and_cface(R):
    """Closed forms: a = sqrt(gamma p/rho); c_f from the quartic; c_face = max(|S_L|,|S_R|)."""
    rng = np.random.default_rng(3)
    for _ in range(200):
        WL, WR, Bn = rand_state(rng), rand_state(rng), rng.uniform(-2, 2)

        def cf(W):
            a2 = G * W[4] / W[0]
            bn2, bt2 = Bn * Bn / W[0], (W[5] ** 2 + W[6] ** 2) / W[0]
            # roots of c^4 - (a2+b2) c^2 + a2 bn2 = 0
            r = np.roots([1.0, -(a2 + bn2 + bt2), a2 * bn2])
            return np.sqrt(r.real.max())
        SL, SR = R.wave_speeds(G, WL, WR, Bn)
        assert SL == pytest.approx(min(WL[1] - cf(WL), WR[1] - cf(WR)), rel=1e-12)
        assert SR == pytest.approx(max(WL[1] + cf(WL), WR[1] + cf(WR)), rel=1e-12)
        for s in (HLL, HLLD, ROE):
            assert R.riemann(s, G, WL, WR, Bn)[1] == max(abs(SL), abs(SR))
    # hydrodynamics: exactly the sound speed
    W = np.array([1.3, 0.2, 0, 0, 0.9, 0, 0])
    SL, SR = R.wave_speeds(1.4, W, W, 0.0)
    a = np.sqrt(1.4 * 0.9 / 1.3)
    assert SL == pytest.approx(0.2 - a, rel=1e-15) and SR == pytest.approx(0.2 + a, rel=1e-15)


def test_hll_supersonic_and_formula(R):
    rng = np.random.default_rng(4)
    for _ in range(100):
        WL, WR, Bn = rand_state(rng), rand_state(rng), rng.uniform(-1, 1)
        SL, SR = R.wave_speeds(G, WL, WR, Bn)
        F = R.riemann(HLL, G, WL, WR, Bn)[0]
        FL, FR, UL, UR = flux_np(WL, Bn, G), flux_np(WR, Bn, G), cons_np(WL, Bn, G), cons_np(WR, Bn, G)
        if SL >= 0:
            ref = FL
        elif SR <= 0:
            ref = FR
        else:
            ref = (SR * FL - SL * FR + SL * SR * (UR - UL)) / (SR - SL)
        np.testing.assert_allclose(F, ref, rtol=1e-13, atol=1e-13)
    # boosted so that the whole fan moves right / left: pure upwinding
    WL, WR = rand_state(rng), rand_state(rng)
    for boost, side in ((20.0, WL), (-20.0, WR)):
        a, b = WL.copy(), WR.copy()
        a[1] += boost
        b[1] += boost
        s = a if boost > 0 else b
        for solver in (HLL, HLLD, ROE):
            F = R.riemann(solver, G, a, b, 0.3)[0]
            np.testing.assert_allclose(F, flux_np(s, 0.3, G), rtol=1e-12)


def test_rusanov_is_central_flux_minus_half_cface_jump(R):
    """PAPER.md:81 "Lax-Friedrichs Rusanov flux": F = (F_L+F_R)/2 - (c/2)(U_R-U_L), c = max(|u|+c_f) of the two sides;
    identical to HLL when the fan is symmetric (S_R = -S_L), and never less diffusive than HLL."""
    rng = np.random.default_rng(41)
    for _ in range(200):
        WL, WR, Bn = rand_state(rng), rand_state(rng), rng.uniform(-1, 1)
        F, c, fb = R.riemann(RUSANOV, G, WL, WR, Bn)

        def cf(W):
            a2, b2 = G * W[4] / W[0], (Bn * Bn + W[5] ** 2 + W[6] ** 2) / W[0]
            return np.sqrt(0.5 * (a2 + b2 + np.sqrt((a2 + b2) ** 2 - 4 * a2 * Bn * Bn / W[0])))
        lam = max(abs(WL[1]) + cf(WL), abs(WR[1]) + cf(WR))
        assert c == pytest.approx(lam, rel=1e-13) and fb == 0
        ref = 0.5 * (flux_np(WL, Bn, G) + flux_np(WR, Bn, G)) - 0.5 * lam * (cons_np(WR, Bn, G) - cons_np(WL, Bn, G))
        np.testing.assert_allclose(F, ref, rtol=1e-13, atol=1e-13)
    # symmetric fan: same speeds on both sides and u = 0  =>  S_R = -S_L  =>  HLL = Rusanov
    for _ in range(50):
        WL = rand_state(rng)
        WL[1] = 0.0
        WR = WL.copy()
        WR[2:4] = rng.uniform(-1, 1, 2)          # a shear and a rotation of B_t keep |u| + c_f equal
        th = rng.uniform(0, 2 * np.pi)
        bt = np.hypot(WL[5], WL[6])
        WR[5], WR[6] = bt * np.cos(th), bt * np.sin(th)
        np.testing.assert_allclose(R.riemann(RUSANOV, G, WL, WR, 0.4)[0], R.riemann(HLL, G, WL, WR, 0.4)[0], atol=1e-13)


def test_hllc_fan_integral_and_pressure(R):
    """Integral of the HLLC fan over [S_L,S_R] equals the HLL average; p* is the same from both sides."""
    rng = np.random.default_rng(5)
    g = 1.4
    for _ in range(300):
        WL, WR = rand_state(rng, False), rand_state(rng, False)
        S, st = R.hllc_fan(g, WL, WR)
        SL, SS, SR = S
        UL, UR = cons_np(WL, 0, g)[:5], cons_np(WR, 0, g)[:5]
        FL, FR = flux_np(WL, 0, g)[:5], flux_np(WR, 0, g)[:5]
        lhs = ((SS - SL) * st[0] + (SR - SS) * st[1]) / (SR - SL)
        rhs = (SR * UR - SL * UL - (FR - FL)) / (SR - SL)
        np.testing.assert_allclose(lhs, rhs, rtol=1e-12, atol=1e-12)
        pL = WL[4] + WL[0] * (SL - WL[1]) * (SS - WL[1])
        pR = WR[4] + WR[0] * (SR - WR[1]) * (SS - WR[1])
        assert pL == pytest.approx(pR, rel=1e-11, abs=1e-11)
        # momentum of the star states moves with S*
        assert st[0][1] == pytest.approx(st[0][0] * SS, rel=1e-13)
        assert st[1][1] == pytest.approx(st[1][0] * SS, rel=1e-13)


def test_hlld_fan_integral(R):
    """sum(fan widths x fan states) = S_R U_R - S_L U_L - (F_R - F_L): the HLLD states satisfy the integral
    conservation law over the Riemann fan (Miyoshi & Kusano 2005)."""
    rng = np.random.default_rng(6)
    for _ in range(300):
        WL, WR, Bn = rand_state(rng), rand_state(rng), rng.uniform(-2, 2)
        S, st = R.hlld_fan(G, WL, WR, Bn)
        SL, SsL, SM, SsR, SR = S
        assert SL < SM < SR and SsL <= SM <= SsR
        UL, UR = cons_np(WL, Bn, G), cons_np(WR, Bn, G)
        FL, FR = flux_np(WL, Bn, G), flux_np(WR, Bn, G)
        lhs = (SsL - SL) * st[0] + (SM - SsL) * st[1] + (SsR - SM) * st[2] + (SR - SsR) * st[3]
        rhs = SR * UR - SL * UL - (FR - FL)
        scale = np.abs(rhs).max() + np.abs(SR * UR).max()
        assert np.abs(lhs - rhs).max() <= 1e-13 * scale
        # normal velocity S_M and total pressure are constant across the fan: rho* S_M = m*_n
        for s in st:
            assert s[1] == pytest.approx(s[0] * SM, rel=1e-13, abs=1e-14)


def test_hlld_fan_ordering_for_moderate_jumps(R):
    """For jumps up to 10 % the five speeds are ordered (with the Davis estimate G5 very strong jumps can
    put S*_K outside [S_L,S_R]; the selection order of O7 then picks the outer state first)."""
    rng = np.random.default_rng(61)
    for _ in range(300):
        WL, Bn = rand_state(rng), rng.uniform(-2, 2)
        WR = WL * (1 + rng.uniform(-0.1, 0.1, 7))
        SL, SsL, SM, SsR, SR = R.hlld_fan(G, WL, WR, Bn)[0]
        assert SL <= SsL <= SM <= SsR <= SR


def test_hlld_bn_zero_and_degenerate(R):
    """B_n = 0 needs no special case (zero-width double-star fan); B_t = 0 with B_n^2 ~ rho a^2 exercises G6."""
    rng = np.random.default_rng(7)
    for _ in range(100):
        WL, WR = rand_state(rng), rand_state(rng)
        S, st = R.hlld_fan(G, WL, WR, 0.0)
        assert S[1] == S[2] == S[3]
        F = R.riemann(HLLD, G, WL, WR, 0.0)[0]
        assert np.all(np.isfinite(F))
    W = np.array([1.0, 0.0, 0.1, -0.1, 0.6, 0.0, 0.0])
    F = R.riemann(HLLD, G, W, W, 1.0)[0]          # gamma p = B_n^2: c_f = c_a = a
    np.testing.assert_allclose(F, flux_np(W, 1.0, G), atol=1e-14)


@pytest.mark.parametrize("solver,mhd", [(HLLC, False), (HLLD, True), (ROE, False), (ROE, True)])
def test_isolated_contact_is_exact(R, solver, mhd):
    """A jump in rho only (u, p, B continuous) moving at speed u: flux = physical flux of the upwind side."""
    rng = np.random.default_rng(8)
    for _ in range(100):
        WL = rand_state(rng, mhd)
        WR = WL.copy()
        WR[0] = rng.uniform(0.2, 3.0)
        Bn = rng.uniform(-1, 1) if mhd else 0.0
        if mhd:
            # a contact carries a jump in rho only if v_t, B_t are continuous; that is what we have
            pass
        for u in (0.0, 0.37, -0.52):
            a, b = WL.copy(), WR.copy()
            a[1] = b[1] = u
            F = R.riemann(solver, G, a, b, Bn)[0]
            up = a if u >= 0 else b
            ref = flux_np(up, Bn, G)
            if u == 0.0:
                ref = flux_np(a, Bn, G)   # both sides give the same flux at rest
                np.testing.assert_allclose(flux_np(b, Bn, G), ref, atol=1e-14)
            assert np.abs(F - ref).max() <= 2e-14 * max(1.0, np.abs(ref).max())


@pytest.mark.parametrize("solver", [HLLD, ROE])
def test_isolated_rotational_discontinuity_is_exact(R, solver):
    """rho, p, |B_t|, u equal on both sides; B_t rotated; dv_t = -+ dB_t/sqrt(rho) (Alfven relation):
    a single Alfven wave moving at u -+ |B_n|/sqrt(rho).  HLLD and Roe resolve it exactly."""
    rng = np.random.default_rng(9)
    for _ in range(100):
        rho, p, u = rng.uniform(0.3, 2), rng.uniform(0.2, 2), rng.uniform(-0.3, 0.3)
        Bn = rng.uniform(0.3, 1.5) * rng.choice([-1, 1])
        bt, th1, th2 = rng.uniform(0.2, 1.5), rng.uniform(0, 2 * np.pi), rng.uniform(0, 2 * np.pi)
        BL = bt * np.array([np.cos(th1), np.sin(th1)])
        BR = bt * np.array([np.cos(th2), np.sin(th2)])
        vL = rng.uniform(-1, 1, 2)
        for right_going in (True, False):
            # right-going Alfven wave (speed u + |Bn|/sqrt(rho)): dv = -sgn(Bn) dB/sqrt(rho)
            sg = -np.sign(Bn) if right_going else np.sign(Bn)
            vR = vL + sg * (BR - BL) / np.sqrt(rho)
            WL = np.array([rho, u, vL[0], vL[1], p, BL[0], BL[1]])
            WR = np.array([rho, u, vR[0], vR[1], p, BR[0], BR[1]])
            speed = u + (1 if right_going else -1) * abs(Bn) / np.sqrt(rho)
            # Rankine-Hugoniot sanity of the construction itself
            dF = flux_np(WR, Bn, G) - flux_np(WL, Bn, G)
            dU = cons_np(WR, Bn, G) - cons_np(WL, Bn, G)
            np.testing.assert_allclose(dF, speed * dU, atol=1e-13)
            F = R.riemann(solver, G, WL, WR, Bn)[0]
            ref = flux_np(WL if speed > 0 else WR, Bn, G)
            assert np.abs(F - ref).max() <= 1e-13 * max(1.0, np.abs(ref).max())


# ---- Roe ---------------------------------------------------------------------------------------
def test_roe_eigensystem_orthonormal(R):
    rng = np.random.default_rng(10)
    for _ in range(200):
        WL, WR, Bn = rand_state(rng), rand_state(rng), rng.uniform(-2, 2)
        ok, lam, Rc, Lc = R.roe_system(G, WL, WR, Bn)
        if not ok:
            continue
        np.testing.assert_allclose(Lc @ Rc.T, np.eye(7), atol=1e-12)
        assert np.all(np.diff(lam) >= -1e-14)


def test_roe_exact_property(R):
    """sum_k lambda_k alpha_k r_k = F_R - F_L for arbitrary state pairs (the defining Roe property)."""
    rng = np.random.default_rng(11)
    n = 0
    for _ in range(400):
        WL, WR, Bn = rand_state(rng), rand_state(rng), rng.uniform(-2, 2)
        ok, lam, Rc, Lc = R.roe_system(G, WL, WR, Bn)
        if not ok:
            continue
        n += 1
        dU = cons_np(WR, Bn, G) - cons_np(WL, Bn, G)
        dF = flux_np(WR, Bn, G) - flux_np(WL, Bn, G)
        alpha = Lc @ dU
        got = (lam * alpha) @ Rc
        assert np.abs(got - dF).max() <= 1e-12 * max(1.0, np.abs(dF).max())
        # and the flux the oracle returns is the upwinded form of the same decomposition
        F = R.riemann(ROE, G, WL, WR, Bn)[0]
        ref = 0.5 * (flux_np(WL, Bn, G) + flux_np(WR, Bn, G)) - 0.5 * (np.abs(lam) * alpha) @ Rc
        np.testing.assert_allclose(F, ref, rtol=1e-12, atol=1e-12)
    assert n > 300


def test_roe_eigenvectors_against_fd_jacobian(R):
    """For L = R the Roe matrix is the flux Jacobian: A r_k = lambda_k r_k, A from central differences."""
    rng = np.random.default_rng(12)
    for _ in range(30):
        W, Bn = rand_state(rng), rng.uniform(-2, 2)
        ok, lam, Rc, Lc = R.roe_system(G, W, W, Bn)
        assert ok
        U = cons_np(W, Bn, G)
        A = np.zeros((7, 7))
        for c in range(7):
            h = 1e-6 * max(1.0, abs(U[c]))
            up, um = U.copy(), U.copy()
            up[c] += h
            um[c] -= h
            A[:, c] = (R.flux_from_cons(G, up, Bn) - R.flux_from_cons(G, um, Bn)) / (2 * h)
        for k in range(7):
            r = Rc[k]
            assert np.abs(A @ r - lam[k] * r).max() <= 1e-6 * max(1.0, np.abs(r).max()) * max(1.0, np.abs(lam).max())


def test_roe_speeds_match_paper_linear_wave(R):
    """PAPER.md:261 prints c_f = 2, c_A = 1, c_s = 0.5 for rho=1, P=3/5, B1=1, B2=3/2."""
    gold = read_golden("linear_wave_speeds.txt")
    W = np.array([1.0, 0, 0, 0, 0.6, 1.5, 0.0])
    ok, lam, _, _ = R.roe_system(G, W, W, 1.0)
    cf, ca, cs = gold["c_fast"], gold["c_alfven"], gold["c_slow"]
    np.testing.assert_allclose(lam, [-cf, -ca, -cs, 0, cs, ca, cf], atol=1e-14)
    SL, SR = R.wave_speeds(G, W, W, 1.0)
    assert SR == pytest.approx(cf, rel=1e-15) and SL == pytest.approx(-cf, rel=1e-15)


def roe_hd_textbook(WL, WR, g):
    """Independent 5-wave Roe solver for the Euler equations (Roe 1981 as in Toro's textbook), no entropy fix."""
    rL, uL, vL, wL, pL = WL[:5]
    rR, uR, vR, wR, pR = WR[:5]
    EL = pL / (g - 1) + 0.5 * rL * (uL ** 2 + vL ** 2 + wL ** 2)
    ER = pR / (g - 1) + 0.5 * rR * (uR ** 2 + vR ** 2 + wR ** 2)
    HL, HR = (EL + pL) / rL, (ER + pR) / rR
    sL, sR = np.sqrt(rL), np.sqrt(rR)
    u = (sL * uL + sR * uR) / (sL + sR)
    v = (sL * vL + sR * vR) / (sL + sR)
    w = (sL * wL + sR * wR) / (sL + sR)
    H = (sL * HL + sR * HR) / (sL + sR)
    q2 = u * u + v * v + w * w
    a = np.sqrt((g - 1) * (H - 0.5 * q2))
    d1, d2, d3, d4, d5 = rR - rL, rR * uR - rL * uL, rR * vR - rL * vL, rR * wR - rL * wL, ER - EL
    a3 = d3 - v * d1
    a4 = d4 - w * d1
    d5b = d5 - a3 * v - a4 * w
    a2 = (g - 1) / (a * a) * (d1 * (H - u * u) + u * d2 - d5b)
    a1 = (d1 * (u + a) - d2 - a * a2) / (2 * a)
    a5 = d1 - (a1 + a2)
    K1 = np.array([1, u - a, v, w, H - u * a])
    K2 = np.array([1, u, v, w, 0.5 * q2])
    K3 = np.array([0, 0, 1, 0, v])
    K4 = np.array([0, 0, 0, 1, w])
    K5 = np.array([1, u + a, v, w, H + u * a])
    FL = np.array([rL * uL, rL * uL * uL + pL, rL * uL * vL, rL * uL * wL, (EL + pL) * uL])
    FR = np.array([rR * uR, rR * uR * uR + pR, rR * uR * vR, rR * uR * wR, (ER + pR) * uR])
    diss = abs(u - a) * a1 * K1 + abs(u) * (a2 * K2 + a3 * K3 + a4 * K4) + abs(u + a) * a5 * K5
    return 0.5 * (FL + FR) - 0.5 * diss


def test_roe_mhd_with_zero_field_is_hd_roe(R):
    rng = np.random.default_rng(13)
    g = 1.4
    for _ in range(300):
        WL, WR = rand_state(rng, False), rand_state(rng, False)
        F, _, fb = R.riemann(ROE, g, WL, WR, 0.0)
        assert fb == 0
        ref = roe_hd_textbook(WL, WR, g)
        assert np.abs(F[:5] - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())
        assert abs(F[5]) <= 1e-15 and abs(F[6]) <= 1e-15   # B-components of the slow pair cancel to round-off


def test_roe_falls_back_to_hll_when_sound_speed_imaginary(R):
    # two cold streams colliding head-on: the Roe-averaged enthalpy is below the kinetic energy
    WL = np.array([1.0, 0.0, 30.0, 0, 1e-3, 0, 0])
    WR = np.array([1.0, 0.0, -30.0, 0, 1e-3, 0, 0])
    ok = R.roe_system(G, WL, WR, 0.0)[0]
    F, c, fb = R.riemann(ROE, G, WL, WR, 0.0)
    if not ok:
        assert fb == 1
        np.testing.assert_allclose(F, R.riemann(HLL, G, WL, WR, 0.0)[0])
    else:
        assert fb == 0


# ---- limiters (O3) -----------------------------------------------------------------------------
def test_limiters(R):
    rng = np.random.default_rng(14)
    for _ in range(500):
        a, b = rng.uniform(-2, 2, 2)
        for lim in (MINMOD, VANLEER):
            s = R.slope(lim, a, b)
            assert s == R.slope(lim, b, a)                       # symmetric
            if a * b <= 0:
                assert s == 0.0                                   # extremum
            else:
                assert min(a, b) - 1e-15 <= s <= 2 * max(abs(a), abs(b))
                assert abs(s) <= 2 * min(abs(a), abs(b)) + 1e-15  # TVD region: face states bounded by neighbours
                assert np.sign(s) == np.sign(a)
        assert R.slope(FLAT, a, b) == 0.0
        assert R.slope(MINMOD, a, a) == a and R.slope(VANLEER, a, a) == pytest.approx(a, rel=1e-15)
    assert R.slope(VANLEER, 1.0, 3.0) == pytest.approx(1.5)   # harmonic mean 2ab/(a+b)
    assert R.slope(MINMOD, 1.0, 3.0) == 1.0
    assert R.slope(MINMOD, -3.0, -1.0) == -1.0
    assert R.slope(VANLEER, 0.0, 1.0) == 0.0
