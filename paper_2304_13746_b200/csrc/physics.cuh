// physics.cuh — point-wise device functions of the idfx CUDA path (sm_100a, fp64).
//
// Reconstruction, ideal HD/MHD fluxes and the approximate Riemann solvers
// of PAPER.md:81: HLL, HLLC (HD), HLLD (MHD), Roe.  Formulas and readings: DESIGN.md O3-O8 / G2-G7.
// A 1D state along the sweep direction is W = (rho, u, v, w, p, By, Bz): u normal velocity, (By,Bz) the
// transverse field after cyclic permutation, Bn the normal (staggered) field.  Fluxes come back in the same
// local ordering F = (rho, m_n, m_t1, m_t2, E, B_t1, B_t2).
//
// This file shares nothing with oracle/: the solvers are written for registers (reciprocals reused,
// analytic Roe projections instead of 7x7 matrix loops, one-sided HLLD star states).
#pragma once
#include <cuda_runtime.h>

namespace idfx {

enum { SOLVER_HLL = 0, SOLVER_HLLC = 1, SOLVER_HLLD = 2, SOLVER_ROE = 3, SOLVER_RUSANOV = 4 };
enum { LIM_FLAT = 0, LIM_MINMOD = 1, LIM_VANLEER = 2, LIM_LIMO3 = 3, LIM_PPM = 4 };
enum { EMF_NONE = 0, EMF_ARITH = 1, EMF_UCT = 2, EMF_UCT0 = 3, EMF_UCT_HLL = 4, EMF_UCT_HLLD = 5 };

#define IDFX_DEV __device__ __forceinline__

// Reciprocal and square root without the IEEE slow paths: hardware seed (upper 32 bits, ~2^-20) refined by one
// third-order step in fp64 (the series in the residual e up to e^2, truncation ~ e^3 < 2^-57), result within ~1 ulp.  All operands on this path are normal, finite and non-negative
// where a root is taken; zero is handled explicitly.  -DIDFX_PRECISE_MATH restores the correctly rounded forms.
IDFX_DEV double rcp(double x) {
#ifdef IDFX_PRECISE_MATH
  return 1.0 / x;
#else
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y, 1.0);     // 1/x = y (1 + e + e^2 + O(e^3)), |e| <~ 2^-20
  return fma(y, fma(e, e, e), y);
#endif
}

// 1/sqrt(x) for x > 0
IDFX_DEV double rsqrt_pos(double x) {
#ifdef IDFX_PRECISE_MATH
  return 1.0 / sqrt(x);
#else
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double h = 0.5 * x;
  const double e = fma(-h * y, y, 0.5);  // (1 - x y^2)/2;  x^-1/2 = y (1 + e + 3/2 e^2 + O(e^3))
  return fma(y, fma(1.5 * e, e, e), y);
#endif
}

// sqrt(x) for x >= 0: x * rsqrt(max(x, tiny)); exact 0 stays 0 and no select is needed
IDFX_DEV double sqrt_nn(double x) {
#ifdef IDFX_PRECISE_MATH
  return sqrt(x);
#else
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(fmax(x, 1e-300)));
  const double s = x * y;
  const double e = fma(-0.5 * s, y, 0.5);
  return fma(s, fma(1.5 * e, e, e), s);
#endif
}

// sqrt(x) for x > 0
IDFX_DEV double sqrt_pos(double x) {
#ifdef IDFX_PRECISE_MATH
  return sqrt(x);
#else
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double s = x * y;                       // sqrt(x) = s (1 + e + 3/2 e^2 + O(e^3)), e = (1 - x y^2)/2
  const double e = fma(-0.5 * s, y, 0.5);
  return fma(s, fma(1.5 * e, e, e), s);
#endif
}

// O3 / G2: limited slope from the backward and forward differences.
template <int LIM>
IDFX_DEV double limited_slope(double dm, double dp) {
  if (LIM == LIM_FLAT) return 0.0;
  const double prod = dm * dp;
  if (LIM == LIM_VANLEER) {
    const bool mono = prod > 0.0;
    const double den = mono ? (dm + dp) : 1.0;  // keeps the division off its slow path at extrema
    const double s = (2.0 * prod) * rcp(den);
    return mono ? s : 0.0;
  } else {
    const double s = (fabs(dm) < fabs(dp)) ? dm : dp;
    return (prod > 0.0) ? s : 0.0;
  }
}

// LimO3 (Cada & Torrilhon 2009; reading G18): the increment phi(theta) * dplus with
// theta = dminus/dplus, limited branch, written without the division: with s = sign(dplus), a = |dplus|, b = s dminus
// and P = (2a + b)/3,  phi dplus = s max(0, min(P, max(-b/2, min(2b, P, 1.6 a)))).
IDFX_DEV double limo3_limited(double dminus, double dplus) {
  const double a = fabs(dplus), b = dplus < 0.0 ? -dminus : dminus;
  const double P = (2.0 * a + b) * (1.0 / 3.0);
  const double l = fmax(0.0, fmin(P, fmax(-0.5 * b, fmin(fmin(2.0 * b, P), 1.6 * a))));
  return dplus < 0.0 ? -l : l;
}

// S2: values of cell i's reconstruction at its lower and upper faces; dm = q_i - q_{i-1}, dp = q_{i+1} - q_i.
// LimO3: the smoothness measure eta = (dm^2 + dp^2)/dx^2 is shared by both faces; where eta < 1 (most cells of a resolved
// flow) the unlimited third-order weights (2 + theta)/3 are used and the limiter is never evaluated; a linear blend
// within 1e-12 of eta = 1 (a true division only there).
template <int LIM>
IDFX_DEV void face_values(double q, double dm, double dp, double dx2, double& lower, double& upper) {
  if (LIM == LIM_LIMO3) {
    const double eps = 1e-12;
    const double num = dm * dm + dp * dp;
    double iu = (2.0 * dp + dm) * (1.0 / 3.0);  // upper face: phi(theta) dp
    double il = (2.0 * dm + dp) * (1.0 / 3.0);  // lower face: phi(1/theta) dm
    if (num > (1.0 - eps) * dx2) {
      const double lu = limo3_limited(dm, dp), ll = limo3_limited(dp, dm);
      if (num >= (1.0 + eps) * dx2) {
        iu = lu;
        il = ll;
      } else {
        const double x = (num / dx2 - 1.0) / eps;
        iu = 0.5 * ((1.0 - x) * iu + (1.0 + x) * lu);
        il = 0.5 * ((1.0 - x) * il + (1.0 + x) * ll);
      }
    }
    upper = q + 0.5 * iu;
    lower = q - 0.5 * il;
  } else if (LIM == LIM_VANLEER) {
    // half the harmonic-mean slope, dm dp / (dm + dp): the same bits as 0.5 * limited_slope (powers of two are exact),
    // one multiplication less; at an extremum the quotient (possibly 0/0) is discarded by the select
    const double prod = dm * dp;
#ifdef IDFX_PRECISE_MATH
    const double h = prod > 0.0 ? prod / (dm + dp) : 0.0;
#else
    const double hq = prod * rcp(dm + dp);
    const double h = prod > 0.0 ? hq : 0.0;
#endif
    lower = q - h;
    upper = q + h;
  } else {
    const double s = limited_slope<LIM>(dm, dp);
    lower = q - 0.5 * s;
    upper = q + 0.5 * s;
  }
}

// PPM with the extremum-preserving limiter (Colella & Woodward 1984, Colella & Sekora 2008; DESIGN.md reading
// G22), uniform grid.  Interface value between cells 0 and 1 from cells -1 .. 2: fourth-order average, and where that is
// not between its two cells the second-difference-limited replacement.
IDFX_DEV double ppm_edge(double am1, double a0, double ap1, double ap2) {
  const double mid = a0 + ap1;
  double f = (7.0 / 12.0) * mid - (1.0 / 12.0) * (am1 + ap2);
  if ((f - a0) * (ap1 - f) < 0.0) {
    const double d2 = 3.0 * (mid - 2.0 * f), d2l = (am1 + ap1) - 2.0 * a0, d2r = (a0 + ap2) - 2.0 * ap1;
    const bool same = d2 * d2l > 0.0 && d2 * d2r > 0.0;
    const double mag = fmin(fabs(d2), 1.25 * fmin(fabs(d2l), fabs(d2r)));
    f = 0.5 * mid - (same ? copysign(mag, d2) : 0.0) * (1.0 / 6.0);
  }
  return f;
}

// Limited parabola of the cell with value a0 and raw edge values em (lower), ep (upper); q[0..4] = cells -2 .. +2.
// At an extremum both edge deviations shrink by D2lim/D2f; elsewhere an edge further than twice the other from a0 is
// pulled in (one side at a time).
IDFX_DEV void ppm_limit(const double q[5], double em, double ep, double& lower, double& upper) {
  const double a0 = q[2];
  const double dm = a0 - em, dp = ep - a0;
  if (dm * dp <= 0.0 || (q[3] - a0) * (a0 - q[1]) <= 0.0) {
    const double d2f = 6.0 * ((ep + em) - 2.0 * a0);
    const double d2l = (q[0] + q[2]) - 2.0 * q[1], d2c = (q[1] + q[3]) - 2.0 * q[2], d2r = (q[2] + q[4]) - 2.0 * q[3];
    const bool same = d2f * d2l > 0.0 && d2f * d2c > 0.0 && d2f * d2r > 0.0;
    const double mag = fmin(fabs(d2f), 1.25 * fmin(fabs(d2c), fmin(fabs(d2l), fabs(d2r))));
    const double ratio = same ? mag / fabs(d2f) : 0.0;   // d2f != 0 whenever same
    lower = a0 - dm * ratio;
    upper = a0 + dp * ratio;
  } else {
    upper = fabs(dp) >= 2.0 * fabs(dm) ? a0 + 2.0 * dm : ep;
    lower = fabs(dm) >= 2.0 * fabs(dp) ? a0 - 2.0 * dp : em;
  }
}

// Conserved vector, physical flux and total pressure of one side.
template <bool MHD>
IDFX_DEV void side_cons_flux(const double W[7], double Bn, double igm1, double U[7], double F[7], double& pT) {
  const double rho = W[0], u = W[1], v = W[2], w = W[3], p = W[4];
  const double mu = rho * u;
  const double ke = 0.5 * rho * (u * u + v * v + w * w);
  U[0] = rho;
  U[1] = mu;
  U[2] = rho * v;
  U[3] = rho * w;
  if (MHD) {
    const double By = W[5], Bz = W[6];
    const double pb = 0.5 * (Bn * Bn + By * By + Bz * Bz);
    const double vB = u * Bn + v * By + w * Bz;
    pT = p + pb;
    U[4] = p * igm1 + ke + pb;
    U[5] = By;
    U[6] = Bz;
    F[0] = mu;
    F[1] = mu * u + pT - Bn * Bn;
    F[2] = mu * v - Bn * By;
    F[3] = mu * w - Bn * Bz;
    F[4] = (U[4] + pT) * u - Bn * vB;
    F[5] = u * By - v * Bn;
    F[6] = u * Bz - w * Bn;
  } else {
    pT = p;
    U[4] = p * igm1 + ke;
    U[5] = U[6] = 0.0;
    F[0] = mu;
    F[1] = mu * u + p;
    F[2] = mu * v;
    F[3] = mu * w;
    F[4] = (U[4] + p) * u;
    F[5] = F[6] = 0.0;
  }
}

// O4: sound speed (HD) or fast magnetosonic speed along the sweep direction (MHD).
template <bool MHD>
IDFX_DEV double signal_speed(const double W[7], double Bn, double g) {
  const double ir = rcp(W[0]);
  const double a2 = g * W[4] * ir;
  if (!MHD) return sqrt_pos(a2);
  // (a2 + b2)^2 - 4 a2 bn2 written as (a2 - b2)^2 + 4 a2 bt2: a sum of non-negative terms, no clamp needed
  const double bt2 = (W[5] * W[5] + W[6] * W[6]) * ir;
  const double b2 = Bn * Bn * ir + bt2;
  const double s = a2 + b2, d = a2 - b2;
  const double disc = fma(d, d, 4.0 * a2 * bt2);
  return sqrt_pos(0.5 * (s + sqrt_nn(disc)));
}

// O4 / G5: Davis estimate of the outer speeds; c_face = max(|S_L|,|S_R|) for every solver.
template <bool MHD>
IDFX_DEV void outer_speeds(const double WL[7], const double WR[7], double Bn, double g, double& SL, double& SR) {
  const double cL = signal_speed<MHD>(WL, Bn, g), cR = signal_speed<MHD>(WR, Bn, g);
  SL = fmin(WL[1] - cL, WR[1] - cR);
  SR = fmax(WL[1] + cL, WR[1] + cR);
}

// O5: HLL average inside the fan (caller handles S_L >= 0 and S_R <= 0).
template <int NV>
IDFX_DEV void hll_inner(const double UL[7], const double UR[7], const double FL[7], const double FR[7], double SL,
                        double SR, double F[7]) {
  const double inv = rcp(SR - SL);
  const double ss = SL * SR;
#pragma unroll
  for (int n = 0; n < NV; ++n) F[n] = (SR * FL[n] - SL * FR[n] + ss * (UR[n] - UL[n])) * inv;
}

// O6: HLLC (hydrodynamics).  Only the star state on the side of the contact is built.
IDFX_DEV void hllc_inner(const double WL[7], const double WR[7], const double UL[7], const double UR[7],
                         const double FL[7], const double FR[7], double SL, double SR, double F[7]) {
  const double qL = WL[0] * (SL - WL[1]);  // rho_L (S_L - u_L)
  const double qR = WR[0] * (SR - WR[1]);
  const double SS = (WR[4] - WL[4] + qL * WL[1] - qR * WR[1]) * rcp(qL - qR);
  const bool left = SS >= 0.0;
  const double SK = left ? SL : SR;
  const double qK = left ? qL : qR;
  const double rK = left ? WL[0] : WR[0], uK = left ? WL[1] : WR[1], vK = left ? WL[2] : WR[2];
  const double wK = left ? WL[3] : WR[3], pK = left ? WL[4] : WR[4], EK = left ? UL[4] : UR[4];
  const double fac = qK * rcp(SK - SS);
  double Us[5];
  Us[0] = fac;
  Us[1] = fac * SS;
  Us[2] = fac * vK;
  Us[3] = fac * wK;
  Us[4] = fac * (EK * rcp(rK) + (SS - uK) * (SS + pK * rcp(qK)));
#pragma unroll
  for (int n = 0; n < 5; ++n) {
    const double Fk = left ? FL[n] : FR[n];
    const double Uk = left ? UL[n] : UR[n];
    F[n] = Fk + SK * (Us[n] - Uk);
  }
}

// O8 / G7: Roe solver with the exact Roe averages of the shifted equation of state, no entropy fix.
// Returns false when a~^2 <= 0 (caller falls back to HLL).  Projections are written out analytically:
// dW = Minv dU, alpha_k = l_k . dW, primitive sum s = sum |lambda_k| alpha_k r_k, flux jump = M s.
template <bool MHD>
IDFX_DEV bool roe_inner(const double WL[7], const double WR[7], double Bn, const double UL[7], const double UR[7],
                        const double FL[7], const double FR[7], double pTL, double pTR, double g, double F[7]) {
  const double sL = sqrt_pos(WL[0]), sR = sqrt_pos(WR[0]);
  const double isum = rcp(sL + sR);
  const double rb = sL * sR;
  const double irb = rcp(rb);
  const double ub = (sL * WL[1] + sR * WR[1]) * isum;
  const double vb = (sL * WL[2] + sR * WR[2]) * isum;
  const double wb = (sL * WL[3] + sR * WR[3]) * isum;
  const double HL = (UL[4] + pTL) * rcp(WL[0]), HR = (UR[4] + pTR) * rcp(WR[0]);
  const double Hb = (sL * HL + sR * HR) * isum;
  const double v2h = 0.5 * (ub * ub + vb * vb + wb * wb);
  const double gm1 = g - 1.0, igm1 = rcp(gm1);
  double Byb = 0.0, Bzb = 0.0, Xp = 0.0, bt2 = 0.0, bn2 = 0.0;
  const double dBy = UR[5] - UL[5], dBz = UR[6] - UL[6];
  if (MHD) {
    Byb = (sR * WL[5] + sL * WR[5]) * isum;
    Bzb = (sR * WL[6] + sL * WR[6]) * isum;
    Xp = (g - 2.0) * (dBy * dBy + dBz * dBz) * 0.5 * isum * isum;
    bt2 = (Byb * Byb + Bzb * Bzb) * irb;
    bn2 = Bn * Bn * irb;
  }
  const double a2 = gm1 * (Hb - v2h - (bn2 + bt2)) - Xp;
  if (!(a2 > 0.0)) return false;

  // jumps in the linearised primitive variables
  const double dr = UR[0] - UL[0];
  const double dmx = UR[1] - UL[1], dmy = UR[2] - UL[2], dmz = UR[3] - UL[3], dE = UR[4] - UL[4];
  const double du = (dmx - ub * dr) * irb;
  const double dv = (dmy - vb * dr) * irb;
  const double dw = (dmz - wb * dr) * irb;
  const double dp = gm1 * (v2h * dr - ub * dmx - vb * dmy - wb * dmz + dE - Byb * dBy - Bzb * dBz) - Xp * dr;

  double s0, s1, s2, s3, s4, s5 = 0.0, s6 = 0.0;
  if (!MHD) {
    const double a = sqrt_pos(a2);
    const double ia2 = rcp(a2);
    // acoustic waves u -+ a: r = (rb, -+a, 0, 0, rb a2), l = (0, -+a, 0, 0, 1/rb)/(2 a2)
    const double am = (-a * du + dp * irb) * 0.5 * ia2;
    const double ap = (a * du + dp * irb) * 0.5 * ia2;
    const double lm = fabs(ub - a) * am, lp = fabs(ub + a) * ap, l0 = fabs(ub);
    const double a0 = dr - dp * ia2;
    s0 = rb * (lm + lp) + l0 * a0;
    s1 = a * (lp - lm);
    s2 = l0 * dv;
    s3 = l0 * dw;
    s4 = rb * a2 * (lm + lp);
  } else {
    const double a = sqrt_pos(a2);
    const double ia2 = rcp(a2);
    const double sum = a2 + bn2 + bt2;
    const double disc = sqrt_nn(fmax(sum * sum - 4.0 * a2 * bn2, 0.0));
    const double Cf2 = 0.5 * (sum + disc);
    const double Cs2 = a2 * bn2 * rcp(Cf2);
    const double Cf = sqrt_nn(Cf2), Cs = sqrt_nn(Cs2), CA = sqrt_nn(bn2);
    double af = 1.0, as = 0.0;
    const double den = Cf2 - Cs2;
    if (den > 0.0) {
      const double iden = rcp(den);
      af = sqrt_nn(fmin(1.0, fmax(0.0, (a2 - Cs2) * iden)));
      as = sqrt_nn(fmin(1.0, fmax(0.0, (Cf2 - a2) * iden)));
    }
    const double Bt2 = Byb * Byb + Bzb * Bzb;
    double by = 0.70710678118654752440, bz = 0.70710678118654752440;
    if (Bt2 > 1e-300) {
      const double iBt = rsqrt_pos(Bt2);
      by = Byb * iBt;
      bz = Bzb * iBt;
    }
    const double S = (Bn >= 0.0) ? 1.0 : -1.0;
    const double isr = rsqrt_pos(rb), sr = rb * isr;
    const double Cff = Cf * af, Css = Cs * as, Qf = Cff * S, Qs = Css * S;
    const double Af = a * af * sr, As = a * as * sr;
    const double i2a2 = 0.5 * ia2;

    const double dvt = by * dv + bz * dw;        // beta . dv_t
    const double dBt = (by * dBy + bz * dBz);    // beta . dB_t
    const double dvx = -bz * dv + by * dw;       // (beta_perp) . dv_t
    const double dBx = (-bz * dBy + by * dBz);   // (beta_perp) . dB_t
    // wave strengths
    const double tf = (af * dp + As * dBt) * irb;
    const double afm = (-Cff * du + Qs * dvt + tf) * i2a2;
    const double afp = (Cff * du - Qs * dvt + tf) * i2a2;
    const double ts = (as * dp - Af * dBt) * irb;
    const double asm_ = (-Css * du - Qf * dvt + ts) * i2a2;
    const double asp = (Css * du + Qf * dvt + ts) * i2a2;
    const double aAm = 0.5 * (dvx + S * dBx * isr);     // l_A- = (0,0,-bz,+by,0,-S bz/sr, S by/sr)/2
    const double aAp = 0.5 * (-dvx + S * dBx * isr);
    const double a0 = dr - dp * ia2;
    // |lambda| alpha
    const double Lfm = fabs(ub - Cf) * afm, Lfp = fabs(ub + Cf) * afp;
    const double Lsm = fabs(ub - Cs) * asm_, Lsp = fabs(ub + Cs) * asp;
    const double LAm = fabs(ub - CA) * aAm, LAp = fabs(ub + CA) * aAp;
    const double L0 = fabs(ub) * a0;
    // primitive-space sum; components along beta (t) and beta_perp (x) for v_t and B_t
    const double fsum = Lfm + Lfp, ssum = Lsm + Lsp;
    s0 = rb * (af * fsum + as * ssum) + L0;
    s1 = Cff * (Lfp - Lfm) + Css * (Lsp - Lsm);
    const double vt = Qs * (Lfm - Lfp) + Qf * (Lsp - Lsm);   // along beta
    const double vx = LAm - LAp;                             // along beta_perp: r_A-+ = (.., -+bz, +-by, ..)
    s2 = by * vt - bz * vx;
    s3 = bz * vt + by * vx;
    s4 = rb * a2 * (af * fsum + as * ssum);
    const double Bt_ = As * fsum - Af * ssum;                // along beta
    const double Bx_ = S * sr * (LAm + LAp);                 // along beta_perp
    s5 = by * Bt_ - bz * Bx_;
    s6 = bz * Bt_ + by * Bx_;
  }
  // conserved-variable jump M s, F = (F_L + F_R)/2 - (M s)/2
  const double j0 = s0;
  const double j1 = ub * s0 + rb * s1;
  const double j2 = vb * s0 + rb * s2;
  const double j3 = wb * s0 + rb * s3;
  const double j4 = (v2h + Xp * igm1) * s0 + rb * (ub * s1 + vb * s2 + wb * s3) + s4 * igm1 + Byb * s5 + Bzb * s6;
  F[0] = 0.5 * (FL[0] + FR[0] - j0);
  F[1] = 0.5 * (FL[1] + FR[1] - j1);
  F[2] = 0.5 * (FL[2] + FR[2] - j2);
  F[3] = 0.5 * (FL[3] + FR[3] - j3);
  F[4] = 0.5 * (FL[4] + FR[4] - j4);
  F[5] = MHD ? 0.5 * (FL[5] + FR[5] - s5) : 0.0;
  F[6] = MHD ? 0.5 * (FL[6] + FR[6] - s6) : 0.0;
  return true;
}

// O7 / G5 / G6: the whole HLLD problem written one-sided and branch-free.  Total pressures, outer speeds, S_M, p_T*
// and the starred transverse components need both sides; conserved vector, physical flux, E*, E** and the flux
// combination are evaluated only for the side K the selection of O7 picks (K = L when S_L >= 0, R when S_R <= 0).
// x with its sign bit flipped where the mask (0 or 0x80000000) says so: the same bits as a multiplication by -1 or +1,
// one integer instruction instead of one on the fp64 pipe
IDFX_DEV double flip_sign(double x, int mask) { return __hiloint2double(__double2hiint(x) ^ mask, __double2loint(x)); }

IDFX_DEV double hlld_onesided(const double WL[7], const double WR[7], double Bn, double g, double F[7]) {
  const double Bn2 = Bn * Bn;
  const double bt2L = WL[5] * WL[5] + WL[6] * WL[6], bt2R = WR[5] * WR[5] + WR[6] * WR[6];
  const double b2L = Bn2 + bt2L, b2R = Bn2 + bt2R;
  const double pbL = 0.5 * b2L, pbR = 0.5 * b2R;
  const double pTL = WL[4] + pbL, pTR = WR[4] + pbR;
  const double uL = WL[1], uR = WR[1];
  double cL, cR;
  {  // fast speed; (a2 + b2)^2 - 4 a2 bn2 = (a2 - b2)^2 + 4 a2 bt2 is a sum of non-negative terms (no clamp)
    const double ir = rcp(WL[0]);
    const double a2 = g * WL[4] * ir, sm = fma(b2L, ir, a2), dm = fma(-b2L, ir, a2);
    cL = sqrt_pos(0.5 * (sm + sqrt_nn(fma(dm, dm, 4.0 * a2 * (bt2L * ir)))));
  }
  {
    const double ir = rcp(WR[0]);
    const double a2 = g * WR[4] * ir, sm = fma(b2R, ir, a2), dm = fma(-b2R, ir, a2);
    cR = sqrt_pos(0.5 * (sm + sqrt_nn(fma(dm, dm, 4.0 * a2 * (bt2R * ir)))));
  }
  const double SL = fmin(uL - cL, uR - cR), SR = fmax(uL + cL, uR + cR);
  const double cface = fmax(fabs(SL), fabs(SR));

  const double sL = SL - uL, sR = SR - uR;
  const double qL = WL[0] * sL, qR = WR[0] * sR;  // rho_K (S_K - u_K)
  const double iD = rcp(qR - qL);
  const double SM = (qR * uR - qL * uL - pTR + pTL) * iD;
  const double pTs = (qR * pTL - qL * pTR + qL * qR * (uR - uL)) * iD;
  const double iL = rcp(SL - SM), iR = rcp(SR - SM);
  const double rsL = qL * iL, rsR = qR * iR;  // rho*_K
  double vsL, wsL, BysL, BzsL, vsR, wsR, BysR, BzsR;
  {
    const double d = qL * (SL - SM) - Bn2;
    const bool deg = fabs(d) < 1e-12 * qL * sL;
    const double id = rcp(d);  // d = 0 gives a non-finite value that the selects below discard
    const double f = deg ? 0.0 : Bn * (SM - uL) * id;
    const double h = deg ? 1.0 : (qL * sL - Bn2) * id;
    vsL = WL[2] - WL[5] * f;
    wsL = WL[3] - WL[6] * f;
    BysL = WL[5] * h;
    BzsL = WL[6] * h;
  }
  {
    const double d = qR * (SR - SM) - Bn2;
    const bool deg = fabs(d) < 1e-12 * qR * sR;
    const double id = rcp(d);  // d = 0 gives a non-finite value that the selects below discard
    const double f = deg ? 0.0 : Bn * (SM - uR) * id;
    const double h = deg ? 1.0 : (qR * sR - Bn2) * id;
    vsR = WR[2] - WR[5] * f;
    wsR = WR[3] - WR[6] * f;
    BysR = WR[5] * h;
    BzsR = WR[6] * h;
  }
  const double ysL = rsqrt_pos(fabs(rsL)), ysR = rsqrt_pos(fabs(rsR));  // 1/sqrt(rho*_K); |.| only guards unused lanes
  const double sqL = fabs(rsL) * ysL, sqR = fabs(rsR) * ysR;
  const double aBn = fabs(Bn);
  const double SsL = SM - aBn * ysL, SsR = SM + aBn * ysR;

  // selection in the order of O7
  const bool pureL = SL >= 0.0, pureR = !pureL && SR <= 0.0;
  const bool starL = SsL >= 0.0, starR = !starL && SsR <= 0.0;
  const bool pure = pureL || pureR;
  const bool left = pureL || (!pureR && (starL || (!starR && SM >= 0.0)));
  const bool dstar = !pure && !starL && !starR;

  // side K: conserved vector and physical flux
  const double rK = left ? WL[0] : WR[0], uK = left ? uL : uR, vK = left ? WL[2] : WR[2];
  const double wK = left ? WL[3] : WR[3], pK = left ? WL[4] : WR[4];
  const double ByK = left ? WL[5] : WR[5], BzK = left ? WL[6] : WR[6];
  const double pbK = left ? pbL : pbR, pTK = left ? pTL : pTR;
  const double muK = rK * uK;
  const double EK = pK * rcp(g - 1.0) + 0.5 * rK * (uK * uK + vK * vK + wK * wK) + pbK;
  const double vBK = uK * Bn + vK * ByK + wK * BzK;
  double UK[7], FK[7];
  UK[0] = rK; UK[1] = muK; UK[2] = rK * vK; UK[3] = rK * wK; UK[4] = EK; UK[5] = ByK; UK[6] = BzK;
  FK[0] = muK;
  FK[1] = muK * uK + pTK - Bn2;
  FK[2] = muK * vK - Bn * ByK;
  FK[3] = muK * wK - Bn * BzK;
  FK[4] = (EK + pTK) * uK - Bn * vBK;
  FK[5] = uK * ByK - vK * Bn;
  FK[6] = uK * BzK - wK * Bn;

  // star and double-star states of side K
  const double SK = left ? SL : SR, sK = left ? sL : sR, iK = left ? iL : iR;
  const double rsK = left ? rsL : rsR, sqK = left ? sqL : sqR, SsK = left ? SsL : SsR;
  const double vsK = left ? vsL : vsR, wsK = left ? wsL : wsR;
  const double BysK = left ? BysL : BysR, BzsK = left ? BzsL : BzsR;
  const double vBsK = SM * Bn + vsK * BysK + wsK * BzsK;
  const double EsK = (sK * EK - pTK * uK + pTs * SM + Bn * (vBK - vBsK)) * iK;
  const int sgn = (Bn >= 0.0) ? 0 : (int)0x80000000;  // sign(B_n) as a sign-bit mask (G7: sign(0) = +1)
  const double inv = rcp(sqL + sqR);
  const double sqq = sqL * sqR;
  const double vss = (sqL * vsL + sqR * vsR + flip_sign(BysR - BysL, sgn)) * inv;
  const double wss = (sqL * wsL + sqR * wsR + flip_sign(BzsR - BzsL, sgn)) * inv;
  const double Byss = (sqL * BysR + sqR * BysL + flip_sign(sqq * (vsR - vsL), sgn)) * inv;
  const double Bzss = (sqL * BzsR + sqR * BzsL + flip_sign(sqq * (wsR - wsL), sgn)) * inv;
  const double vBss = SM * Bn + vss * Byss + wss * Bzss;
  // E**_L = E*_L - sqrt(rho*_L)(vB*_L - vB**) sgn ;  E**_R = E*_R + sqrt(rho*_R)(vB*_R - vB**) sgn
  const int sside = left ? sgn ^ (int)0x80000000 : sgn;
  const double EssK = EsK + flip_sign(sqK * (vBsK - vBss), sside);
  double Us[7], Uss[7];
  Us[0] = rsK; Us[1] = rsK * SM; Us[2] = rsK * vsK; Us[3] = rsK * wsK; Us[4] = EsK; Us[5] = BysK; Us[6] = BzsK;
  Uss[0] = rsK; Uss[1] = Us[1]; Uss[2] = rsK * vss; Uss[3] = rsK * wss; Uss[4] = EssK; Uss[5] = Byss; Uss[6] = Bzss;
  // star:        F = F_K + S_K (U* - U_K)
  // double star: F = F_K + S*_K U** - (S*_K - S_K) U* - S_K U_K
  const double c1 = dstar ? SK - SsK : SK;
  const double c2 = dstar ? SsK : 0.0;
#pragma unroll
  for (int n = 0; n < 7; ++n) {
    // density and normal momentum: U** = U* and c1 + c2 = S_K
    const double f = n < 2 ? FK[n] + SK * (Us[n] - UK[n]) : FK[n] + c1 * Us[n] + c2 * Uss[n] - SK * UK[n];
    F[n] = pure ? FK[n] : f;
  }
  return cface;
}

// What the 2D-HLLD edge EMF needs of a face (reading G24): how the HLLD flux of a transverse field
// component responds to the two face values of that component and to the normal field,
//     F_n[B_t] = (u_L dirL + kL) B_t,L + (u_R (1 - dirL) - kR) B_t,R - vt B_n .
// dirL says whether the face lies left of the contact; (kL, kR) is the response that is not plain upwind transport; vt slides
// from v_L to v_R across the double-star fan.  One formula for all regions: a side's outer shock contributes
// eK = S_K (h_K - 1) once the face is inside the fan, and inside the double-star fan both sides add -z h_K + m g_K with
// z = +-S*_K s_K / (s_L + s_R) (+ left of the contact, - right) and m = +-z s_O sgn(B_n), s_O the root density of the other side.
IDFX_DEV void hlld_uct_face(const double WL[7], const double WR[7], double Bn, double g, double& dirL, double& kL, double& kR,
                            double& vt1, double& vt2) {
  double SL, SR;
  outer_speeds<true>(WL, WR, Bn, g, SL, SR);
  const double Bn2 = Bn * Bn;
  const double pTL = WL[4] + 0.5 * (Bn2 + WL[5] * WL[5] + WL[6] * WL[6]);
  const double pTR = WR[4] + 0.5 * (Bn2 + WR[5] * WR[5] + WR[6] * WR[6]);
  const double mL = WL[0] * (SL - WL[1]), mR = WR[0] * (SR - WR[1]);  // mass fluxes through the outer waves
  const double SM = (mR * WR[1] - mL * WL[1] - pTR + pTL) / (mR - mL);
  // per side: compression of the transverse field h, coupling g between B_t and v_t, root of the star density
  double hK[2], gK[2], sK[2];
  {
    const double m[2] = {mL, mR}, S[2] = {SL, SR}, u[2] = {WL[1], WR[1]};
#pragma unroll
    for (int K = 0; K < 2; ++K) {
      const double den = m[K] * (S[K] - SM) - Bn2;
      const bool flat = fabs(den) < 1e-12 * m[K] * (S[K] - u[K]);  // G6
      hK[K] = flat ? 1.0 : (m[K] * (S[K] - u[K]) - Bn2) / den;
      gK[K] = flat ? 0.0 : Bn * (SM - u[K]) / den;
      sK[K] = sqrt(m[K] / (S[K] - SM));
    }
  }
  const double aB = fabs(Bn);
  const double SsL = SM - aB / sK[0], SsR = SM + aB / sK[1];
  // where the face lies (the order of O7)
  const bool outerL = SL >= 0.0, outerR = !outerL && SR <= 0.0;
  const bool starL = !outerL && !outerR && SsL >= 0.0, starR = !outerL && !outerR && !starL && SsR <= 0.0;
  const bool inner = !outerL && !outerR && !starL && !starR;
  const bool left = outerL || starL || (inner && SM >= 0.0);
  dirL = left ? 1.0 : 0.0;
  const bool fan = !outerL && !outerR;
  const double eL = (fan && left) ? SL * (hK[0] - 1.0) : 0.0;
  const double eR = (fan && !left) ? SR * (hK[1] - 1.0) : 0.0;
  const double ssum = sK[0] + sK[1];
  const double z = inner ? (left ? SsL * sK[0] : -SsR * sK[1]) / ssum : 0.0;
  const double m = (left ? z * sK[1] : -z * sK[0]) * (Bn >= 0.0 ? 1.0 : -1.0);
  kL = eL - z * hK[0] + m * gK[0];
  kR = -eR - z * hK[1] + m * gK[1];
  // share of v_R in the effective transverse velocity
  const double om = inner ? sK[1] * (1.0 - SM * sK[0] / aB) / ssum : (left ? 0.0 : 1.0);
  vt1 = WL[2] + om * (WR[2] - WL[2]);
  vt2 = WL[3] + om * (WR[3] - WL[3]);
}

// One Riemann problem.  Returns the flux in F and c_face = max(|S_L|,|S_R|).
template <int SOLVER, bool MHD>
IDFX_DEV double riemann(const double WL[7], const double WR[7], double Bn, double g, double F[7]) {
  if (SOLVER == SOLVER_HLLD) return hlld_onesided(WL, WR, Bn, g, F);
  const double igm1 = rcp(g - 1.0);
  double UL[7], UR[7], FL[7], FR[7], pTL, pTR, SL, SR;
  side_cons_flux<MHD>(WL, Bn, igm1, UL, FL, pTL);
  side_cons_flux<MHD>(WR, Bn, igm1, UR, FR, pTR);
  outer_speeds<MHD>(WL, WR, Bn, g, SL, SR);
  const double cface = fmax(fabs(SL), fabs(SR));
  constexpr int NV = MHD ? 7 : 5;
  if (SOLVER == SOLVER_RUSANOV) {  // local Lax-Friedrichs: central flux minus c_face/2 times the jump
    const double hc = 0.5 * cface;
#pragma unroll
    for (int n = 0; n < 7; ++n) F[n] = n < NV ? 0.5 * (FL[n] + FR[n]) - hc * (UR[n] - UL[n]) : 0.0;
    return cface;
  }
  if (SOLVER == SOLVER_ROE) {
    if (!roe_inner<MHD>(WL, WR, Bn, UL, UR, FL, FR, pTL, pTR, g, F)) {
      if (SL >= 0.0) {
#pragma unroll
        for (int n = 0; n < 7; ++n) F[n] = FL[n];
      } else if (SR <= 0.0) {
#pragma unroll
        for (int n = 0; n < 7; ++n) F[n] = FR[n];
      } else {
        F[5] = F[6] = 0.0;
        hll_inner<NV>(UL, UR, FL, FR, SL, SR, F);
      }
    }
    return cface;
  }
  if (SL >= 0.0) {
#pragma unroll
    for (int n = 0; n < 7; ++n) F[n] = FL[n];
  } else if (SR <= 0.0) {
#pragma unroll
    for (int n = 0; n < 7; ++n) F[n] = FR[n];
  } else {
    if (!MHD) F[5] = F[6] = 0.0;
    if (SOLVER == SOLVER_HLL) hll_inner<NV>(UL, UR, FL, FR, SL, SR, F);
    if (SOLVER == SOLVER_HLLC) hllc_inner(WL, WR, UL, UR, FL, FR, SL, SR, F);
  }
  return cface;
}

}  // namespace idfx
