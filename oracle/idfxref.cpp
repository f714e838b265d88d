// idfxref — the ORACLE for the idfx B200 library.
//
// TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may build, load or call anything in this directory.
// The CUDA path (paper_2304_13746_b200/) shares no source, header, table or helper with it.
//
// What it is: a plain, slow, single-threaded fp64 CPU implementation of one explicit cycle (RK2 by default;
// Euler and RK3 of Tab. 1 as options) of the
// Godunov finite-volume scheme of IDEFIX (Lesur et al., arXiv 2304.13746) for
// compressible HD and ideal MHD on a uniform periodic 3D Cartesian grid, written step by step in the
// paper's order.  Citations "PAPER.md:<line>" refer to /root/reference/PAPER.md; "O<n>" / "G<n>" refer
// to SURVEY.md §8(c) (the written-out formulas and the readings of points the paper leaves open;
// they are restated in DESIGN.md).
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): flux consistency F(U,U)=F(U); HLL/HLLC/HLLD
// fan-integral identity; HLLC p* continuity; isolated contact and rotational discontinuities; Roe
// L·R=I, A·r=λr against a finite-difference Jacobian, Σλαr = F_R−F_L; MHD-Roe(B=0) = 5-wave HD Roe;
// Rusanov = HLL with symmetric speeds; limiter properties; exact Sod solution along x, y, z; direction symmetry; uniform state; conservation;
// div B; Eᶜ plane-parallel identity AND its upwind-side rule (test_oracle_emf_upwind.py: domain of dependence of a one-edge
// potential bump in supersonic flow for every sign quadrant and edge family, donor-cell closed form, field-loop advection,
// zero mass flux => mean = E^0); RK2 amplification factor; closed-form dt; 2nd-order convergence of
// linear fast/Alfvén waves.  Options (tests/test_oracle_options.py, test_oracle_emf_hlld2d.py): Euler/RK2/RK3 amplification
// polynomials and temporal order; LimO3 exact for parabolas, bounded at jumps, 3rd-order linear-wave convergence with RK3;
// vector-potential CT equal to face CT up to rounding with div B that does not accumulate; advance_to lands on t_end; 2D-HLL and
// 2D-HLLD EMFs: plane-parallel limit = the 1D HLL / HLLD flux EMF along x, y, z, and for HLLD the coefficient decomposition
// reproduces the pinned HLLD flux in all six fan regions; outflow boundaries with a magnetic field: Brio-Wu tube stays 1D and
// equals the periodic double tube away from the ends, fixed point, div B on interior cells.
// PARITY UNPINNED (the paper fixes none of these CHOICES and prints no number that depends on them, see
// DESIGN.md "Readings"; each has pins that a wrong implementation of the stated reading fails): the limiter flavour (G2),
// the Davis wave-speed estimate (G5), the HLLD degeneracy threshold (G6), the Roe fallback/degenerate-eigenvector conventions
// (G7), the face→cell mapping of c_max in dt (G8), un-lagged dt (G9), the reference state of E^c (G10: -v x Bc of the stage
// input), the LimO3 constants (1.6, r = 1, eps = 1e-12; G18: PAPER.md:79 only names the scheme of Cada & Torrilhon 2009), the
// composition of the 2D-HLL and 2D-HLLD EMFs beyond their plane-parallel limit (G21, G24: PAPER.md:109 only names Mignone &
// Del Zanna 2021), the form of the PPM limiter (G22: PAPER.md:79 only names Colella & Woodward 1984 and Colella & Sekora 2008;
// pinned here by what the construction must do: exact for cubics, smooth extrema kept, steps monotone, fourth-order face
// values), and the zero-gradient continuation of the staggered field at outflow boundaries (G23).
//
// Build: g++ -O2 -ffp-contract=off -std=c++17 -shared -fPIC idfxref.cpp -o libidfxref.so
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstring>
#include <vector>

#define IDFXREF_API extern "C" __attribute__((visibility("default")))

namespace {

constexpr int NG = 3;  // ghost layers: PLM and LimO3 need 2, PPM 3 ("number of ghost cells ... adjusted")

enum { SOLVER_HLL = 0, SOLVER_HLLC = 1, SOLVER_HLLD = 2, SOLVER_ROE = 3, SOLVER_RUSANOV = 4 };
enum { LIM_FLAT = 0, LIM_MINMOD = 1, LIM_VANLEER = 2, LIM_LIMO3 = 3, LIM_PPM = 4 };
enum { OPT_INTEGRATOR = 0, OPT_CT_FORM = 1, OPT_PRESSURE_FLOOR = 2, OPT_BOUNDARY = 3 };  // idfxref_set_option / idfxref_set_option_real
enum { CT_FACE = 0, CT_POTENTIAL = 1 };
enum { EMF_NONE = 0, EMF_ARITH = 1, EMF_UCT = 2, EMF_UCT0 = 3, EMF_UCT_HLL = 4, EMF_UCT_HLLD = 5 };
enum { OK = 0, ERR_INVALID_ARG = -1, ERR_UNSUPPORTED = -2, ERR_UNPHYSICAL = -5 };

// ---------------------------------------------------------------------------------------------
// Point-wise physics.  A 1D state along direction d is W = (rho, u, v, w, p, By, Bz) with u the
// normal velocity and (By, Bz) the transverse field after cyclic permutation; Bn is the normal field.
// The conserved vector is U = (rho, rho u, rho v, rho w, E, By, Bz).
// ---------------------------------------------------------------------------------------------

// O1 / PAPER.md:61: E = p/(gamma-1) + rho v^2/2 + B^2/2.
void cons_from_prim(const double W[7], double Bn, double g, double U[7]) {
  const double rho = W[0], u = W[1], v = W[2], w = W[3], p = W[4], By = W[5], Bz = W[6];
  U[0] = rho;
  U[1] = rho * u;
  U[2] = rho * v;
  U[3] = rho * w;
  U[4] = p / (g - 1.0) + 0.5 * rho * (u * u + v * v + w * w) + 0.5 * (Bn * Bn + By * By + Bz * Bz);
  U[5] = By;
  U[6] = Bz;
}

// O4 / PAPER.md:43-53 (Eq. 1-4, ideal part), P = p + B^2/2.
void phys_flux(const double W[7], double Bn, const double U[7], double F[7]) {
  const double rho = W[0], u = W[1], v = W[2], w = W[3], p = W[4], By = W[5], Bz = W[6];
  const double pT = p + 0.5 * (Bn * Bn + By * By + Bz * Bz);
  F[0] = rho * u;
  F[1] = rho * u * u + pT - Bn * Bn;
  F[2] = rho * u * v - Bn * By;
  F[3] = rho * u * w - Bn * Bz;
  F[4] = (U[4] + pT) * u - Bn * (u * Bn + v * By + w * Bz);
  F[5] = u * By - v * Bn;
  F[6] = u * Bz - w * Bn;
}

// O4: a^2 = gamma p / rho; c_f^2 = (1/2)[a^2 + b^2 + sqrt((a^2+b^2)^2 - 4 a^2 Bn^2/rho)], b^2 = |B|^2/rho.
// With B = 0 this is exactly a.
double fast_speed(const double W[7], double Bn, double g) {
  const double rho = W[0], p = W[4], By = W[5], Bz = W[6];
  const double a2 = g * p / rho;
  const double b2 = (Bn * Bn + By * By + Bz * Bz) / rho;
  const double s = a2 + b2;
  double disc = s * s - 4.0 * a2 * Bn * Bn / rho;
  if (disc < 0.0) disc = 0.0;
  return std::sqrt(0.5 * (s + std::sqrt(disc)));
}

// O4 / G5 (Davis): S_L = min(u_L - c_L, u_R - c_R), S_R = max(u_L + c_L, u_R + c_R).
void davis_speeds(const double WL[7], const double WR[7], double Bn, double g, double& SL, double& SR) {
  const double cL = fast_speed(WL, Bn, g), cR = fast_speed(WR, Bn, g);
  SL = std::min(WL[1] - cL, WR[1] - cR);
  SR = std::max(WL[1] + cL, WR[1] + cR);
}

// O5 HLL.
void hll_flux(const double UL[7], const double UR[7], const double FL[7], const double FR[7], double SL,
              double SR, double F[7]) {
  if (SL >= 0.0) {
    for (int n = 0; n < 7; ++n) F[n] = FL[n];
  } else if (SR <= 0.0) {
    for (int n = 0; n < 7; ++n) F[n] = FR[n];
  } else {
    for (int n = 0; n < 7; ++n) F[n] = (SR * FL[n] - SL * FR[n] + SL * SR * (UR[n] - UL[n])) / (SR - SL);
  }
}

// Rusanov / local Lax-Friedrichs flux ("Lax-Friedrichs Rusanov flux (Rusanov 1962)", the most diffusive
// solver of the paper's list): F = (F_L + F_R)/2 - (c_face/2)(U_R - U_L) with c_face = max(|S_L|,|S_R|) (O4).
void rusanov_flux(const double UL[7], const double UR[7], const double FL[7], const double FR[7], double cface,
                  double F[7]) {
  for (int n = 0; n < 7; ++n) F[n] = 0.5 * (FL[n] + FR[n]) - 0.5 * cface * (UR[n] - UL[n]);
}

// O6 HLLC, hydrodynamics only (Toro et al. 1994).  Star states are returned for the pins.
struct HllcFan {
  double SL, SS, SR;
  double UsL[5], UsR[5];
};

void hllc_fan(const double WL[7], const double WR[7], const double UL[7], const double UR[7], double SL,
              double SR, HllcFan& f) {
  const double rL = WL[0], uL = WL[1], pL = WL[4];
  const double rR = WR[0], uR = WR[1], pR = WR[4];
  const double SS = (pR - pL + rL * uL * (SL - uL) - rR * uR * (SR - uR)) / (rL * (SL - uL) - rR * (SR - uR));
  f.SL = SL;
  f.SS = SS;
  f.SR = SR;
  {
    const double fac = rL * (SL - uL) / (SL - SS);
    f.UsL[0] = fac;
    f.UsL[1] = fac * SS;
    f.UsL[2] = fac * WL[2];
    f.UsL[3] = fac * WL[3];
    f.UsL[4] = fac * (UL[4] / rL + (SS - uL) * (SS + pL / (rL * (SL - uL))));
  }
  {
    const double fac = rR * (SR - uR) / (SR - SS);
    f.UsR[0] = fac;
    f.UsR[1] = fac * SS;
    f.UsR[2] = fac * WR[2];
    f.UsR[3] = fac * WR[3];
    f.UsR[4] = fac * (UR[4] / rR + (SS - uR) * (SS + pR / (rR * (SR - uR))));
  }
}

void hllc_flux(const double WL[7], const double WR[7], const double UL[7], const double UR[7],
               const double FL[7], const double FR[7], double SL, double SR, double F[7]) {
  F[5] = 0.0;
  F[6] = 0.0;
  if (SL >= 0.0) {
    for (int n = 0; n < 5; ++n) F[n] = FL[n];
    return;
  }
  if (SR <= 0.0) {
    for (int n = 0; n < 5; ++n) F[n] = FR[n];
    return;
  }
  HllcFan f;
  hllc_fan(WL, WR, UL, UR, SL, SR, f);
  if (f.SS >= 0.0) {
    for (int n = 0; n < 5; ++n) F[n] = FL[n] + SL * (f.UsL[n] - UL[n]);
  } else {
    for (int n = 0; n < 5; ++n) F[n] = FR[n] + SR * (f.UsR[n] - UR[n]);
  }
}

// O7 HLLD (Miyoshi & Kusano 2005).  The five speeds and four intermediate states are
// returned for the pins.
struct HlldFan {
  double SL, SsL, SM, SsR, SR;
  double UsL[7], UssL[7], UssR[7], UsR[7];
};

void hlld_fan(const double WL[7], const double WR[7], double Bn, const double UL[7], const double UR[7],
              double SL, double SR, HlldFan& f) {
  const double rL = WL[0], uL = WL[1], vL = WL[2], wL = WL[3], pL = WL[4], ByL = WL[5], BzL = WL[6];
  const double rR = WR[0], uR = WR[1], vR = WR[2], wR = WR[3], pR = WR[4], ByR = WR[5], BzR = WR[6];
  const double pTL = pL + 0.5 * (Bn * Bn + ByL * ByL + BzL * BzL);
  const double pTR = pR + 0.5 * (Bn * Bn + ByR * ByR + BzR * BzR);
  const double sgn = (Bn >= 0.0) ? 1.0 : -1.0;

  const double D = (SR - uR) * rR - (SL - uL) * rL;
  const double SM = ((SR - uR) * rR * uR - (SL - uL) * rL * uL - pTR + pTL) / D;
  const double pTs =
      ((SR - uR) * rR * pTL - (SL - uL) * rL * pTR + rL * rR * (SR - uR) * (SL - uL) * (uR - uL)) / D;

  // star states, K = L, R
  double rsL, vsL, wsL, BysL, BzsL, EsL;
  double rsR, vsR, wsR, BysR, BzsR, EsR;
  {
    rsL = rL * (SL - uL) / (SL - SM);
    const double dK = rL * (SL - uL) * (SL - SM) - Bn * Bn;
    if (std::fabs(dK) < 1e-12 * rL * (SL - uL) * (SL - uL)) {  // G6
      vsL = vL;
      wsL = wL;
      BysL = ByL;
      BzsL = BzL;
    } else {
      vsL = vL - Bn * ByL * (SM - uL) / dK;
      wsL = wL - Bn * BzL * (SM - uL) / dK;
      const double num = rL * (SL - uL) * (SL - uL) - Bn * Bn;
      BysL = ByL * num / dK;
      BzsL = BzL * num / dK;
    }
    const double vB = uL * Bn + vL * ByL + wL * BzL;
    const double vBs = SM * Bn + vsL * BysL + wsL * BzsL;
    EsL = ((SL - uL) * UL[4] - pTL * uL + pTs * SM + Bn * (vB - vBs)) / (SL - SM);
  }
  {
    rsR = rR * (SR - uR) / (SR - SM);
    const double dK = rR * (SR - uR) * (SR - SM) - Bn * Bn;
    if (std::fabs(dK) < 1e-12 * rR * (SR - uR) * (SR - uR)) {  // G6
      vsR = vR;
      wsR = wR;
      BysR = ByR;
      BzsR = BzR;
    } else {
      vsR = vR - Bn * ByR * (SM - uR) / dK;
      wsR = wR - Bn * BzR * (SM - uR) / dK;
      const double num = rR * (SR - uR) * (SR - uR) - Bn * Bn;
      BysR = ByR * num / dK;
      BzsR = BzR * num / dK;
    }
    const double vB = uR * Bn + vR * ByR + wR * BzR;
    const double vBs = SM * Bn + vsR * BysR + wsR * BzsR;
    EsR = ((SR - uR) * UR[4] - pTR * uR + pTs * SM + Bn * (vB - vBs)) / (SR - SM);
  }
  const double sqL = std::sqrt(rsL), sqR = std::sqrt(rsR);
  f.SL = SL;
  f.SR = SR;
  f.SM = SM;
  f.SsL = SM - std::fabs(Bn) / sqL;
  f.SsR = SM + std::fabs(Bn) / sqR;

  // double-star states
  const double inv = 1.0 / (sqL + sqR);
  const double vss = (sqL * vsL + sqR * vsR + (BysR - BysL) * sgn) * inv;
  const double wss = (sqL * wsL + sqR * wsR + (BzsR - BzsL) * sgn) * inv;
  const double Byss = (sqL * BysR + sqR * BysL + sqL * sqR * (vsR - vsL) * sgn) * inv;
  const double Bzss = (sqL * BzsR + sqR * BzsL + sqL * sqR * (wsR - wsL) * sgn) * inv;
  const double vBss = SM * Bn + vss * Byss + wss * Bzss;
  const double vBsL = SM * Bn + vsL * BysL + wsL * BzsL;
  const double vBsR = SM * Bn + vsR * BysR + wsR * BzsR;
  const double EssL = EsL - sqL * (vBsL - vBss) * sgn;
  const double EssR = EsR + sqR * (vBsR - vBss) * sgn;

  f.UsL[0] = rsL; f.UsL[1] = rsL * SM; f.UsL[2] = rsL * vsL; f.UsL[3] = rsL * wsL; f.UsL[4] = EsL;
  f.UsL[5] = BysL; f.UsL[6] = BzsL;
  f.UsR[0] = rsR; f.UsR[1] = rsR * SM; f.UsR[2] = rsR * vsR; f.UsR[3] = rsR * wsR; f.UsR[4] = EsR;
  f.UsR[5] = BysR; f.UsR[6] = BzsR;
  f.UssL[0] = rsL; f.UssL[1] = rsL * SM; f.UssL[2] = rsL * vss; f.UssL[3] = rsL * wss; f.UssL[4] = EssL;
  f.UssL[5] = Byss; f.UssL[6] = Bzss;
  f.UssR[0] = rsR; f.UssR[1] = rsR * SM; f.UssR[2] = rsR * vss; f.UssR[3] = rsR * wss; f.UssR[4] = EssR;
  f.UssR[5] = Byss; f.UssR[6] = Bzss;
}

void hlld_flux(const double WL[7], const double WR[7], double Bn, const double UL[7], const double UR[7],
               const double FL[7], const double FR[7], double SL, double SR, double F[7]) {
  if (SL >= 0.0) {
    for (int n = 0; n < 7; ++n) F[n] = FL[n];
    return;
  }
  if (SR <= 0.0) {
    for (int n = 0; n < 7; ++n) F[n] = FR[n];
    return;
  }
  HlldFan f;
  hlld_fan(WL, WR, Bn, UL, UR, SL, SR, f);
  // selection in exactly the order of O7
  if (f.SsL >= 0.0) {
    for (int n = 0; n < 7; ++n) F[n] = FL[n] + SL * (f.UsL[n] - UL[n]);
  } else if (f.SsR <= 0.0) {
    for (int n = 0; n < 7; ++n) F[n] = FR[n] + SR * (f.UsR[n] - UR[n]);
  } else if (f.SM >= 0.0) {
    for (int n = 0; n < 7; ++n)
      F[n] = FL[n] + f.SsL * f.UssL[n] - (f.SsL - SL) * f.UsL[n] - SL * UL[n];
  } else {
    for (int n = 0; n < 7; ++n)
      F[n] = FR[n] + f.SsR * f.UssR[n] - (f.SsR - SR) * f.UsR[n] - SR * UR[n];
  }
}

// 2D-HLLD EMF, face part ("2D ... HLLD Riemann solvers ... following the method of Mignone & Del Zanna
// (2021)"; reading G24).  In every region of the HLLD fan the flux of a transverse field component is LINEAR in the two
// face states and can be written, for t = t1, t2 alike,
//     F_n[B_t] = a_L u_L B_t,L + a_R u_R B_t,R - (d_R B_t,R - d_L B_t,L) - vbar_t B_n ,      a_L + a_R = 1,
// i.e. an upwinded transport of B_t along n plus the stretching of B_n by an effective transverse velocity.  With
// h_K = [rho_K (S_K-u_K)^2 - B_n^2]/d_K, g_K = B_n (S_M-u_K)/d_K (B*_t,K = h_K B_t,K, v*_t,K = v_t,K - g_K B_t,K; G6: h = 1, g = 0),
// s_K = sqrt(rho*_K), sgn = sign(B_n), sigma_K = S*_K s_K/(s_L+s_R), and the regions in the order of O7:
//   L  : a_L = 1, d = 0, vbar = v_L                           R  : mirror image
//   L* : a_L = 1, d_L = S_L (h_L - 1), d_R = 0, vbar = v_L    R* : a_R = 1, d_R = -S_R (h_R - 1), d_L = 0, vbar = v_R
//   L**: a_L = 1, d_L = S_L (h_L - 1) - sigma_L (h_L - s_R sgn g_L), d_R = -sigma_L (h_R - s_R sgn g_R)
//   R**: a_R = 1, d_R = -S_R (h_R - 1) + sigma_R (h_R + s_L sgn g_R), d_L = sigma_R (h_L + s_L sgn g_L)
//   both **: vbar = (s_L v_L + s_R v_R)/(s_L+s_R) - S_M s_L s_R (v_R - v_L) / ((s_L+s_R) |B_n|)
// (write out F = F*_K + S*_K (B**_t - B*_t,K) with the double-star states of O7 and collect the terms; the |B_n| part of
// S*_K turns v_K into the density-weighted mean, the S_M part is the last term; |S_M| <= |B_n|/s_K inside the ** fan).
// For equal states h = 1, g = 0 and d_L = d_R, as consistency demands.  out = (a_L, d_L, d_R, vbar_t1, vbar_t2).
void hlld_uct_coeffs(const double WL[7], const double WR[7], double Bn, double g, double out[5]) {
  double UL[7], UR[7], SL, SR;
  cons_from_prim(WL, Bn, g, UL);
  cons_from_prim(WR, Bn, g, UR);
  davis_speeds(WL, WR, Bn, g, SL, SR);
  if (SL >= 0.0) {
    out[0] = 1.0; out[1] = 0.0; out[2] = 0.0; out[3] = WL[2]; out[4] = WL[3];
    return;
  }
  if (SR <= 0.0) {
    out[0] = 0.0; out[1] = 0.0; out[2] = 0.0; out[3] = WR[2]; out[4] = WR[3];
    return;
  }
  HlldFan f;
  hlld_fan(WL, WR, Bn, UL, UR, SL, SR, f);
  const double SM = f.SM;
  double h[2], gk[2];
  const double* W[2] = {WL, WR};
  const double SK[2] = {SL, SR};
  for (int K = 0; K < 2; ++K) {
    const double r = W[K][0], u = W[K][1];
    const double dK = r * (SK[K] - u) * (SK[K] - SM) - Bn * Bn;
    if (std::fabs(dK) < 1e-12 * r * (SK[K] - u) * (SK[K] - u)) {  // G6
      h[K] = 1.0;
      gk[K] = 0.0;
    } else {
      h[K] = (r * (SK[K] - u) * (SK[K] - u) - Bn * Bn) / dK;
      gk[K] = Bn * (SM - u) / dK;
    }
  }
  const double sL = std::sqrt(f.UsL[0]), sR = std::sqrt(f.UsR[0]);
  const double sgn = (Bn >= 0.0) ? 1.0 : -1.0;
  if (f.SsL >= 0.0) {
    out[0] = 1.0; out[1] = SL * (h[0] - 1.0); out[2] = 0.0; out[3] = WL[2]; out[4] = WL[3];
  } else if (f.SsR <= 0.0) {
    out[0] = 0.0; out[1] = 0.0; out[2] = -SR * (h[1] - 1.0); out[3] = WR[2]; out[4] = WR[3];
  } else {
    if (SM >= 0.0) {
      const double sig = f.SsL * sL / (sL + sR);
      out[0] = 1.0;
      out[1] = SL * (h[0] - 1.0) - sig * (h[0] - sR * sgn * gk[0]);
      out[2] = -sig * (h[1] - sR * sgn * gk[1]);
    } else {
      const double sig = f.SsR * sR / (sL + sR);
      out[0] = 0.0;
      out[2] = -SR * (h[1] - 1.0) + sig * (h[1] + sL * sgn * gk[1]);
      out[1] = sig * (h[0] + sL * sgn * gk[0]);
    }
    const double theta = -SM * sL * sR / ((sL + sR) * std::fabs(Bn));  // |B_n| > 0 here: the ** fan has zero width otherwise
    out[3] = (sL * WL[2] + sR * WR[2]) / (sL + sR) + theta * (WR[2] - WL[2]);
    out[4] = (sL * WL[3] + sR * WR[3]) / (sL + sR) + theta * (WR[3] - WL[3]);
  }
}

// O8 Roe ("approximate linear Roe Riemann solver (Cargo & Gallice 1997)").
// Eigen-system in primitive variables W = (rho,u,v,w,p,By,Bz) at the Roe-averaged state, plus the
// matrices M = dU/dW and Minv = dW/dU of the shifted equation of state (O8).  Returns false when
// a~^2 <= 0 (G7: the caller then falls back to HLL).
struct RoeSys {
  double lam[7];
  double R[7][7];  // R[k][:] = k-th right eigenvector (primitive)
  double L[7][7];  // L[k][:] = k-th left eigenvector (primitive)
  double M[7][7];
  double Minv[7][7];
};

bool roe_system(const double WL[7], const double WR[7], double Bn, const double UL[7], const double UR[7],
                double g, RoeSys& s) {
  const double rL = WL[0], rR = WR[0];
  const double sL = std::sqrt(rL), sR = std::sqrt(rR);
  const double isum = 1.0 / (sL + sR);
  const double rb = sL * sR;
  const double ub = (sL * WL[1] + sR * WR[1]) * isum;
  const double vb = (sL * WL[2] + sR * WR[2]) * isum;
  const double wb = (sL * WL[3] + sR * WR[3]) * isum;
  const double pTL = WL[4] + 0.5 * (Bn * Bn + WL[5] * WL[5] + WL[6] * WL[6]);
  const double pTR = WR[4] + 0.5 * (Bn * Bn + WR[5] * WR[5] + WR[6] * WR[6]);
  const double HL = (UL[4] + pTL) / rL, HR = (UR[4] + pTR) / rR;
  const double Hb = (sL * HL + sR * HR) * isum;
  const double Byb = (sR * WL[5] + sL * WR[5]) * isum;  // weights swapped (O8)
  const double Bzb = (sR * WL[6] + sL * WR[6]) * isum;
  const double dBy = WR[5] - WL[5], dBz = WR[6] - WL[6];
  const double X = (dBy * dBy + dBz * dBz) * 0.5 * isum * isum;
  const double Xp = (g - 2.0) * X;
  const double v2 = ub * ub + vb * vb + wb * wb;
  const double a2 = (g - 1.0) * (Hb - 0.5 * v2 - (Bn * Bn + Byb * Byb + Bzb * Bzb) / rb) - Xp;
  if (!(a2 > 0.0)) return false;
  const double a = std::sqrt(a2);

  const double bn2 = Bn * Bn / rb;
  const double bt2 = (Byb * Byb + Bzb * Bzb) / rb;
  const double sum = a2 + bn2 + bt2;
  double disc = sum * sum - 4.0 * a2 * bn2;
  if (disc < 0.0) disc = 0.0;
  const double Cf2 = 0.5 * (sum + std::sqrt(disc));
  const double Cs2 = a2 * bn2 / Cf2;
  const double Cf = std::sqrt(Cf2), Cs = std::sqrt(Cs2);
  const double CA = std::sqrt(bn2);

  double af, as;
  if (Cf2 - Cs2 <= 0.0) {
    af = 1.0;
    as = 0.0;
  } else {
    double af2 = (a2 - Cs2) / (Cf2 - Cs2), as2 = (Cf2 - a2) / (Cf2 - Cs2);
    af2 = std::min(1.0, std::max(0.0, af2));
    as2 = std::min(1.0, std::max(0.0, as2));
    af = std::sqrt(af2);
    as = std::sqrt(as2);
  }
  const double Bt = std::sqrt(Byb * Byb + Bzb * Bzb);
  double by, bz;
  if (Bt == 0.0) {
    by = bz = 1.0 / std::sqrt(2.0);
  } else {
    by = Byb / Bt;
    bz = Bzb / Bt;
  }
  const double S = (Bn >= 0.0) ? 1.0 : -1.0;
  const double sr = std::sqrt(rb);
  const double Cff = Cf * af, Css = Cs * as, Qf = Cf * af * S, Qs = Cs * as * S;
  const double Af = a * af * sr, As = a * as * sr;

  s.lam[0] = ub - Cf; s.lam[1] = ub - CA; s.lam[2] = ub - Cs; s.lam[3] = ub;
  s.lam[4] = ub + Cs; s.lam[5] = ub + CA; s.lam[6] = ub + Cf;

  const double i2a2 = 1.0 / (2.0 * a2);
  for (int k = 0; k < 7; ++k)
    for (int n = 0; n < 7; ++n) s.R[k][n] = s.L[k][n] = 0.0;
  // fast, sign = -1 for k=0 (u - Cf), +1 for k=6
  for (int pm = 0; pm < 2; ++pm) {
    const int k = pm ? 6 : 0;
    const double sg = pm ? 1.0 : -1.0;
    double* r = s.R[k];
    double* l = s.L[k];
    r[0] = rb * af; r[1] = sg * Cff; r[2] = -sg * Qs * by; r[3] = -sg * Qs * bz; r[4] = rb * a2 * af;
    r[5] = As * by; r[6] = As * bz;
    l[0] = 0.0; l[1] = sg * Cff * i2a2; l[2] = -sg * Qs * by * i2a2; l[3] = -sg * Qs * bz * i2a2;
    l[4] = af / rb * i2a2; l[5] = As * by / rb * i2a2; l[6] = As * bz / rb * i2a2;
  }
  // Alfven, k=1 (u - CA), k=5 (u + CA)
  for (int pm = 0; pm < 2; ++pm) {
    const int k = pm ? 5 : 1;
    const double sg = pm ? 1.0 : -1.0;
    double* r = s.R[k];
    double* l = s.L[k];
    r[2] = sg * bz; r[3] = -sg * by; r[5] = -S * sr * bz; r[6] = S * sr * by;
    l[2] = 0.5 * sg * bz; l[3] = -0.5 * sg * by; l[5] = -0.5 * S * bz / sr; l[6] = 0.5 * S * by / sr;
  }
  // slow, k=2 (u - Cs), k=4 (u + Cs)
  for (int pm = 0; pm < 2; ++pm) {
    const int k = pm ? 4 : 2;
    const double sg = pm ? 1.0 : -1.0;
    double* r = s.R[k];
    double* l = s.L[k];
    r[0] = rb * as; r[1] = sg * Css; r[2] = sg * Qf * by; r[3] = sg * Qf * bz; r[4] = rb * a2 * as;
    r[5] = -Af * by; r[6] = -Af * bz;
    l[0] = 0.0; l[1] = sg * Css * i2a2; l[2] = sg * Qf * by * i2a2; l[3] = sg * Qf * bz * i2a2;
    l[4] = as / rb * i2a2; l[5] = -Af * by / rb * i2a2; l[6] = -Af * bz / rb * i2a2;
  }
  // entropy
  s.R[3][0] = 1.0;
  s.L[3][0] = 1.0;
  s.L[3][4] = -1.0 / a2;

  for (int r = 0; r < 7; ++r)
    for (int c = 0; c < 7; ++c) s.M[r][c] = s.Minv[r][c] = 0.0;
  const double gm1 = g - 1.0;
  s.M[0][0] = 1.0;
  s.M[1][0] = ub; s.M[1][1] = rb;
  s.M[2][0] = vb; s.M[2][2] = rb;
  s.M[3][0] = wb; s.M[3][3] = rb;
  s.M[4][0] = 0.5 * v2 + Xp / gm1; s.M[4][1] = rb * ub; s.M[4][2] = rb * vb; s.M[4][3] = rb * wb;
  s.M[4][4] = 1.0 / gm1; s.M[4][5] = Byb; s.M[4][6] = Bzb;
  s.M[5][5] = 1.0;
  s.M[6][6] = 1.0;
  s.Minv[0][0] = 1.0;
  s.Minv[1][0] = -ub / rb; s.Minv[1][1] = 1.0 / rb;
  s.Minv[2][0] = -vb / rb; s.Minv[2][2] = 1.0 / rb;
  s.Minv[3][0] = -wb / rb; s.Minv[3][3] = 1.0 / rb;
  s.Minv[4][0] = gm1 * 0.5 * v2 - Xp; s.Minv[4][1] = -gm1 * ub; s.Minv[4][2] = -gm1 * vb;
  s.Minv[4][3] = -gm1 * wb; s.Minv[4][4] = gm1; s.Minv[4][5] = -gm1 * Byb; s.Minv[4][6] = -gm1 * Bzb;
  s.Minv[5][5] = 1.0;
  s.Minv[6][6] = 1.0;
  return true;
}

// F = (F_L+F_R)/2 - (1/2) sum_k |lambda_k| alpha_k r_k, alpha = L (Minv dU), r^cons = M r  (O8, no entropy fix).
bool roe_flux(const double WL[7], const double WR[7], double Bn, const double UL[7], const double UR[7],
              const double FL[7], const double FR[7], double g, double F[7]) {
  RoeSys s;
  if (!roe_system(WL, WR, Bn, UL, UR, g, s)) return false;
  double dU[7], dW[7], acc[7];
  for (int n = 0; n < 7; ++n) dU[n] = UR[n] - UL[n];
  for (int r = 0; r < 7; ++r) {
    double t = 0.0;
    for (int c = 0; c < 7; ++c) t += s.Minv[r][c] * dU[c];
    dW[r] = t;
  }
  for (int n = 0; n < 7; ++n) acc[n] = 0.0;
  for (int k = 0; k < 7; ++k) {
    double alpha = 0.0;
    for (int n = 0; n < 7; ++n) alpha += s.L[k][n] * dW[n];
    const double c = std::fabs(s.lam[k]) * alpha;
    for (int n = 0; n < 7; ++n) acc[n] += c * s.R[k][n];
  }
  for (int r = 0; r < 7; ++r) {
    double t = 0.0;
    for (int c = 0; c < 7; ++c) t += s.M[r][c] * acc[c];
    F[r] = 0.5 * (FL[r] + FR[r]) - 0.5 * t;
  }
  return true;
}

// One Riemann problem: flux F and the face signal speed c_face = max(|S_L|,|S_R|) for every solver (O4).
// Returns 1 when the Roe solver fell back to HLL (G7), else 0.
int riemann(int solver, double g, const double WL[7], const double WR[7], double Bn, double F[7],
            double& cface) {
  double UL[7], UR[7], FL[7], FR[7], SL, SR;
  cons_from_prim(WL, Bn, g, UL);
  cons_from_prim(WR, Bn, g, UR);
  phys_flux(WL, Bn, UL, FL);
  phys_flux(WR, Bn, UR, FR);
  davis_speeds(WL, WR, Bn, g, SL, SR);
  cface = std::max(std::fabs(SL), std::fabs(SR));
  int fallback = 0;
  switch (solver) {
    case SOLVER_HLL: hll_flux(UL, UR, FL, FR, SL, SR, F); break;
    case SOLVER_HLLC: hllc_flux(WL, WR, UL, UR, FL, FR, SL, SR, F); break;
    case SOLVER_HLLD: hlld_flux(WL, WR, Bn, UL, UR, FL, FR, SL, SR, F); break;
    case SOLVER_RUSANOV: rusanov_flux(UL, UR, FL, FR, cface, F); break;
    default:
      if (!roe_flux(WL, WR, Bn, UL, UR, FL, FR, g, F)) {
        hll_flux(UL, UR, FL, FR, SL, SR, F);
        fallback = 1;
      }
  }
  return fallback;
}

// O3 limited slope (G2): zero at extrema; van Leer = harmonic mean; minmod = smaller one.
double slope(int limiter, double dm, double dp) {
  if (limiter == LIM_FLAT) return 0.0;
  if (dm * dp <= 0.0) return 0.0;
  if (limiter == LIM_VANLEER) return 2.0 * dm * dp / (dm + dp);
  const double s = (dm > 0.0) ? 1.0 : -1.0;
  return s * std::min(std::fabs(dm), std::fabs(dp));
}

// LimO3 ("LimO3 (Cada & Torrilhon 2009)"; reading G18).  With d- = q_i - q_{i-1},
// d+ = q_{i+1} - q_i and theta = d-/d+, the value at the upper face of cell i is q_i + phi(theta) d+ / 2, where the
// unlimited third-order weight is phi^(theta) = (2 + theta)/3 (exact for cell averages of a parabola) and the limited
// one phi_O3 = max(0, min(phi^, max(-theta/2, min(2 theta, phi^, 1.6)))).  The limiter is switched off where the data
// are smooth: eta = (d-^2 + d+^2)/(r dx)^2 with r = 1; eta <= 1 - eps -> phi^, eta >= 1 + eps -> phi_O3, linear blend
// in between, eps = 1e-12.  The lower face is the mirror image (d- and d+ exchanged, sign flipped).
// Returns phi(theta) * dplus, the full increment; the face value is q + half of it.
double limo3_increment(double dminus, double dplus, double dx) {
  const double eps = 1e-12, r = 1.0;
  const double unlimited = (2.0 * dplus + dminus) / 3.0;  // phi^(theta) d+
  double limited = 0.0;
  if (dplus != 0.0) {
    const double theta = dminus / dplus;
    const double phat = (2.0 + theta) / 3.0;
    const double phi = std::max(0.0, std::min(phat, std::max(-0.5 * theta, std::min(std::min(2.0 * theta, phat), 1.6))));
    limited = phi * dplus;
  }
  const double eta = (dminus * dminus + dplus * dplus) / ((r * dx) * (r * dx));
  if (eta <= 1.0 - eps) return unlimited;
  if (eta >= 1.0 + eps) return limited;
  return 0.5 * ((1.0 - (eta - 1.0) / eps) * unlimited + (1.0 + (eta - 1.0) / eps) * limited);
}

// S2: values of the reconstruction of cell i at its lower and upper faces from (q_{i-1}, q_i, q_{i+1}).
void reconstruct(int limiter, double qm, double q0, double qp, double dx, double& lower, double& upper) {
  if (limiter == LIM_LIMO3) {
    upper = q0 + 0.5 * limo3_increment(q0 - qm, qp - q0, dx);
    lower = q0 - 0.5 * limo3_increment(qp - q0, q0 - qm, dx);
    return;
  }
  const double s = slope(limiter, q0 - qm, qp - q0);
  lower = q0 - 0.5 * s;
  upper = q0 + 0.5 * s;
}

// PPM ("piecewise parabolic reconstruction using an extremum-preserving limiter (4th order accurate on
// regularly spaced grids, Colella & Woodward 1984; Colella & Sekora 2008)"; only named there: reading G22).  On a uniform
// grid, with a_j the cell values:
//  (1) interface value, CW84 Eq. 1.9:  a_{j+1/2} = 7/12 (a_j + a_{j+1}) - 1/12 (a_{j-1} + a_{j+2});
//  (2) CS08 Sec. 2.3: where a_{j+1/2} does not lie between a_j and a_{j+1} it is replaced by
//      (a_j + a_{j+1})/2 - D2lim/6, with D2 = 3 (a_j - 2 a_{j+1/2} + a_{j+1}), D2L = a_{j-1} - 2 a_j + a_{j+1},
//      D2R = a_j - 2 a_{j+1} + a_{j+2}, and D2lim = s min(C |D2L|, C |D2R|, |D2|) when the three share the sign s, else 0;
//  (3) CS08 Sec. 2.4, parabola of cell j with edge values a- = a_{j-1/2}, a+ = a_{j+1/2}:
//      at a local extremum ((a+ - a_j)(a_j - a-) <= 0 or (a_{j+1} - a_j)(a_j - a_{j-1}) <= 0) both edge deviations are scaled
//      by D2lim/D2f, D2f = 6 (a+ - 2 a_j + a-), D2lim = s min(|D2f|, C |D2L|, C |D2C|, C |D2R|) from the second differences
//      of the cell values centred at j-1, j, j+1 when all four share the sign s, else 0 (a smooth extremum keeps its
//      parabola, a non-smooth one is flattened); elsewhere the CW84 overshoot rule, one side at a time:
//      |a+ - a_j| >= 2 |a- - a_j|  ->  a+ = a_j - 2 (a- - a_j), and the mirror image.  C = 1.25.
double ppm_interface(double am1, double a0, double ap1, double ap2) {
  const double C = 1.25;
  double f = (7.0 * (a0 + ap1) - (am1 + ap2)) / 12.0;
  if ((f - a0) * (ap1 - f) < 0.0) {
    const double D2 = 3.0 * (a0 - 2.0 * f + ap1);
    const double D2L = am1 - 2.0 * a0 + ap1;
    const double D2R = a0 - 2.0 * ap1 + ap2;
    double D2lim = 0.0;
    if (D2 > 0.0 && D2L > 0.0 && D2R > 0.0) D2lim = std::min(std::min(C * D2L, C * D2R), D2);
    if (D2 < 0.0 && D2L < 0.0 && D2R < 0.0) D2lim = -std::min(std::min(-C * D2L, -C * D2R), -D2);
    f = 0.5 * (a0 + ap1) - D2lim / 6.0;
  }
  return f;
}

// a[0..4] = a_{j-2} .. a_{j+2}; values of cell j's limited parabola at its lower and upper faces
void ppm_faces(const double a[5], double& lower, double& upper) {
  const double C = 1.25;
  const double a0 = a[2];
  double am = ppm_interface(a[0], a[1], a[2], a[3]);
  double ap = ppm_interface(a[1], a[2], a[3], a[4]);
  const double dm = a0 - am, dp = ap - a0;
  if (dm * dp <= 0.0 || (a[3] - a0) * (a0 - a[1]) <= 0.0) {
    const double D2f = 6.0 * (ap - 2.0 * a0 + am);
    const double D2L = a[0] - 2.0 * a[1] + a[2];
    const double D2C = a[1] - 2.0 * a[2] + a[3];
    const double D2R = a[2] - 2.0 * a[3] + a[4];
    double D2lim = 0.0;
    if (D2f > 0.0 && D2L > 0.0 && D2C > 0.0 && D2R > 0.0)
      D2lim = std::min(std::min(C * D2L, C * D2R), std::min(C * D2C, D2f));
    if (D2f < 0.0 && D2L < 0.0 && D2C < 0.0 && D2R < 0.0)
      D2lim = -std::min(std::min(-C * D2L, -C * D2R), std::min(-C * D2C, -D2f));
    const double ratio = (D2f == 0.0) ? 0.0 : D2lim / D2f;
    ap = a0 + dp * ratio;
    am = a0 - dm * ratio;
  } else {
    if (std::fabs(dp) >= 2.0 * std::fabs(dm)) ap = a0 + 2.0 * dm;
    if (std::fabs(dm) >= 2.0 * std::fabs(dp)) am = a0 - 2.0 * dp;
  }
  lower = am;
  upper = ap;
}

// ---------------------------------------------------------------------------------------------
// Grid-level scheme
// ---------------------------------------------------------------------------------------------
typedef std::vector<double> Arr;

struct Ctx {
  int n[3];
  double dx, g;
  int solver, limiter, emf;
  bool mhd;
  int p[3];
  size_t st[3];  // strides in doubles: st[0] = 1
  size_t N;
  Arr U[5], U0[5], U1[5], Us[5];    // master conserved state, saved state, stage-1 state, scratch
  Arr Bf[3], Bf0[3], Bf1[3], Bfs[3];
  Arr V[8];                         // rho, vx, vy, vz, p, Bcx, Bcy, Bcz
  Arr F[3][7];                      // face fluxes per direction in that direction's local ordering
  Arr cf[3];                        // c_face per direction
  Arr E[3];                         // edge EMFs: E[0] at (i, j-1/2, k-1/2), E[1] at (i-1/2, j, k-1/2), E[2] at (i-1/2, j-1/2, k)
  Arr Vt[3][2], Al[3][2];           // EMF_UCT_HLL: per d-face, the HLL-weighted transverse velocities (components d+1, d+2)
                                    // and the one-sided speeds alpha+ = max(0, S_R), alpha- = max(0, -S_L)
  Arr Hc[3][5];                     // EMF_UCT_HLLD: per d-face (a_L, d_L, d_R, vbar_t1, vbar_t2) of hlld_uct_coeffs
  const Arr* Bstage;                // face field of the stage input (edge_emf reads it for EMF_UCT_HLL / EMF_UCT_HLLD)
  int nstages;                      // 1 Euler, 2 RK2, 3 RK3 (Tab. 1)
  int ct_form;                      // CT_FACE: Eq. 6; CT_POTENTIAL: Eq. 7-8
  Arr A[3], A0[3], As[3], Bref[3];  // CT_POTENTIAL: edge potential accumulated since set_state (same places as E),
                                    // its saved and scratch copies, and the face field given to set_state (G19)
  double t;                         // time since set_state
  int outflow;                      // 0: periodic; 1: zero-gradient ghosts on all six sides.  With a
                                    // magnetic field (reading G23) the staggered components are zero-gradient too: every ghost
                                    // face copies the nearest active face of its line, the upper boundary face (index n, not
                                    // part of the state) included; it is not evolved, and div B is kept on the cells whose six
                                    // faces all belong to the state
  double pfloor;                    // optional pressure floor (0 = none, G13); see compute_prims
  long long nfloor;                 // how often it acted since set_state
  double last_dt;
  int status;
  long long roe_fallbacks;

  size_t at(int i, int j, int k) const {
    return (size_t)(k + NG) * st[2] + (size_t)(j + NG) * st[1] + (size_t)(i + NG);
  }
};

inline int pmod(int a, int n) {
  int r = a % n;
  return r < 0 ? r + n : r;
}

// a1 / O2(i): periodic fill, 2 layers, x then y then z (PAPER.md:233 sequential per-dimension order).
void fill_periodic(const Ctx& c, Arr& a) {
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  if (c.outflow) {  // zero gradient, same sequential order: each ghost layer copies the last active cell of its line
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int gI = 1; gI <= NG; ++gI) {
          a[c.at(-gI, j, k)] = a[c.at(0, j, k)];
          a[c.at(nx - 1 + gI, j, k)] = a[c.at(nx - 1, j, k)];
        }
    for (int k = 0; k < nz; ++k)
      for (int gI = 1; gI <= NG; ++gI)
        for (int i = -NG; i < nx + NG; ++i) {
          a[c.at(i, -gI, k)] = a[c.at(i, 0, k)];
          a[c.at(i, ny - 1 + gI, k)] = a[c.at(i, ny - 1, k)];
        }
    for (int gI = 1; gI <= NG; ++gI)
      for (int j = -NG; j < ny + NG; ++j)
        for (int i = -NG; i < nx + NG; ++i) {
          a[c.at(i, j, -gI)] = a[c.at(i, j, 0)];
          a[c.at(i, j, nz - 1 + gI)] = a[c.at(i, j, nz - 1)];
        }
    return;
  }
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int gI = 1; gI <= NG; ++gI) {
        a[c.at(-gI, j, k)] = a[c.at(pmod(-gI, nx), j, k)];
        a[c.at(nx - 1 + gI, j, k)] = a[c.at(pmod(nx - 1 + gI, nx), j, k)];
      }
  for (int k = 0; k < nz; ++k)
    for (int gI = 1; gI <= NG; ++gI)
      for (int i = -NG; i < nx + NG; ++i) {
        a[c.at(i, -gI, k)] = a[c.at(i, pmod(-gI, ny), k)];
        a[c.at(i, ny - 1 + gI, k)] = a[c.at(i, pmod(ny - 1 + gI, ny), k)];
      }
  for (int gI = 1; gI <= NG; ++gI)
    for (int j = -NG; j < ny + NG; ++j)
      for (int i = -NG; i < nx + NG; ++i) {
        a[c.at(i, j, -gI)] = a[c.at(i, j, pmod(-gI, nz))];
        a[c.at(i, j, nz - 1 + gI)] = a[c.at(i, j, pmod(nz - 1 + gI, nz))];
      }
}

// a2 / O1: Bc = mean of the two bounding faces (G1); v = m/rho; p = (gamma-1)(E - rho v^2/2 - Bc^2/2).
// Needs the face ghosts of Bf (face index n).  Prims are computed on active cells and then filled
// periodically, which is bit-identical to computing them in the ghosts from filled U and Bf (O2 (i)-(ii)).
// Optional (reading G20, off by default): a pressure below c.pfloor is raised to it and E is rewritten to match.
void compute_prims(Ctx& c, Arr U[5], const Arr Bf[3]) {
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        const size_t q = c.at(i, j, k);
        double bx = 0.0, by = 0.0, bz = 0.0;
        if (c.mhd) {
          bx = 0.5 * (Bf[0][q] + Bf[0][q + c.st[0]]);
          by = 0.5 * (Bf[1][q] + Bf[1][q + c.st[1]]);
          bz = 0.5 * (Bf[2][q] + Bf[2][q + c.st[2]]);
        }
        const double rho = U[0][q];
        const double vx = U[1][q] / rho, vy = U[2][q] / rho, vz = U[3][q] / rho;
        double p =
            (c.g - 1.0) * (U[4][q] - 0.5 * rho * (vx * vx + vy * vy + vz * vz) - 0.5 * (bx * bx + by * by + bz * bz));
        if (c.pfloor > 0.0 && p < c.pfloor) {
          // a cell floored before recomputes to the floor within rounding: its energy is left as it is
          if (p < c.pfloor * (1.0 - 1e-9)) {
            U[4][q] = c.pfloor / (c.g - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * (bx * bx + by * by + bz * bz);
            c.nfloor += 1;
          }
          p = c.pfloor;
        }
        if (!(rho > 0.0) || !(p > 0.0)) c.status = ERR_UNPHYSICAL;
        c.V[0][q] = rho; c.V[1][q] = vx; c.V[2][q] = vy; c.V[3][q] = vz; c.V[4][q] = p;
        c.V[5][q] = bx; c.V[6][q] = by; c.V[7][q] = bz;
      }
  for (int n = 0; n < (c.mhd ? 8 : 5); ++n) fill_periodic(c, c.V[n]);
}

// a3+a4 / O3-O8: face states and Riemann flux on every face of direction d whose 4-cell stencil exists:
// index 0..n along d, and one transverse ghost layer (needed by the EMFs).
void sweep(Ctx& c, int d, const Arr Bf[3], bool want_flux) {
  const int a = d, b = (d + 1) % 3, e = (d + 2) % 3;
  int lo[3], hi[3];
  lo[a] = 0; hi[a] = c.n[a];
  lo[b] = -1; hi[b] = c.n[b];
  lo[e] = -1; hi[e] = c.n[e];
  if (c.emf == EMF_UCT_HLL || c.emf == EMF_UCT_HLLD) {  // the 2D EMFs reconstruct face quantities across two more transverse faces
    lo[b] = lo[e] = -NG;
    hi[b] = c.n[b] + NG - 1;
    hi[e] = c.n[e] + NG - 1;
  }
  const size_t sa = c.st[a];
  const Arr* q[7] = {&c.V[0], &c.V[1 + a], &c.V[1 + b], &c.V[1 + e], &c.V[4], &c.V[5 + b], &c.V[5 + e]};
  const int nq = c.mhd ? 7 : 5;
  int ijk[3];
  for (ijk[2] = lo[2]; ijk[2] <= hi[2]; ++ijk[2])
    for (ijk[1] = lo[1]; ijk[1] <= hi[1]; ++ijk[1])
      for (ijk[0] = lo[0]; ijk[0] <= hi[0]; ++ijk[0]) {
        const size_t i0 = c.at(ijk[0], ijk[1], ijk[2]);  // cell to the right of the face
        double WL[7] = {0, 0, 0, 0, 0, 0, 0}, WR[7] = {0, 0, 0, 0, 0, 0, 0};
        for (int n = 0; n < nq; ++n) {
          const double* v = q[n]->data();
          const double qm2 = v[i0 - 2 * sa], qm1 = v[i0 - sa], q0 = v[i0], qp1 = v[i0 + sa];
          double lo_unused, hi_unused;
          if (c.limiter == LIM_PPM) {  // five-cell stencils: cells i-3 .. i+1 and i-2 .. i+2
            const double sL[5] = {v[i0 - 3 * sa], qm2, qm1, q0, qp1}, sR[5] = {qm2, qm1, q0, qp1, v[i0 + 2 * sa]};
            ppm_faces(sL, lo_unused, WL[n]);
            ppm_faces(sR, WR[n], hi_unused);
            continue;
          }
          reconstruct(c.limiter, qm2, qm1, q0, c.dx, lo_unused, WL[n]);   // cell i-1 at its upper face
          reconstruct(c.limiter, qm1, q0, qp1, c.dx, WR[n], hi_unused);   // cell i at its lower face
        }
        const double Bn = c.mhd ? Bf[a][i0] : 0.0;  // G3: staggered value on both sides
        if (!(WL[0] > 0.0) || !(WR[0] > 0.0) || !(WL[4] > 0.0) || !(WR[4] > 0.0)) c.status = ERR_UNPHYSICAL;
        if (want_flux) {
          double F[7], cface;
          c.roe_fallbacks += riemann(c.solver, c.g, WL, WR, Bn, F, cface);
          for (int n = 0; n < 7; ++n) c.F[d][n][i0] = F[n];
          c.cf[d][i0] = cface;
          if (c.emf == EMF_UCT_HLL) {
            // G21 (Mignone & Del Zanna 2021, HLL case): with the Davis speeds of this face, alpha+ = max(0, S_R),
            // alpha- = max(0, -S_L); the face carries the HLL-weighted transverse velocities
            // (alpha+ v_t^L + alpha- v_t^R)/(alpha+ + alpha-), which is how v_t enters the HLL flux of the normal field
            double SL, SR;
            davis_speeds(WL, WR, Bn, c.g, SL, SR);
            const double ap = std::max(0.0, SR), am = std::max(0.0, -SL);
            c.Al[d][0][i0] = ap;
            c.Al[d][1][i0] = am;
            c.Vt[d][0][i0] = (ap * WL[2] + am * WR[2]) / (ap + am);
            c.Vt[d][1][i0] = (ap * WL[3] + am * WR[3]) / (ap + am);
          }
          if (c.emf == EMF_UCT_HLLD) {
            double co[5];
            hlld_uct_coeffs(WL, WR, Bn, c.g, co);
            for (int m = 0; m < 5; ++m) c.Hc[d][m][i0] = co[m];
          }
        } else {
          double SL, SR;
          davis_speeds(WL, WR, Bn, c.g, SL, SR);
          c.cf[d][i0] = std::max(std::fabs(SL), std::fabs(SR));
        }
      }
}

// a6 / O10: edge EMF E_c at (a-1/2, b-1/2) with (a,b,c) cyclic.
void edge_emf(Ctx& c, int comp) {
  const int a = (comp + 1) % 3, b = (comp + 2) % 3;
  const size_t ea = c.st[a], eb = c.st[b];
  int lo[3] = {0, 0, 0}, hi[3];
  hi[a] = c.n[a]; hi[b] = c.n[b]; hi[comp] = c.n[comp] - 1;
  // face-centred EMFs from the Riemann fluxes of B: E_c^(a) = -F_a[B_b] = -F[a][5]; E_c^(b) = +F_b[B_a] = +F[b][6]
  const double* Fa5 = c.F[a][5].data();
  const double* Fb6 = c.F[b][6].data();
  const double* Fa0 = c.F[a][0].data();
  const double* Fb0 = c.F[b][0].data();
  const double* va = c.V[1 + a].data();
  const double* vb = c.V[1 + b].data();
  const double* Ba = c.V[5 + a].data();
  const double* Bb = c.V[5 + b].data();
  auto Ea = [&](size_t P) { return -Fa5[P]; };
  auto Eb = [&](size_t P) { return Fb6[P]; };
  auto Ec = [&](size_t Q) { return vb[Q] * Ba[Q] - va[Q] * Bb[Q]; };  // -(v x B)_c at the cell centre (G10)
  auto upwind = [](double flux, double gm, double gp) {
    if (flux > 0.0) return gm;
    if (flux < 0.0) return gp;
    return 0.5 * (gm + gp);
  };
  int ijk[3];
  for (ijk[2] = lo[2]; ijk[2] <= hi[2]; ++ijk[2])
    for (ijk[1] = lo[1]; ijk[1] <= hi[1]; ++ijk[1])
      for (ijk[0] = lo[0]; ijk[0] <= hi[0]; ++ijk[0]) {
        const size_t P = c.at(ijk[0], ijk[1], ijk[2]);
        double e = 0.25 * (Ea(P) + Ea(P - eb) + Eb(P) + Eb(P - ea));
        if (c.emf == EMF_UCT_HLL) {
          // 2D HLL EMF (G21).  E_c = -(v_a B_b - v_b B_a) at the edge (a-1/2, b-1/2):
          //   E_c = -[al_a+ (v_a B_b)^W + al_a- (v_a B_b)^E - al_a+ al_a- (B_b^E - B_b^W)] / (al_a+ + al_a-)
          //         +[al_b+ (v_b B_a)^S + al_b- (v_b B_a)^N - al_b+ al_b- (B_a^N - B_a^S)] / (al_b+ + al_b-)
          // W/E: the staggered B_b and the face velocity v_a of the b-faces on either side of the edge, reconstructed
          // along a with the scheme's limiter; S/N likewise along b on the a-faces; al_a+- the larger of the two
          // a-faces that touch the edge (and al_b+- of the two b-faces).
          const double* Bb = c.Bstage[b].data();   // on b-faces
          const double* Ba = c.Bstage[a].data();   // on a-faces
          const double* va_f = c.Vt[b][1].data();  // v_a on b-faces (b-sweep local order: n = b, t1 = c, t2 = a)
          const double* vb_f = c.Vt[a][0].data();  // v_b on a-faces (a-sweep local order: n = a, t1 = b, t2 = c)
          double unused, BbW, BbE, vaW, vaE, BaS, BaN, vbS, vbN;
          reconstruct(c.limiter, Bb[P - 2 * ea], Bb[P - ea], Bb[P], c.dx, unused, BbW);
          reconstruct(c.limiter, Bb[P - ea], Bb[P], Bb[P + ea], c.dx, BbE, unused);
          reconstruct(c.limiter, va_f[P - 2 * ea], va_f[P - ea], va_f[P], c.dx, unused, vaW);
          reconstruct(c.limiter, va_f[P - ea], va_f[P], va_f[P + ea], c.dx, vaE, unused);
          reconstruct(c.limiter, Ba[P - 2 * eb], Ba[P - eb], Ba[P], c.dx, unused, BaS);
          reconstruct(c.limiter, Ba[P - eb], Ba[P], Ba[P + eb], c.dx, BaN, unused);
          reconstruct(c.limiter, vb_f[P - 2 * eb], vb_f[P - eb], vb_f[P], c.dx, unused, vbS);
          reconstruct(c.limiter, vb_f[P - eb], vb_f[P], vb_f[P + eb], c.dx, vbN, unused);
          const double aap = std::max(c.Al[a][0][P - eb], c.Al[a][0][P]), aam = std::max(c.Al[a][1][P - eb], c.Al[a][1][P]);
          const double abp = std::max(c.Al[b][0][P - ea], c.Al[b][0][P]), abm = std::max(c.Al[b][1][P - ea], c.Al[b][1][P]);
          const double term_a = (aap * vaW * BbW + aam * vaE * BbE - aap * aam * (BbE - BbW)) / (aap + aam);
          const double term_b = (abp * vbS * BaS + abm * vbN * BaN - abp * abm * (BaN - BaS)) / (abp + abm);
          e = -term_a + term_b;
        }
        if (c.emf == EMF_UCT_HLLD) {
          // 2D HLLD EMF (G24): the two transports of the 2D-HLL EMF with the coefficients of hlld_uct_coeffs,
          //   E_c = -[aL_a (v_a B_b)^W + aR_a (v_a B_b)^E - (dR_a B_b^E - dL_a B_b^W)]
          //         +[aL_b (v_b B_a)^S + aR_b (v_b B_a)^N - (dR_b B_a^N - dL_b B_a^S)]
          // W/E: staggered B_b and the effective velocity vbar_a of the b-faces on either side of the edge, reconstructed
          // along a; S/N likewise along b on the a-faces; coefficients: the mean of the two faces that touch the edge.
          const double* Bb = c.Bstage[b].data();
          const double* Ba = c.Bstage[a].data();
          const double* va_f = c.Hc[b][4].data();  // vbar_a on b-faces (b-sweep local order: n = b, t1 = c, t2 = a)
          const double* vb_f = c.Hc[a][3].data();  // vbar_b on a-faces (a-sweep local order: n = a, t1 = b, t2 = c)
          double unused, BbW, BbE, vaW, vaE, BaS, BaN, vbS, vbN;
          reconstruct(c.limiter, Bb[P - 2 * ea], Bb[P - ea], Bb[P], c.dx, unused, BbW);
          reconstruct(c.limiter, Bb[P - ea], Bb[P], Bb[P + ea], c.dx, BbE, unused);
          reconstruct(c.limiter, va_f[P - 2 * ea], va_f[P - ea], va_f[P], c.dx, unused, vaW);
          reconstruct(c.limiter, va_f[P - ea], va_f[P], va_f[P + ea], c.dx, vaE, unused);
          reconstruct(c.limiter, Ba[P - 2 * eb], Ba[P - eb], Ba[P], c.dx, unused, BaS);
          reconstruct(c.limiter, Ba[P - eb], Ba[P], Ba[P + eb], c.dx, BaN, unused);
          reconstruct(c.limiter, vb_f[P - 2 * eb], vb_f[P - eb], vb_f[P], c.dx, unused, vbS);
          reconstruct(c.limiter, vb_f[P - eb], vb_f[P], vb_f[P + eb], c.dx, vbN, unused);
          const double aLa = 0.5 * (c.Hc[a][0][P - eb] + c.Hc[a][0][P]), dLa = 0.5 * (c.Hc[a][1][P - eb] + c.Hc[a][1][P]);
          const double dRa = 0.5 * (c.Hc[a][2][P - eb] + c.Hc[a][2][P]);
          const double aLb = 0.5 * (c.Hc[b][0][P - ea] + c.Hc[b][0][P]), dLb = 0.5 * (c.Hc[b][1][P - ea] + c.Hc[b][1][P]);
          const double dRb = 0.5 * (c.Hc[b][2][P - ea] + c.Hc[b][2][P]);
          const double Ta = aLa * vaW * BbW + (1.0 - aLa) * vaE * BbE - (dRa * BbE - dLa * BbW);
          const double Tb = aLb * vbS * BaS + (1.0 - aLb) * vbN * BaN - (dRb * BaN - dLb * BaS);
          e = -Ta + Tb;
        }
        if (c.emf == EMF_UCT0) {
          // E^0 of Gardiner & Stone 2005: the E^c construction with the two candidate gradients
          // averaged instead of upwinded, which collapses to (1/2) sum of the four face values - (1/4) sum of the
          // four cell-centred reference values
          e = 0.5 * (Ea(P) + Ea(P - eb) + Eb(P) + Eb(P - ea)) - 0.25 * (Ec(P) + Ec(P - ea) + Ec(P - eb) + Ec(P - ea - eb));
        }
        if (c.emf == EMF_UCT) {
          // d/db at the a-face (ia-1/2): quarter points ib-1/4 (cells P-ea, P) and ib-3/4 (cells P-ea-eb, P-eb)
          const double gbp_m = 2.0 * (Ec(P - ea) - Eb(P - ea));          // g_b+ of cell P-ea
          const double gbp_p = 2.0 * (Ec(P) - Eb(P));                    // g_b+ of cell P
          const double gbm_m = 2.0 * (Eb(P - ea) - Ec(P - ea - eb));     // g_b- of cell P-ea-eb
          const double gbm_p = 2.0 * (Eb(P) - Ec(P - eb));               // g_b- of cell P-eb
          const double Gb_q1 = upwind(Fa0[P], gbp_m, gbp_p);             // (ia-1/2, ib-1/4)
          const double Gb_q3 = upwind(Fa0[P - eb], gbm_m, gbm_p);        // (ia-1/2, ib-3/4)
          // d/da at the b-face (ib-1/2): quarter points ia-1/4 (cells P-eb, P) and ia-3/4 (cells P-ea-eb, P-ea)
          const double gap_m = 2.0 * (Ec(P - eb) - Ea(P - eb));          // g_a+ of cell P-eb
          const double gap_p = 2.0 * (Ec(P) - Ea(P));                    // g_a+ of cell P
          const double gam_m = 2.0 * (Ea(P - eb) - Ec(P - ea - eb));     // g_a- of cell P-ea-eb
          const double gam_p = 2.0 * (Ea(P) - Ec(P - ea));               // g_a- of cell P-ea
          const double Ga_q1 = upwind(Fb0[P], gap_m, gap_p);             // (ia-1/4, ib-1/2)
          const double Ga_q3 = upwind(Fb0[P - ea], gam_m, gam_p);        // (ia-3/4, ib-1/2)
          e += 0.125 * (Gb_q3 - Gb_q1) + 0.125 * (Ga_q3 - Ga_q1);
        }
        c.E[comp][P] = e;
      }
}

// O2: U* = S_dt(U), Bf* = S_dt(Bf) (CT_FACE) or A* = S_dt(A) (CT_POTENTIAL).  `Uin`/`Bin` are modified only in
// their ghost zones.
void stage(Ctx& c, Arr Uin[5], Arr Bin[3], const Arr Ain[3], double dt, Arr Uout[5], Arr Bout[3], Arr Aout[3]) {
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  for (int n = 0; n < 5; ++n) fill_periodic(c, Uin[n]);
  if (c.mhd)
    for (int n = 0; n < 3; ++n) fill_periodic(c, Bin[n]);
  compute_prims(c, Uin, Bin);
  c.Bstage = Bin;
  for (int d = 0; d < 3; ++d) sweep(c, d, Bin, true);
  // a5 / Eq. 5: flux divergence; local flux ordering (rho, m_n, m_t1, m_t2, E) -> global momentum
  const double dtdx = dt / c.dx;
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        const size_t q = c.at(i, j, k);
        double div[5] = {0, 0, 0, 0, 0};
        for (int d = 0; d < 3; ++d) {
          const int a = d, b = (d + 1) % 3, e = (d + 2) % 3;
          const size_t s = c.st[d];
          div[0] += c.F[d][0][q + s] - c.F[d][0][q];
          div[1 + a] += c.F[d][1][q + s] - c.F[d][1][q];
          div[1 + b] += c.F[d][2][q + s] - c.F[d][2][q];
          div[1 + e] += c.F[d][3][q + s] - c.F[d][3][q];
          div[4] += c.F[d][4][q + s] - c.F[d][4][q];
        }
        for (int n = 0; n < 5; ++n) Uout[n][q] = Uin[n][q] - dtdx * div[n];
      }
  if (!c.mhd) return;
  for (int comp = 0; comp < 3; ++comp) edge_emf(c, comp);
  if (c.ct_form == CT_POTENTIAL) {
    // Eq. 7: dA/dt = -E on every edge where E was evaluated (the lattice of the active faces)
    for (int comp = 0; comp < 3; ++comp) {
      int hi[3] = {c.n[0], c.n[1], c.n[2]};
      hi[comp] = c.n[comp] - 1;
      for (int k = 0; k <= hi[2]; ++k)
        for (int j = 0; j <= hi[1]; ++j)
          for (int i = 0; i <= hi[0]; ++i) {
            const size_t q = c.at(i, j, k);
            Aout[comp][q] = Ain[comp][q] - dt * c.E[comp][q];
          }
    }
    return;
  }
  // a7 / O11 / Eq. 6: discrete Stokes theorem on each face
  const size_t sx = c.st[0], sy = c.st[1], sz = c.st[2];
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        const size_t q = c.at(i, j, k);
        Bout[0][q] = Bin[0][q] - dtdx * ((c.E[2][q + sy] - c.E[2][q]) - (c.E[1][q + sz] - c.E[1][q]));
        Bout[1][q] = Bin[1][q] - dtdx * ((c.E[0][q + sz] - c.E[0][q]) - (c.E[2][q + sx] - c.E[2][q]));
        Bout[2][q] = Bin[2][q] - dtdx * ((c.E[1][q + sx] - c.E[1][q]) - (c.E[0][q + sy] - c.E[0][q]));
      }
}

// a9 / O9 / Eq. 10: dt = cfl / max_cells sum_d c_d/dx, c_d = max over the cell's two faces (G8).
double compute_dt(Ctx& c, double cfl) {
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  for (int n = 0; n < 5; ++n) fill_periodic(c, c.U[n]);
  if (c.mhd)
    for (int n = 0; n < 3; ++n) fill_periodic(c, c.Bf[n]);
  compute_prims(c, c.U, c.Bf);
  for (int d = 0; d < 3; ++d) sweep(c, d, c.Bf, false);
  double mx = 0.0;
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        const size_t q = c.at(i, j, k);
        double s = 0.0;
        for (int d = 0; d < 3; ++d) s += std::max(c.cf[d][q], c.cf[d][q + c.st[d]]);
        mx = std::max(mx, s / c.dx);
      }
  return cfl / mx;
}

// Eq. 8 with the gauge of G19: Bf = Bref + curl A on the active faces (same differences as Eq. 6).
void field_from_potential(const Ctx& c, const Arr A[3], Arr Bout[3]) {
  const size_t sx = c.st[0], sy = c.st[1], sz = c.st[2];
  for (int k = 0; k < c.n[2]; ++k)
    for (int j = 0; j < c.n[1]; ++j)
      for (int i = 0; i < c.n[0]; ++i) {
        const size_t q = c.at(i, j, k);
        Bout[0][q] = c.Bref[0][q] + ((A[2][q + sy] - A[2][q]) - (A[1][q + sz] - A[1][q])) / c.dx;
        Bout[1][q] = c.Bref[1][q] + ((A[0][q + sz] - A[0][q]) - (A[2][q + sx] - A[2][q])) / c.dx;
        Bout[2][q] = c.Bref[2][q] + ((A[1][q + sx] - A[1][q]) - (A[0][q + sy] - A[0][q])) / c.dx;
      }
}

// a8 / O12 / Eq. 9 with Tab. 1: U_s = w_s S_dt(U_{s-1}) + w_s^0 U_0.
//   Euler: w1 = 1, w1^0 = 0.   RK2: + w2 = w2^0 = 1/2.   RK3: w2 = 1/4, w2^0 = 3/4, w3 = 2/3, w3^0 = 1/3.
void step(Ctx& c, double dt) {
  static const double W[3][3] = {{1.0, 0.0, 0.0}, {1.0, 0.5, 0.0}, {1.0, 0.25, 2.0 / 3.0}};
  static const double W0[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.5, 0.0}, {0.0, 0.75, 1.0 / 3.0}};
  const int nb = c.mhd ? 3 : 0;
  const bool pot = c.mhd && c.ct_form == CT_POTENTIAL;
  for (int n = 0; n < 5; ++n) c.U0[n] = c.U[n];
  for (int n = 0; n < nb; ++n) c.Bf0[n] = c.Bf[n];
  if (pot)
    for (int n = 0; n < 3; ++n) c.A0[n] = c.A[n];
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  for (int s = 0; s < c.nstages; ++s) {
    const double w = W[c.nstages - 1][s], w0 = W0[c.nstages - 1][s];
    const bool last = s == c.nstages - 1;
    Arr* Uin = s == 0 ? c.U0 : c.U1;
    Arr* Bin = s == 0 ? c.Bf0 : c.Bf1;
    stage(c, Uin, Bin, c.A, dt, c.Us, c.Bfs, c.As);
    Arr* Unew = last ? c.U : c.U1;
    Arr* Bnew = last ? c.Bf : c.Bf1;
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          const size_t q = c.at(i, j, k);
          for (int n = 0; n < 5; ++n) Unew[n][q] = w0 == 0.0 ? c.Us[n][q] : w0 * c.U0[n][q] + w * c.Us[n][q];
          if (!pot)
            for (int n = 0; n < nb; ++n) Bnew[n][q] = w0 == 0.0 ? c.Bfs[n][q] : w0 * c.Bf0[n][q] + w * c.Bfs[n][q];
        }
    if (pot) {
      for (int n = 0; n < 3; ++n)
        for (size_t q = 0; q < c.N; ++q) c.A[n][q] = w0 == 0.0 ? c.As[n][q] : w0 * c.A0[n][q] + w * c.As[n][q];
      field_from_potential(c, c.A, Bnew);
    }
  }
  if (c.pfloor > 0.0) {  // G20: the floor belongs to the cons->prim conversion of the result, so the state a cycle
    for (int n = 0; n < nb; ++n) fill_periodic(c, c.Bf[n]);  // leaves behind is already fixed
    compute_prims(c, c.U, c.Bf);
  }
  c.last_dt = dt;
  c.t += dt;
}

}  // namespace

// =============================================================================================
// C ABI (host pointers everywhere).  Layouts as in include/idfx.h: [var][nz][ny][nx], x fastest;
// bface[d][k][j][i] is the d-component on the LEFT d-face of cell (i,j,k).
// =============================================================================================
struct idfxref_ctx {
  Ctx c;
};

IDFXREF_API idfxref_ctx* idfxref_create(int nx, int ny, int nz, double dx, double gamma, int solver,
                                        int limiter, int emf_mode) {
  if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0.0) || !(gamma > 1.0)) return nullptr;
  if (solver < 0 || solver > 4 || limiter < 0 || limiter > 4 || emf_mode < 0 || emf_mode > 5) return nullptr;
  if (limiter == LIM_PPM && (emf_mode == EMF_UCT_HLL || emf_mode == EMF_UCT_HLLD)) return nullptr;  // the 2D EMFs reconstruct with 3-cell stencils only
  if (emf_mode == EMF_UCT_HLLD && solver != SOLVER_HLLD) return nullptr;  // its coefficients are those of the HLLD face solve
  const bool mhd = emf_mode != EMF_NONE;
  if (mhd && solver == SOLVER_HLLC) return nullptr;
  if (!mhd && solver == SOLVER_HLLD) return nullptr;
  idfxref_ctx* h = new idfxref_ctx;
  Ctx& c = h->c;
  c.n[0] = nx; c.n[1] = ny; c.n[2] = nz;
  c.dx = dx; c.g = gamma; c.solver = solver; c.limiter = limiter; c.emf = emf_mode; c.mhd = mhd;
  for (int d = 0; d < 3; ++d) c.p[d] = c.n[d] + 2 * NG;
  c.st[0] = 1; c.st[1] = (size_t)c.p[0]; c.st[2] = (size_t)c.p[0] * c.p[1];
  c.N = c.st[2] * c.p[2];
  for (int n = 0; n < 5; ++n) {
    c.U[n].assign(c.N, 0.0); c.U0[n].assign(c.N, 0.0); c.U1[n].assign(c.N, 0.0); c.Us[n].assign(c.N, 0.0);
  }
  for (int n = 0; n < 8; ++n) c.V[n].assign(c.N, 0.0);
  for (int d = 0; d < 3; ++d) {
    c.Bf[d].assign(c.N, 0.0); c.Bf0[d].assign(c.N, 0.0); c.Bf1[d].assign(c.N, 0.0); c.Bfs[d].assign(c.N, 0.0);
    for (int n = 0; n < 7; ++n) c.F[d][n].assign(c.N, 0.0);
    c.cf[d].assign(c.N, 0.0);
    c.E[d].assign(c.N, 0.0);
    if (emf_mode == EMF_UCT_HLLD)
      for (int m = 0; m < 5; ++m) c.Hc[d][m].assign(c.N, 0.0);
    if (emf_mode == EMF_UCT_HLL)
      for (int m = 0; m < 2; ++m) {
        c.Vt[d][m].assign(c.N, 0.0);
        c.Al[d][m].assign(c.N, 0.0);
      }
  }
  c.Bstage = nullptr;
  c.nstages = 2; c.ct_form = CT_FACE; c.t = 0.0; c.pfloor = 0.0; c.nfloor = 0; c.outflow = 0;
  c.last_dt = 0.0; c.status = OK; c.roe_fallbacks = 0;
  return h;
}

IDFXREF_API void idfxref_destroy(idfxref_ctx* h) { delete h; }

// Options beyond the create() arguments; call before set_state.  OPT_INTEGRATOR: number of stages 1..3 (Tab. 1);
// OPT_CT_FORM: CT_FACE (Eq. 6) or CT_POTENTIAL (Eq. 7-8).
IDFXREF_API int idfxref_set_option(idfxref_ctx* h, int option, int value) {
  if (!h) return ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (option == OPT_INTEGRATOR && value >= 1 && value <= 3) {
    c.nstages = value;
    return OK;
  }
  if (option == OPT_BOUNDARY && (value == 0 || value == 1)) {
    // with a magnetic field: face CT, three-cell reconstructions and the face-flux EMFs only (the 2D-HLL EMF and PPM reach
    // further into the ghost zones, the vector potential has no zero-gradient form)
    if (value == 1 && c.mhd && (c.emf == EMF_UCT_HLL || c.emf == EMF_UCT_HLLD || c.limiter == LIM_PPM || c.ct_form == CT_POTENTIAL)) return ERR_UNSUPPORTED;
    c.outflow = value;
    return OK;
  }
  if (option == OPT_CT_FORM && (value == CT_FACE || (value == CT_POTENTIAL && c.mhd && !c.outflow))) {
    c.ct_form = value;
    if (value == CT_POTENTIAL)
      for (int d = 0; d < 3; ++d) {
        c.A[d].assign(c.N, 0.0); c.A0[d].assign(c.N, 0.0); c.As[d].assign(c.N, 0.0); c.Bref[d].assign(c.N, 0.0);
      }
    return OK;
  }
  return ERR_INVALID_ARG;
}

// O1 set_state: Bc from faces, then U from prims.
IDFXREF_API int idfxref_set_state(idfxref_ctx* h, const double* prim, const double* bface) {
  if (!h || !prim) return ERR_INVALID_ARG;
  Ctx& c = h->c;
  if (c.mhd && !bface) return ERR_INVALID_ARG;
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  const size_t nc = (size_t)nx * ny * nz;
  if (c.mhd) {
    for (int d = 0; d < 3; ++d) {
      for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
          for (int i = 0; i < nx; ++i) c.Bf[d][c.at(i, j, k)] = bface[d * nc + ((size_t)k * ny + j) * nx + i];
      fill_periodic(c, c.Bf[d]);
      if (c.ct_form == CT_POTENTIAL) {  // G19: the potential is counted from this state on
        c.Bref[d] = c.Bf[d];
        std::fill(c.A[d].begin(), c.A[d].end(), 0.0);
      }
    }
  }
  c.t = 0.0;
  c.nfloor = 0;
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        const size_t q = c.at(i, j, k), s = ((size_t)k * ny + j) * nx + i;
        double bx = 0, by = 0, bz = 0;
        if (c.mhd) {
          bx = 0.5 * (c.Bf[0][q] + c.Bf[0][q + c.st[0]]);
          by = 0.5 * (c.Bf[1][q] + c.Bf[1][q + c.st[1]]);
          bz = 0.5 * (c.Bf[2][q] + c.Bf[2][q + c.st[2]]);
        }
        const double rho = prim[0 * nc + s], vx = prim[1 * nc + s], vy = prim[2 * nc + s], vz = prim[3 * nc + s],
                     p = prim[4 * nc + s];
        if (!(rho > 0.0) || !(p > 0.0)) c.status = ERR_UNPHYSICAL;
        c.U[0][q] = rho; c.U[1][q] = rho * vx; c.U[2][q] = rho * vy; c.U[3][q] = rho * vz;
        c.U[4][q] = p / (c.g - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * (bx * bx + by * by + bz * bz);
      }
  return OK;
}

IDFXREF_API int idfxref_get_conserved(idfxref_ctx* h, double* cons, double* bface) {
  if (!h || !cons) return ERR_INVALID_ARG;
  Ctx& c = h->c;
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  const size_t nc = (size_t)nx * ny * nz;
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        const size_t q = c.at(i, j, k), s = ((size_t)k * ny + j) * nx + i;
        for (int n = 0; n < 5; ++n) cons[n * nc + s] = c.U[n][q];
        if (c.mhd && bface)
          for (int d = 0; d < 3; ++d) bface[d * nc + s] = c.Bf[d][q];
      }
  return OK;
}

IDFXREF_API int idfxref_get_state(idfxref_ctx* h, double* prim, double* bface) {
  if (!h || !prim) return ERR_INVALID_ARG;
  Ctx& c = h->c;
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  const size_t nc = (size_t)nx * ny * nz;
  if (c.mhd)
    for (int d = 0; d < 3; ++d) fill_periodic(c, c.Bf[d]);
  compute_prims(c, c.U, c.Bf);
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        const size_t q = c.at(i, j, k), s = ((size_t)k * ny + j) * nx + i;
        for (int n = 0; n < 5; ++n) prim[n * nc + s] = c.V[n][q];
        if (c.mhd && bface)
          for (int d = 0; d < 3; ++d) bface[d * nc + s] = c.Bf[d][q];
      }
  return OK;
}

IDFXREF_API int idfxref_compute_dt(idfxref_ctx* h, double cfl, double* dt_out) {
  if (!h || !dt_out || !(cfl > 0.0) || !(cfl < 1.0)) return ERR_INVALID_ARG;
  *dt_out = compute_dt(h->c, cfl);
  return h->c.status;
}

IDFXREF_API int idfxref_step(idfxref_ctx* h, double dt) {
  if (!h || !(dt > 0.0)) return ERR_INVALID_ARG;
  step(h->c, dt);
  return h->c.status;
}

// G9: advance = nsteps x { dt = compute_dt(cfl); step(dt) }, dt evaluated on the current state each time.
IDFXREF_API int idfxref_advance(idfxref_ctx* h, int nsteps, double cfl) {
  if (!h || nsteps < 0 || !(cfl > 0.0) || !(cfl < 1.0)) return ERR_INVALID_ARG;
  for (int s = 0; s < nsteps; ++s) step(h->c, compute_dt(h->c, cfl));
  return h->c.status;
}

IDFXREF_API int idfxref_set_option_real(idfxref_ctx* h, int option, double value) {
  if (!h || option != OPT_PRESSURE_FLOOR || !(value >= 0.0)) return ERR_INVALID_ARG;
  h->c.pfloor = value;
  return OK;
}

IDFXREF_API long long idfxref_floor_count(const idfxref_ctx* h) { return h ? h->c.nfloor : -1; }

// Cycles with the CFL step until t_end: a step that would reach or pass t_end is shortened to land on it.
IDFXREF_API int idfxref_advance_to(idfxref_ctx* h, double t_end, double cfl, int max_steps, int* nsteps_out) {
  if (!h || max_steps < 0 || !(cfl > 0.0) || !(cfl < 1.0)) return ERR_INVALID_ARG;
  Ctx& c = h->c;
  int n = 0;
  while (c.t < t_end && n < max_steps) {
    double dt = compute_dt(c, cfl);
    const double remaining = t_end - c.t;
    const bool lands = dt >= remaining;
    if (lands) dt = remaining;
    step(c, dt);
    if (lands) c.t = t_end;
    ++n;
  }
  if (nsteps_out) *nsteps_out = n;
  return c.status;
}

IDFXREF_API int idfxref_time(const idfxref_ctx* h, double* t_out) {
  if (!h || !t_out) return ERR_INVALID_ARG;
  *t_out = h->c.t;
  return OK;
}

// Edge potential accumulated since set_state (CT_POTENTIAL), layout as idfxref_get_emf.
IDFXREF_API int idfxref_get_potential(const idfxref_ctx* h, double* pot) {
  if (!h || !pot || h->c.ct_form != CT_POTENTIAL) return ERR_INVALID_ARG;
  const Ctx& c = h->c;
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  const size_t nc = (size_t)nx * ny * nz;
  for (int comp = 0; comp < 3; ++comp)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) pot[comp * nc + ((size_t)k * ny + j) * nx + i] = c.A[comp][c.at(i, j, k)];
  return OK;
}

// Point-wise S2 for the pins: values of cell i's reconstruction at its lower and upper faces.
IDFXREF_API void idfxref_reconstruct(int limiter, double qm, double q0, double qp, double dx, double* lower,
                                     double* upper) {
  reconstruct(limiter, qm, q0, qp, dx, *lower, *upper);
}

// Point-wise PPM for the pins: a[0..4] = a_{j-2} .. a_{j+2}.
IDFXREF_API void idfxref_ppm_faces(const double* a, double* lower, double* upper) { ppm_faces(a, *lower, *upper); }

IDFXREF_API int idfxref_last_dt(const idfxref_ctx* h, double* dt_out) {
  if (!h || !dt_out) return ERR_INVALID_ARG;
  *dt_out = h->c.last_dt;
  return OK;
}

IDFXREF_API int idfxref_status(const idfxref_ctx* h) { return h ? h->c.status : ERR_INVALID_ARG; }
IDFXREF_API long long idfxref_roe_fallbacks(const idfxref_ctx* h) { return h ? h->c.roe_fallbacks : -1; }

// Edge EMFs of the most recent stage, emf[c][k][j][i] = E_c at the lower edges of cell (i,j,k)
// (E_x at (i, j-1/2, k-1/2), E_y at (i-1/2, j, k-1/2), E_z at (i-1/2, j-1/2, k)).
IDFXREF_API int idfxref_get_emf(const idfxref_ctx* h, double* emf) {
  if (!h || !emf) return ERR_INVALID_ARG;
  const Ctx& c = h->c;
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  const size_t nc = (size_t)nx * ny * nz;
  for (int comp = 0; comp < 3; ++comp)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) emf[comp * nc + ((size_t)k * ny + j) * nx + i] = c.E[comp][c.at(i, j, k)];
  return OK;
}

// Face fluxes of the most recent stage in direction d, flux[n][k][j][i] on the LEFT d-face of cell (i,j,k),
// local ordering n = (rho, m_n, m_t1, m_t2, E, B_t1, B_t2); cface likewise.
IDFXREF_API int idfxref_get_flux(const idfxref_ctx* h, int d, double* flux, double* cface) {
  if (!h || d < 0 || d > 2) return ERR_INVALID_ARG;
  const Ctx& c = h->c;
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  const size_t nc = (size_t)nx * ny * nz;
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        const size_t q = c.at(i, j, k), s = ((size_t)k * ny + j) * nx + i;
        if (flux)
          for (int n = 0; n < 7; ++n) flux[n * nc + s] = c.F[d][n][q];
        if (cface) cface[s] = c.cf[d][q];
      }
  return OK;
}

// ---- point-wise entry points used only by the pins --------------------------------------------
IDFXREF_API void idfxref_cons_from_prim(double gamma, const double* W, double Bn, double* U) {
  cons_from_prim(W, Bn, gamma, U);
}
IDFXREF_API void idfxref_phys_flux(double gamma, const double* W, double Bn, double* F) {
  double U[7];
  cons_from_prim(W, Bn, gamma, U);
  phys_flux(W, Bn, U, F);
}
// Flux as a function of the conserved vector (for finite-difference Jacobians).
IDFXREF_API void idfxref_flux_from_cons(double gamma, const double* U, double Bn, double* F) {
  double W[7];
  W[0] = U[0]; W[1] = U[1] / U[0]; W[2] = U[2] / U[0]; W[3] = U[3] / U[0];
  W[5] = U[5]; W[6] = U[6];
  W[4] = (gamma - 1.0) * (U[4] - 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / U[0] -
                          0.5 * (Bn * Bn + U[5] * U[5] + U[6] * U[6]));
  phys_flux(W, Bn, U, F);
}
IDFXREF_API int idfxref_riemann(int solver, double gamma, const double* WL, const double* WR, double Bn,
                                double* F, double* cface) {
  return riemann(solver, gamma, WL, WR, Bn, F, *cface);
}
// out[5] = (a_L, d_L, d_R, vbar_t1, vbar_t2) of the 2D-HLLD EMF (G24)
IDFXREF_API void idfxref_hlld_uct_coeffs(double gamma, const double* WL, const double* WR, double Bn, double* out) {
  hlld_uct_coeffs(WL, WR, Bn, gamma, out);
}
IDFXREF_API void idfxref_wave_speeds(double gamma, const double* WL, const double* WR, double Bn, double* SL,
                                     double* SR) {
  davis_speeds(WL, WR, Bn, gamma, *SL, *SR);
}
IDFXREF_API double idfxref_slope(int limiter, double dm, double dp) { return slope(limiter, dm, dp); }
// speeds[3] = (S_L, S*, S_R); states[2][5] = (U*_L, U*_R)
IDFXREF_API void idfxref_hllc_fan(double gamma, const double* WL, const double* WR, double* speeds,
                                  double* states) {
  double UL[7], UR[7], SL, SR;
  cons_from_prim(WL, 0.0, gamma, UL);
  cons_from_prim(WR, 0.0, gamma, UR);
  davis_speeds(WL, WR, 0.0, gamma, SL, SR);
  HllcFan f;
  hllc_fan(WL, WR, UL, UR, SL, SR, f);
  speeds[0] = f.SL; speeds[1] = f.SS; speeds[2] = f.SR;
  for (int n = 0; n < 5; ++n) { states[n] = f.UsL[n]; states[5 + n] = f.UsR[n]; }
}
// speeds[5] = (S_L, S*_L, S_M, S*_R, S_R); states[4][7] = (U*_L, U**_L, U**_R, U*_R)
IDFXREF_API void idfxref_hlld_fan(double gamma, const double* WL, const double* WR, double Bn, double* speeds,
                                  double* states) {
  double UL[7], UR[7], SL, SR;
  cons_from_prim(WL, Bn, gamma, UL);
  cons_from_prim(WR, Bn, gamma, UR);
  davis_speeds(WL, WR, Bn, gamma, SL, SR);
  HlldFan f;
  hlld_fan(WL, WR, Bn, UL, UR, SL, SR, f);
  speeds[0] = f.SL; speeds[1] = f.SsL; speeds[2] = f.SM; speeds[3] = f.SsR; speeds[4] = f.SR;
  for (int n = 0; n < 7; ++n) {
    states[n] = f.UsL[n]; states[7 + n] = f.UssL[n]; states[14 + n] = f.UssR[n]; states[21 + n] = f.UsR[n];
  }
}
// lam[7]; Rc[7][7] with Rc[k][:] the k-th right eigenvector in CONSERVED variables (M r_k);
// Lc[7][7] with Lc[k][:] the k-th left eigenvector in conserved variables (l_k Minv).  Returns 0 if a~^2 <= 0.
IDFXREF_API int idfxref_roe_system(double gamma, const double* WL, const double* WR, double Bn, double* lam,
                                   double* Rc, double* Lc) {
  double UL[7], UR[7];
  cons_from_prim(WL, Bn, gamma, UL);
  cons_from_prim(WR, Bn, gamma, UR);
  RoeSys s;
  if (!roe_system(WL, WR, Bn, UL, UR, gamma, s)) return 0;
  for (int k = 0; k < 7; ++k) {
    lam[k] = s.lam[k];
    for (int n = 0; n < 7; ++n) {
      double r = 0.0, l = 0.0;
      for (int m = 0; m < 7; ++m) {
        r += s.M[n][m] * s.R[k][m];
        l += s.L[k][m] * s.Minv[m][n];
      }
      Rc[k * 7 + n] = r;
      Lc[k * 7 + n] = l;
    }
  }
  return 1;
}
