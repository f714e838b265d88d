// flux_march.cuh — the hot kernels: reconstruct -> Riemann -> flux (a3 + a4) fused with the flux divergence
// (a5) and the CFL reduction (a9), one launch per direction.  DESIGN.md "Kernels".
//
// The path is bound by fp64 issue, not by HBM, so the design goal is that every limited
// slope and every Riemann problem is computed exactly once and that no warp waits on a global load:
//   * y and z: one thread per pencil, marching along the sweep direction with the three-cell stencil, the left
//     face state and the previous face flux carried in registers; threads of a warp are adjacent in x, so all
//     loads/stores are coalesced 256-byte rows; the next plane is prefetched one iteration ahead;
//   * x: one lane per cell of a 32-cell window (31 faces), neighbour states exchanged with warp shuffles; each
//     warp marches over rows with the next row prefetched.
// The x kernel stores its face fluxes; the y kernel turns them into the divergence together with its own; the
// z kernel adds its part and (stage 1) reduces max_cells sum_d c_d/dx: warp shuffle -> block -> atomicMax.
#pragma once
#include "common.cuh"
#include "physics.cuh"

#ifndef IDFX_MINB_X
#define IDFX_MINB_X 3
#endif
#ifndef IDFX_MINB_M
#define IDFX_MINB_M 2
#endif

namespace idfx {

struct FluxXArgs {
  const double* q[7];  // rho, vx, vy, vz, p, Bc_y, Bc_z
  const double* bn;    // B_x on x-faces
  double* FH[5];       // F_x of (rho, mx, my, mz, E) on faces 0..nx (face nx is written too)
  double* FB[2];       // F_x[B_y], F_x[B_z]
  double* cf;          // c_face (stage 1 only, else null)
  signed char* sg;     // sign of the mass flux (upwind-contact EMF only, else null)
  int rows_per_warp;
};

// lane l of a warp owns cell ci = f0 - 1 + l of one row; lanes 1..31 solve the left face of their cell.
template <int SOLVER, int LIM, bool MHD>
__global__ void __launch_bounds__(128, IDFX_MINB_X) k_flux_x(Geom g, FluxXArgs a) {
  constexpr int NQ = MHD ? 7 : 5;
  const double dx2 = g.dx * g.dx;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int f0 = 31 * blockIdx.x;
  const int ci = f0 - 1 + lane;
  const int nrows = g.ny * g.nz;
  // The trip count comes from a kernel argument, so it is uniform as far as the compiler can prove, and no lane leaves
  // the loop early: the warp shuffles below then compile to plain SHFL (with a per-warp row range they were wrapped in
  // WARPSYNC.COLLECTIVE / ENDCOLLECTIVE pairs, 84 instructions per row).  Rows past the end are clamped and not stored.
  const int rbase = (blockIdx.y * 4 + warp) * a.rows_per_warp;
  const int cl = min(ci, g.nx + 1);               // clamp the load column into the padded row
  const int ce = lane == 0 ? ci - 1 : min(ci + 1, g.nx + 1);  // edge lanes fetch the neighbour outside the window
  const bool edge = lane == 0 || lane == 31;
  const bool solve = lane >= 1 && ci <= g.nx;

  double qn[7], qen[7], bnn = 0.0;  // next row (prefetched)
  auto fetch = [&](int row) {
    row = min(row, nrows - 1);
    const int j = row % g.ny, k = row / g.ny;
    const long long c = g.at(cl, j, k);
#pragma unroll
    for (int n = 0; n < NQ; ++n) qn[n] = a.q[n][c];
    if (MHD) bnn = a.bn[c];
    if (edge) {
      const long long e = g.at(ce, j, k);
#pragma unroll
      for (int n = 0; n < NQ; ++n) qen[n] = a.q[n][e];
    }
  };
#ifndef IDFX_X_PF_L1
#define IDFX_X_PF_L1 0   // 1: the next row is prefetched into L1 (no registers) instead of into registers
#endif
  if (!IDFX_X_PF_L1) fetch(rbase);
  for (int it = 0; it < a.rows_per_warp; ++it) {
    const int r = rbase + it;
    const bool rowok = r < nrows;
    const int rr = min(r, nrows - 1);
    if (IDFX_X_PF_L1) {
      fetch(r);
      if (it + 1 < a.rows_per_warp) {
        const int rn = min(r + 1, nrows - 1);
        const long long cn = g.at(cl, rn % g.ny, rn / g.ny);
#pragma unroll
        for (int n = 0; n < NQ; ++n) prefetch_l1(a.q[n] + cn);
        if (MHD) prefetch_l1(a.bn + cn);
      }
    }
    double q[7], qe[7], Bn = bnn;
#pragma unroll
    for (int n = 0; n < NQ; ++n) {
      q[n] = qn[n];
      qe[n] = qen[n];
    }
    const long long c = g.at(cl, rr % g.ny, rr / g.ny);
    if (!IDFX_X_PF_L1 && it + 1 < a.rows_per_warp) fetch(r + 1);
    double WL[7], WR[7];
#pragma unroll
    for (int n = 0; n < NQ; ++n) {
      double qm = __shfl_up_sync(0xffffffffu, q[n], 1);
      double qp = __shfl_down_sync(0xffffffffu, q[n], 1);
      if (lane == 0) qm = qe[n];
      if (lane == 31) qp = qe[n];
      double up;
      face_values<LIM>(q[n], q[n] - qm, qp - q[n], dx2, WR[n], up);
      WL[n] = __shfl_up_sync(0xffffffffu, up, 1);
    }
    if (!MHD) WL[5] = WL[6] = WR[5] = WR[6] = 0.0;
    if (solve && rowok) {
      double F[7];
      const double cface = riemann<SOLVER, MHD>(WL, WR, MHD ? Bn : 0.0, g.gamma, F);
#pragma unroll
      for (int n = 0; n < 5; ++n) a.FH[n][c] = F[n];
      if (MHD) {
        a.FB[0][c] = F[5];
        a.FB[1][c] = F[6];
      }
      if (a.cf) a.cf[c] = cface;  // only the dt evaluation of stage 1 reads it
      if (a.sg) a.sg[c] = flux_sign(F[0]);
    }
  }
}

struct FluxMArgs {
  const double* q[7];   // primitives permuted for the sweep: rho, u, v, w, p, B_t1, B_t2
  const double* bn;     // normal field on the sweep faces
  long long sd, st;     // strides along the sweep and along the transverse (non-x) direction
  int ns, nt;           // active cells along the sweep / transverse direction
  int chunk;            // sweep cells per thread
  const double* FX[5];  // DIR = 1: x-face fluxes (faces 0..nx) and c_face of the x sweep
  const double* cfx;
  double* R[5];         // flux divergence, global ordering (rho, mx, my, mz, E)
  double* csum;         // sum_d c_d of the cell, accumulated over x and y
  double* FB[2];        // face fluxes of B_t1, B_t2
  signed char* SG;      // sign of the face mass flux (upwind-contact EMF only)
  DevScalars* sc;
};

// DIR = 1: y sweep, R = dF_x + dF_y (and csum = c_x + c_y).  DIR = 2: z sweep, R += dF_z (and the dt reduction).
template <int SOLVER, int LIM, bool MHD, int DIR, bool WANT_DT, bool WANT_FM>
__global__ void __launch_bounds__(128, IDFX_MINB_M) k_flux_march(Geom g, FluxMArgs a) {
  constexpr int NQ = MHD ? 7 : 5;
  const double dx2 = g.dx * g.dx;
  // local momentum components (n, t1, t2) -> global slot in R
  constexpr int PN = 1 + DIR, PT1 = 1 + (DIR + 1) % 3, PT2 = 1 + (DIR + 2) % 3;
  const int i = blockIdx.x * 32 + (threadIdx.x & 31);
  const int t = blockIdx.y * 4 + (threadIdx.x >> 5);
  const int s0 = blockIdx.z * a.chunk;
  const int s1 = min(s0 + a.chunk, a.ns);
  const bool active = i < g.nx && t < a.nt && s0 < s1;
  double smax = 0.0;
  if (active) {
    const long long sd = a.sd;
    long long c = g.at(i, 0, 0) + (long long)t * a.st + (long long)(s0 - 2) * sd;  // cell s0-2
    double dm[7], q0[7], qp[7], WL[7];  // dm = q(s) - q(s-1): the forward difference of the previous cell
#pragma unroll
    for (int n = 0; n < NQ; ++n) {
      const double qm = a.q[n][c];
      const double qc = a.q[n][c + sd];
      q0[n] = a.q[n][c + 2 * sd];
      dm[n] = q0[n] - qc;
      double lo_unused;
      face_values<LIM>(qc, qc - qm, dm[n], dx2, lo_unused, WL[n]);  // cell s0-1 at its upper face
    }
    c += 2 * sd;  // cell s0 = right cell of face s0
#pragma unroll
    for (int n = 0; n < NQ; ++n) qp[n] = a.q[n][c + sd];
    double Bn = MHD ? a.bn[c] : 0.0;
    if (!MHD) WL[5] = WL[6] = 0.0;
    double Fp[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, cfp = 0.0;

    for (int s = s0; s <= s1; ++s, c += sd) {
      // ---- loads for the next iteration and for the cell update at the bottom, issued before the solve ----
      double qn[7], Bnn = 0.0;
      if (s < s1) {
#pragma unroll
        for (int n = 0; n < NQ; ++n) qn[n] = a.q[n][c + 2 * sd];
        if (MHD) Bnn = a.bn[c + sd];
      }
      const long long cu = c - sd;  // cell s-1, completed by this face
      if (s + 1 < s1) {  // lines of the iteration after next, and of the next cell update, into L1
#pragma unroll
        for (int n = 0; n < NQ; ++n) prefetch_l1(a.q[n] + c + 3 * sd);
        if (MHD) prefetch_l1(a.bn + c + 2 * sd);
#pragma unroll
        for (int n = 0; n < 5; ++n) prefetch_l1(DIR == 1 ? a.FX[n] + c + 1 : a.R[n] + c);
      }
      double r_in[5], cs_in = 0.0;
      if (s > s0) {
        if (DIR == 1) {
#pragma unroll
          for (int n = 0; n < 5; ++n) r_in[n] = a.FX[n][cu + 1] - a.FX[n][cu];
          if (WANT_DT) cs_in = fmax(a.cfx[cu], a.cfx[cu + 1]);
        } else {
#pragma unroll
          for (int n = 0; n < 5; ++n) r_in[n] = a.R[n][cu];
          if (WANT_DT) cs_in = a.csum[cu];
        }
      }
      // ---- slope of cell s, face states, Riemann problem of face s ----
      double WR[7], WLn[7];
#pragma unroll
      for (int n = 0; n < NQ; ++n) {
        const double dp = qp[n] - q0[n];
        face_values<LIM>(q0[n], dm[n], dp, dx2, WR[n], WLn[n]);
        dm[n] = dp;
      }
      if (!MHD) WR[5] = WR[6] = 0.0;
      double F[7];
      const double cf = riemann<SOLVER, MHD>(WL, WR, Bn, g.gamma, F);
      if (s < s1 && MHD) {  // faces s0..s1-1 belong to this chunk
        a.FB[0][c] = F[5];
        a.FB[1][c] = F[6];
        if (WANT_FM) a.SG[c] = flux_sign(F[0]);
      }
      if (s > s0) {
        a.R[0][cu] = r_in[0] + (F[0] - Fp[0]);
        a.R[PN][cu] = r_in[PN] + (F[1] - Fp[1]);
        a.R[PT1][cu] = r_in[PT1] + (F[2] - Fp[2]);
        a.R[PT2][cu] = r_in[PT2] + (F[3] - Fp[3]);
        a.R[4][cu] = r_in[4] + (F[4] - Fp[4]);
        if (WANT_DT) {
          const double cs = cs_in + fmax(cfp, cf);  // G8: larger of the cell's two faces
          if (DIR == 1) a.csum[cu] = cs;
          else smax = fmax(smax, cs);
        }
      }
#pragma unroll
      for (int n = 0; n < 5; ++n) Fp[n] = F[n];
      cfp = cf;
#pragma unroll
      for (int n = 0; n < NQ; ++n) {
        WL[n] = WLn[n];
        q0[n] = qp[n];
        qp[n] = qn[n];
      }
      Bn = Bnn;
    }
  }
  if (WANT_DT && DIR == 2) {
    const double m = block_max_128(smax / g.dx);
    if (threadIdx.x == 0) atomicMax(&a.sc->smax_bits, (unsigned long long)__double_as_longlong(m));
  }
}

}  // namespace idfx
