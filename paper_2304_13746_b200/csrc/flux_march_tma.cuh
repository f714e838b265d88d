// flux_march_tma.cuh — the y / z marching sweep (flux_march.cuh) with its stencil planes staged through shared
// memory by TMA.  Each CTA owns a 32 (x) by 4 (transverse) strip of pencils; per sweep plane one elected thread
// issues two cp.async.bulk.tensor.4d loads (8 primitive fields and the staggered normal field, 9 KB) into a
// 5-stage ring guarded by full / empty mbarriers, three planes ahead of the consumers.  Consumers read only their
// own element of every field, so the ring replaces the register prefetch and the per-load address arithmetic.
// MHD only (the HD sweeps keep the register-prefetch kernel).
#pragma once
#include <cuda.h>

#include <cstdint>

#include "common.cuh"
#include "tma.cuh"
#include "flux_march.cuh"
#include "physics.cuh"

namespace idfx {

#ifndef IDFX_MINB_T
#define IDFX_MINB_T 3
#endif
#ifndef IDFX_TMA_PF
#define IDFX_TMA_PF 1                    // L1 prefetch of the next plane's directly loaded fields
#endif
#ifndef IDFX_PF_DIST
#define IDFX_PF_DIST 1                   // planes ahead
#endif
constexpr int TMA_NST = 5;               // ring stages
constexpr int TMA_SLACK = 2;             // a stage is refilled two planes after it was consumed
constexpr int TMA_PLANE_V = 8 * 4 * 32;  // doubles of the primitive box (8 fields x 4 rows x 32 columns)
constexpr int TMA_PLANE = TMA_PLANE_V + 4 * 32;
constexpr uint32_t TMA_PLANE_BYTES = TMA_PLANE * 8;

struct FluxTArgs {
  int fV0;              // first field of the stage-input primitive buffer inside the V tensor map (0 or 11)
  int fB;               // field of the normal face component inside the B tensor map
  int ns, nt, chunk;
  long long sd, st;
  const double* FX[5];
  const double* cfx;
  double* R[5];
  double* csum;
  double* FB[2];
  signed char* SG;      // sign of the face mass flux (upwind-contact EMF only)
  DevScalars* sc;
  // APPLY (stages >= 2 of the z sweep): the completed divergence is applied at once, U_s = w0 U_0 + w (U_{s-1} - dt/dx R)
  const double* Uin[5];
  const double* U0[5];
  double* Uout[5];
  double w, w0;
};

template <int SOLVER, int LIM, int DIR, bool WANT_DT, bool WANT_FM, bool APPLY>
__global__ void __launch_bounds__(128, IDFX_MINB_T) k_flux_march_tma(Geom g, FluxTArgs a, const __grid_constant__ CUtensorMap mapV,
                                                           const __grid_constant__ CUtensorMap mapB) {
  __shared__ alignas(128) double ring[TMA_NST][TMA_PLANE];
  __shared__ uint64_t full[TMA_NST], empty[TMA_NST];
  const double dx2 = g.dx * g.dx;
  constexpr int PN = 1 + DIR, PT1 = 1 + (DIR + 1) % 3, PT2 = 1 + (DIR + 2) % 3;
  // primitive field ids inside the box, in the sweep's local order (rho, u, v, w, p, B_t1, B_t2)
  constexpr int FQ[7] = {0, 1 + DIR, 1 + (DIR + 1) % 3, 1 + (DIR + 2) % 3, 4, 5 + (DIR + 1) % 3, 5 + (DIR + 2) % 3};
  const int lx = threadIdx.x & 31, lt = threadIdx.x >> 5;
  const int i = blockIdx.x * 32 + lx;
  const int t = blockIdx.y * 4 + lt;
  const int s0 = blockIdx.z * a.chunk;
  const int s1 = min(s0 + a.chunk, a.ns);
  const bool active = i < g.nx && t < a.nt;
  const int np = s1 - s0 + 4;  // planes s0-2 .. s1+1
  if (threadIdx.x == 0) {
#pragma unroll
    for (int st = 0; st < TMA_NST; ++st) {
      mbar_init(&full[st], 1);
      mbar_init(&empty[st], 128);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  const int cx = IOFF + blockIdx.x * 32, ct = NG + blockIdx.y * 4, cs0 = NG + s0 - 2;
  auto issue = [&](int j) {
    uint64_t* bar = &full[j % TMA_NST];
    double* dst = ring[j % TMA_NST];
    mbar_expect_tx(bar, TMA_PLANE_BYTES);
    if (DIR == 1) {
      tma_load_4d(dst, &mapV, bar, cx, cs0 + j, ct, a.fV0);
      tma_load_4d(dst + TMA_PLANE_V, &mapB, bar, cx, cs0 + j, ct, a.fB);
    } else {
      tma_load_4d(dst, &mapV, bar, cx, ct, cs0 + j, a.fV0);
      tma_load_4d(dst + TMA_PLANE_V, &mapB, bar, cx, ct, cs0 + j, a.fB);
    }
  };
  if (threadIdx.x == 0)
    for (int j = 0; j < min(np, TMA_NST); ++j) issue(j);
  const int so = lt * 32 + lx;  // this thread's element inside one field of a plane
  // waits for plane j, copies this thread's 7 primitives and normal field out, releases the stage
  auto consume = [&](int j, double q[7], double& bn) {
    const int st = j % TMA_NST;
    mbar_wait(&full[st], (j / TMA_NST) & 1);
    const double* p = ring[st];
#pragma unroll
    for (int n = 0; n < 7; ++n) q[n] = p[FQ[n] * 128 + so];
    bn = p[TMA_PLANE_V + so];
    mbar_arrive(&empty[st]);
    if (threadIdx.x == 0) {
      const int jr = j - TMA_SLACK;
      if (jr >= 0 && jr + TMA_NST < np) {
        mbar_wait(&empty[jr % TMA_NST], (jr / TMA_NST) & 1);
        issue(jr + TMA_NST);
      }
    }
  };

  double smax = 0.0, dtdx = 0.0;
  if (APPLY) dtdx = a.sc->dt_used / g.dx;  // published by the first stage's update kernel
  double dm[7], q0[7], WL[7], Bn, dummy;
  {
    double qm[7], qc[7];
    consume(0, qm, dummy);
    consume(1, qc, dummy);
    consume(2, q0, Bn);
#pragma unroll
    for (int n = 0; n < 7; ++n) {
      dm[n] = q0[n] - qc[n];
      double lo_unused;
      face_values<LIM>(qc[n], qc[n] - qm[n], dm[n], dx2, lo_unused, WL[n]);  // cell s0-1 at its upper face
    }
  }
  long long c = g.at(min(i, g.nx - 1), 0, 0) + (long long)min(t, a.nt - 1) * a.st + (long long)s0 * a.sd;
  const long long sd = a.sd;
  double Fp[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, cfp = 0.0;
  // z sweeps: two planes per trip, so that the carried state (left face state, forward differences, previous flux) needs
  // no register-to-register rotation (5.66 -> 5.50 ms at 512^3; the y sweep is slower that way, 5.17 -> 5.25 ms)
#ifndef IDFX_MARCH_UNROLL_Z
#define IDFX_MARCH_UNROLL_Z 2
#endif
  constexpr int UNROLL = DIR == 2 ? IDFX_MARCH_UNROLL_Z : 1;
#pragma unroll UNROLL
  for (int s = s0; s <= s1; ++s, c += sd) {
    double qp[7], Bnn;
    consume(s - s0 + 3, qp, Bnn);  // plane s+1
    if (active) {
      const long long cu = c - sd;  // cell s-1, completed by this face
      if (IDFX_TMA_PF && s + IDFX_PF_DIST < s1) {
        const long long cpf = c + (IDFX_PF_DIST - 1) * sd;
#pragma unroll
        for (int n = 0; n < 5; ++n) prefetch_l1(DIR == 1 ? a.FX[n] + cpf + 1 : a.R[n] + cpf);
        if (APPLY) {
#pragma unroll
          for (int n = 0; n < 5; ++n) {
            prefetch_l1(a.Uin[n] + cpf);
            prefetch_l1(a.U0[n] + cpf);
          }
        }
      }
      // Directly loaded inputs of cell s-1 (prefetched into L1 one plane ago).  The y sweep (two loads per x flux) reads
      // them only after the solve: placed behind the face-flux stores, which they might alias as far as the compiler
      // knows, they cannot be hoisted over the Riemann solve and hold no registers during it (158 registers, no spills;
      // 5.43 -> 5.23 ms at 512^3).  The z sweeps are faster with the loads in flight early (5.8 against 6.2 ms).
      double uin[5], u0[5], r_in[5], cs_in = 0.0;
      auto load_inputs = [&]() {
        if (APPLY && s > s0) {
#pragma unroll
          for (int n = 0; n < 5; ++n) {
            uin[n] = a.Uin[n][cu];
            u0[n] = a.U0[n][cu];
          }
        }
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
      };
#ifndef IDFX_LATE_MODE
#define IDFX_LATE_MODE 0
#endif
      constexpr bool LATE = IDFX_LATE_MODE == 1 ? true : (IDFX_LATE_MODE == 2 ? !APPLY : DIR == 1);
      if (!LATE) load_inputs();
      double WR[7], WLn[7];
#pragma unroll
      for (int n = 0; n < 7; ++n) {
        const double dp = qp[n] - q0[n];
        face_values<LIM>(q0[n], dm[n], dp, dx2, WR[n], WLn[n]);
        dm[n] = dp;
      }
      double F[7];
      const double cf = riemann<SOLVER, true>(WL, WR, Bn, g.gamma, F);
      if (s < s1) {  // faces s0..s1-1 belong to this chunk
        a.FB[0][c] = F[5];
        a.FB[1][c] = F[6];
        if (WANT_FM) a.SG[c] = flux_sign(F[0]);
      }
      if (LATE) load_inputs();
      if (s > s0) {
        double rt[5];
        rt[0] = r_in[0] + (F[0] - Fp[0]);
        rt[PN] = r_in[PN] + (F[1] - Fp[1]);
        rt[PT1] = r_in[PT1] + (F[2] - Fp[2]);
        rt[PT2] = r_in[PT2] + (F[3] - Fp[3]);
        rt[4] = r_in[4] + (F[4] - Fp[4]);
#pragma unroll
        for (int n = 0; n < 5; ++n) {
          if (APPLY) a.Uout[n][cu] = dtdx == 0.0 ? u0[n] : a.w0 * u0[n] + a.w * (uin[n] - dtdx * rt[n]);  // Eq. 9
          else a.R[n][cu] = rt[n];
        }
        if (WANT_DT) {
          const double cs = cs_in + fmax(cfp, cf);  // G8
          if (DIR == 1) a.csum[cu] = cs;
          else smax = fmax(smax, cs);
        }
      }
#pragma unroll
      for (int n = 0; n < 5; ++n) Fp[n] = F[n];
      cfp = cf;
#pragma unroll
      for (int n = 0; n < 7; ++n) WL[n] = WLn[n];
    }
#pragma unroll
    for (int n = 0; n < 7; ++n) q0[n] = qp[n];
    Bn = Bnn;
  }
  if (WANT_DT && DIR == 2) {
    const double m = block_max_128(smax / g.dx);
    if (threadIdx.x == 0) atomicMax(&a.sc->smax_bits, (unsigned long long)__double_as_longlong(m));
  }
}

// ---------------------------------------------------------------------------------------------
// x sweep with TMA-staged rows.  A CTA owns a window of 31 x-faces (cells f0-1 .. f0+30, one lane each, plus one halo
// cell on either side) of four consecutive rows (one warp per row) and marches over z planes; per plane two boxes
// (36 columns x 4 rows x 8 primitive fields, and the B_x faces) land in a 4-stage ring.  Lanes read their three-cell
// stencil from shared memory, so no edge loads and no shuffles of the primitives are needed; only the left face state
// comes from the neighbouring lane by shuffle.  Lanes 1..31 solve the left face of their cell.
// ---------------------------------------------------------------------------------------------
constexpr int TX_NST = 4, TX_SLACK = 1;
constexpr int TX_W = 36;
constexpr int TX_PLANE_V = 8 * 4 * TX_W;
constexpr int TX_PLANE = TX_PLANE_V + 4 * TX_W;
constexpr uint32_t TX_PLANE_BYTES = TX_PLANE * 8;

struct FluxXTArgs {
  int fV0, fB;   // first primitive field inside the V tensor map; field of B_x inside the B tensor map
  int chunk;     // z planes per CTA
  double* FH[5];
  double* FB[2];
  double* cf;
  signed char* sg;  // sign of the mass flux (upwind-contact EMF only, else null)
};

template <int SOLVER, int LIM>
__global__ void __launch_bounds__(128, 4) k_flux_x_tma(Geom g, FluxXTArgs a, const __grid_constant__ CUtensorMap mapV,
                                                       const __grid_constant__ CUtensorMap mapB) {
  __shared__ alignas(128) double ring[TX_NST][TX_PLANE];
  __shared__ uint64_t full[TX_NST], empty[TX_NST];
  const double dx2 = g.dx * g.dx;
  constexpr int FQ[7] = {0, 1, 2, 3, 4, 6, 7};  // rho, vx, vy, vz, p, Bc_y, Bc_z
  const int lane = threadIdx.x & 31, row = threadIdx.x >> 5;
  const int f0 = 31 * blockIdx.x;
  const int ci = f0 - 1 + lane;
  const int j = blockIdx.y * 4 + row;
  const int k0 = blockIdx.z * a.chunk;
  const int np = min(k0 + a.chunk, g.nz) - k0;
  const bool solve = lane >= 1 && ci <= g.nx && j < g.ny;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int st = 0; st < TX_NST; ++st) {
      mbar_init(&full[st], 1);
      mbar_init(&empty[st], 128);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  // TMA needs the box to start on a 16-byte boundary: shift odd windows one column left (36 >= 34 + 1 columns)
  const int sh = f0 & 1;
  const int cx = IOFF + f0 - 2 - sh, cy = NG + blockIdx.y * 4, cz0 = NG + k0;
  auto issue = [&](int p) {
    uint64_t* bar = &full[p % TX_NST];
    double* dst = ring[p % TX_NST];
    mbar_expect_tx(bar, TX_PLANE_BYTES);
    tma_load_4d(dst, &mapV, bar, cx, cy, cz0 + p, a.fV0);
    tma_load_4d(dst + TX_PLANE_V, &mapB, bar, cx, cy, cz0 + p, a.fB);
  };
  if (threadIdx.x == 0)
    for (int p = 0; p < min(np, TX_NST); ++p) issue(p);
  const int so = row * TX_W + lane + sh;  // stencil cells ci-1, ci, ci+1 sit at so, so+1, so+2
  long long c = g.at(min(ci, g.nx + 1), min(j, g.ny - 1), k0);
  for (int p = 0; p < np; ++p, c += g.sz) {
    const int st = p % TX_NST;
    mbar_wait(&full[st], (p / TX_NST) & 1);
    __syncwarp();  // the lanes leave the wait loop one by one: reconverge once here rather than around every shuffle below
    const double* r = ring[st];
    double WL[7], WR[7];
#pragma unroll
    for (int n = 0; n < 7; ++n) {
      const double* f = r + FQ[n] * (4 * TX_W) + so;
      const double qm = f[0], q = f[1], qp = f[2];
      double up;
      face_values<LIM>(q, q - qm, qp - q, dx2, WR[n], up);
      WL[n] = __shfl_up_sync(0xffffffffu, up, 1);
    }
    const double Bn = r[TX_PLANE_V + so + 1];
    mbar_arrive(&empty[st]);
    if (threadIdx.x == 0) {
      const int pr = p - TX_SLACK;
      if (pr >= 0 && pr + TX_NST < np) {
        mbar_wait(&empty[pr % TX_NST], (pr / TX_NST) & 1);
        issue(pr + TX_NST);
      }
    }
    if (solve) {
      double F[7];
      const double cface = riemann<SOLVER, true>(WL, WR, Bn, g.gamma, F);
#pragma unroll
      for (int n = 0; n < 5; ++n) a.FH[n][c] = F[n];
      a.FB[0][c] = F[5];
      a.FB[1][c] = F[6];
      if (a.cf) a.cf[c] = cface;  // only the dt evaluation of stage 1 reads it
      if (a.sg) a.sg[c] = flux_sign(F[0]);
    }
  }
}

}  // namespace idfx
