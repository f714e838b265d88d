// hd_stage_u.cuh — hydrodynamics, RK2 on a periodic box: the stage kernels of hd_stage.cuh fed with the CONSERVED fields.
// A hydrodynamic stage couples cells through the flux stencil only, so the primitives a stage reconstructs from need never
// exist in memory: every z plane of U_0 (second stage: of U_0 and of the first stage's divergence R_1) arrives with its
// two-cell halo as TMA boxes, the CTA turns it into the primitives of the stage input (first stage: of U_0; second stage:
// of U_1 = U_0 - dt/dx R_1, the a5 + a2 work of k_update_hd) in shared memory, and the sweeps of hd_stage.cuh run on that.
// What is gone from the cycle: the update kernel between the stages (10 doubles read, 5 written per cell), the primitives
// the second stage wrote for the next cycle (5) and read back (5 + halo).  The halo of R_1 and of the result U comes from
// the ghost-fill kernel (a1) after each stage; the one after the first stage also publishes the dt of the cycle.
// (Measured at 512^3: alternating the two landing slots in the first stage, one plane more of look-ahead, changes nothing:
// the kernels do not wait for their loads.  Images written by the owners of the boundary cells inside these kernels, as the MHD update kernel
// does, cost the stage kernels 3 %, more than the two fill launches take: 16.84 against 16.72 ms per cycle.)
//   first stage : R_1 = flux divergence of prim(U_0), max_cells sum_d c_d / dx
//   second stage: U = w0 U_0 + w (U_1 - dt/dx R_2) (Eq. 9), written to the OTHER conserved buffer: neighbouring tiles still
//                 read the halo of U_0 (the host swaps the roles of the two buffers after the cycle)
// Shared memory: one landing slot per TMA box (U_0, R_1), a ring of three converted planes (the plane being solved, the
// next one, the one being converted), the exchange array of hd_stage.cuh: 104 KB, two CTAs per SM.
#pragma once
#include "hd_stage.cuh"

namespace idfx {

constexpr int HDU_NPRIM = 3;
constexpr int HDU_RAW_BYTES = 2 * HD_STRIDE * 8;
constexpr int HDU_PRIM_BYTES = HDU_NPRIM * HD_STRIDE * 8;
constexpr int HDU_SMEM_BYTES = HDU_RAW_BYTES + HDU_PRIM_BYTES + HD_EXCH_BYTES + 16 + 128;

template <int SOLVER, int LIM, bool FIRST>
__global__ void __launch_bounds__(HD_THREADS, HD_MINB) k_hd_stage_u(Geom g, HdStageArgs a, const __grid_constant__ CUtensorMap mapU,
                                                                    const __grid_constant__ CUtensorMap mapR) {
  extern __shared__ __align__(128) unsigned char hdu_smem_raw[];
  unsigned char* smem = hdu_smem_raw + ((128u - (smem_u32(hdu_smem_raw) & 127u)) & 127u);
  double (*raw)[HD_STRIDE] = reinterpret_cast<double (*)[HD_STRIDE]>(smem);  // [0]: U_0, [1]: R_1 of the plane that landed last
  double (*prim)[HD_STRIDE] = reinterpret_cast<double (*)[HD_STRIDE]>(smem + HDU_RAW_BYTES);
  double (*exch)[6][HD_TY][HD_TX] = reinterpret_cast<double (*)[6][HD_TY][HD_TX]>(smem + HDU_RAW_BYTES + HDU_PRIM_BYTES);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + HDU_RAW_BYTES + HDU_PRIM_BYTES + HD_EXCH_BYTES);
  const double dx2 = g.dx * g.dx;
  const double gm1 = g.gamma - 1.0;
  const int lx = threadIdx.x & 31, ly = threadIdx.x >> 5;
  const int x0 = blockIdx.x * HD_CX, y0 = blockIdx.y * HD_CY;
  const int i = x0 + lx, j = y0 + ly;
  const int s0 = blockIdx.z * a.chunk;
  const int s1 = min(s0 + a.chunk, g.nz);
  const int np = s1 - s0 + 4;  // planes s0-2 .. s1+1
  const bool complete = lx < HD_CX && ly < HD_CY && i < g.nx && j < g.ny;
  if (threadIdx.x == 0) {
    mbar_init(full, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  const int sh = x0 & 1;  // a box must start on a 16-byte boundary: odd tiles start one column further left
  const int cx = IOFF + x0 - 2 - sh, cy = NG + y0 - 2, cz0 = NG + s0 - 2;
  // plane q of the chunk into the landing slots; the threads have all let go of them (a __syncthreads precedes every call)
  auto issue = [&](int q) {
    mbar_expect_tx(full, FIRST ? HD_PLANE_BYTES : 2 * HD_PLANE_BYTES);
    tma_load_4d(raw[0], &mapU, full, cx, cy, cz0 + q, a.fV0);
    if (!FIRST) tma_load_4d(raw[1], &mapR, full, cx, cy, cz0 + q, 0);
  };
  auto wait_raw = [&](int q) { mbar_wait(full, q & 1); };
  double dtdx = 0.0;
  if (!FIRST) dtdx = a.sc->dt_used / g.dx;  // published after the first stage (k_fill_ghost_dt)
  // primitives of the stage input in cell e of the landed plane (a2; second stage: after a5 of the first stage)
  auto convert = [&](int e, double v[5]) {
    double u[5];
#pragma unroll
    for (int n = 0; n < 5; ++n) {
      u[n] = raw[0][n * HD_FIELD + e];
      if (!FIRST) u[n] = hd_apply(u[n], dtdx, raw[1][n * HD_FIELD + e]);
    }
    hd_prims(gm1, u, v);
  };
  auto convert_plane = [&](int q) {
    double* dst = prim[q % HDU_NPRIM];
#pragma unroll
    for (int e = threadIdx.x; e < HD_FIELD; e += HD_THREADS) {
      double v[5];
      convert(e, v);
#pragma unroll
      for (int n = 0; n < 5; ++n) dst[n * HD_FIELD + e] = v[n];
    }
  };
  const int so = (ly + 2) * HD_BW + lx + 2 + sh;  // this thread's cell inside one field of a plane
  auto own = [&](int q, double t[5]) {
    const double* r = prim[q % HDU_NPRIM];
#pragma unroll
    for (int n = 0; n < 5; ++n) t[n] = r[n * HD_FIELD + so];
  };
  // an unphysical U_1 raises the flag as k_update_hd does: every active cell once, by the thread that owns it
  auto check = [&](const double t[5]) {
    if (!FIRST && complete && (!(t[0] > 0.0) || !(t[4] > 0.0))) a.sc->flag = 1;
  };

  // z marching state in the local order of the z sweep: (rho, vz, vx, vy, p)
  constexpr int ZQ[5] = {0, 3, 1, 2, 4};
  double dm[5], q0[5], WL[7];
  {
    double qm[5], qc[5], t[5];
    if (threadIdx.x == 0) issue(0);
    wait_raw(0);  // planes s0-2 and s0-1: only this thread's own cell is needed
    convert(so, t);
#pragma unroll
    for (int n = 0; n < 5; ++n) qm[n] = t[ZQ[n]];
    __syncthreads();
    if (threadIdx.x == 0) issue(1);
    wait_raw(1);
    convert(so, t);
#pragma unroll
    for (int n = 0; n < 5; ++n) qc[n] = t[ZQ[n]];
    __syncthreads();
    if (threadIdx.x == 0) issue(2);
    wait_raw(2);
    convert_plane(2);
    __syncthreads();
    if (threadIdx.x == 0) issue(3);
    own(2, t);
    check(t);
#pragma unroll
    for (int n = 0; n < 5; ++n) {
      q0[n] = t[ZQ[n]];
      dm[n] = q0[n] - qc[n];
      double lo_unused;
      face_values<LIM>(qc[n], qc[n] - qm[n], dm[n], dx2, lo_unused, WL[n]);  // cell s0-1 at its upper face
    }
    WL[5] = WL[6] = 0.0;
    wait_raw(3);
    convert_plane(3);
    __syncthreads();
    if (threadIdx.x == 0 && 4 < np) issue(4);
  }
  long long c = g.at(min(i, g.nx - 1), min(j, g.ny - 1), s0);
  double Fzp[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, cfzp = 0.0;
  double rxy[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, csxy = 0.0;  // x and y parts of cell s-1
  double smax = 0.0;
  for (int s = s0; s <= s1; ++s, c += g.sz) {
    const int p = s - s0 + 2;  // plane s of the chunk; plane s+1 is p + 1
    double qp[5];
    {
      double t[5];
      own(p + 1, t);
      if (s + 1 < s1) check(t);
#pragma unroll
      for (int n = 0; n < 5; ++n) qp[n] = t[ZQ[n]];
    }
    if (!FIRST && complete && s < s1) {  // the conserved inputs of cell s are needed one plane from now
#pragma unroll
      for (int n = 0; n < 5; ++n) {
        prefetch_l1(a.Uin[n] + c);
        prefetch_l1(a.U0[n] + c);
      }
    }
    // ---- z face s-1/2: closes cell s-1 ----
    double WR[7], WLn[7], F[7];
#pragma unroll
    for (int n = 0; n < 5; ++n) {
      const double dp = qp[n] - q0[n];
      face_values<LIM>(q0[n], dm[n], dp, dx2, WR[n], WLn[n]);
      dm[n] = dp;
    }
    WR[5] = WR[6] = WLn[5] = WLn[6] = 0.0;
    const double cfz = riemann<SOLVER, false>(WL, WR, 0.0, g.gamma, F);
    if (s > s0 && complete) {
      const long long cu = c - g.sz;
      double rt[5];
      rt[0] = rxy[0] + (F[0] - Fzp[0]);
      rt[3] = rxy[3] + (F[1] - Fzp[1]);  // z sweep: normal = z, t1 = x, t2 = y
      rt[1] = rxy[1] + (F[2] - Fzp[2]);
      rt[2] = rxy[2] + (F[3] - Fzp[3]);
      rt[4] = rxy[4] + (F[4] - Fzp[4]);
      if (FIRST) {
#pragma unroll
        for (int n = 0; n < 5; ++n) a.R[n][cu] = rt[n];
        smax = fmax(smax, csxy + fmax(cfzp, cfz));  // G8
      } else {
        double u[5];
#pragma unroll
        for (int n = 0; n < 5; ++n) {
          const double u0 = a.U0[n][cu];
          const double us = hd_apply(u0, dtdx, a.Uin[n][cu]);  // U_1 again, as the conversion formed it
          u[n] = dtdx == 0.0 ? u0 : hd_combine(a.w0, u0, a.w, us, dtdx, rt[n]);  // Eq. 9
        }
        double v[5];
        hd_prims(gm1, u, v);
        if (!(u[0] > 0.0) || !(v[4] > 0.0)) a.sc->flag = 1;
#pragma unroll
        for (int n = 0; n < 5; ++n) a.Uout[n][cu] = u[n];
      }
    }
#pragma unroll
    for (int n = 0; n < 5; ++n) Fzp[n] = F[n];
    cfzp = cfz;
#pragma unroll
    for (int n = 0; n < 7; ++n) WL[n] = WLn[n];
    // ---- x and y faces of plane s (cells s0 .. s1-1 only) ----
    if (s < s1) {
      const double* r = prim[p % HDU_NPRIM];
      double Fx[7], Fy[7], cfx, cfy;
      {  // x: local order (rho, vx, vy, vz, p) = field order
        double a2[5], a1[5], b0[5], b1[5];
#pragma unroll
        for (int n = 0; n < 5; ++n) {
          const double* f = r + n * HD_FIELD + so;
          a2[n] = f[-2]; a1[n] = f[-1]; b0[n] = f[0]; b1[n] = f[1];
        }
        cfx = hd_face<SOLVER, LIM>(a2, a1, b0, b1, dx2, g.gamma, Fx);
      }
      {  // y: local order (rho, vy, vz, vx, p)
        constexpr int YQ[5] = {0, 2, 3, 1, 4};
        double a2[5], a1[5], b0[5], b1[5];
#pragma unroll
        for (int n = 0; n < 5; ++n) {
          const double* f = r + YQ[n] * HD_FIELD + so;
          a2[n] = f[-2 * HD_BW]; a1[n] = f[-HD_BW]; b0[n] = f[0]; b1[n] = f[HD_BW];
        }
        cfy = hd_face<SOLVER, LIM>(a2, a1, b0, b1, dx2, g.gamma, Fy);
      }
      // plane s+2 (it exists: s < s1) into the slot plane s-1 left, whose last reader passed the barrier of the previous trip
      wait_raw(p + 2);
      convert_plane(p + 2);
      double (*ex)[HD_TY][HD_TX] = exch[s & 1];
#pragma unroll
      for (int n = 0; n < 5; ++n) ex[n][ly][lx] = Fy[n];
      ex[5][ly][lx] = cfy;
      __syncthreads();  // orders the exchange array, the converted plane and the reads of the landing slots
      if (threadIdx.x == 0 && p + 3 < np) issue(p + 3);
      const int lyu = min(ly + 1, HD_TY - 1);
      double d[5];
      // upper x face from the next lane; x sweep: (n, t1, t2) = (x, y, z)
      d[0] = __shfl_down_sync(0xffffffffu, Fx[0], 1) - Fx[0];
      d[1] = __shfl_down_sync(0xffffffffu, Fx[1], 1) - Fx[1];
      d[2] = __shfl_down_sync(0xffffffffu, Fx[2], 1) - Fx[2];
      d[3] = __shfl_down_sync(0xffffffffu, Fx[3], 1) - Fx[3];
      d[4] = __shfl_down_sync(0xffffffffu, Fx[4], 1) - Fx[4];
      const double cfxu = __shfl_down_sync(0xffffffffu, cfx, 1);
      // upper y face from the next row; y sweep: (n, t1, t2) = (y, z, x)
      rxy[0] = d[0] + (ex[0][lyu][lx] - Fy[0]);
      rxy[2] = d[2] + (ex[1][lyu][lx] - Fy[1]);
      rxy[3] = d[3] + (ex[2][lyu][lx] - Fy[2]);
      rxy[1] = d[1] + (ex[3][lyu][lx] - Fy[3]);
      rxy[4] = d[4] + (ex[4][lyu][lx] - Fy[4]);
      csxy = fmax(cfx, cfxu) + fmax(cfy, ex[5][lyu][lx]);
    }
#pragma unroll
    for (int n = 0; n < 5; ++n) q0[n] = qp[n];
  }
  if (FIRST) {
    const double m = block_max_hd(complete ? smax / g.dx : 0.0);
    if (threadIdx.x == 0) atomicMax(&a.sc->smax_bits, (unsigned long long)__double_as_longlong(m));
  }
}

}  // namespace idfx
