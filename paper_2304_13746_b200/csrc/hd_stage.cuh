// hd_stage.cuh — hydrodynamics: the three flux sweeps of a stage in ONE kernel (a3 + a4 + a5, and for stages >= 2 also
// a8, a2 and a1).  Without a magnetic field nothing couples neighbouring cells beyond the flux stencil, so a stage needs
// no intermediate field at all: a CTA of 32 x 8 threads owns a column of (x, y) tiles and marches along z; every z plane
// of the five primitive fields arrives once, with its two-cell halo, as one TMA box (36 x 11 x 5 doubles) in a 4-stage
// shared-memory ring.  Thread (lx, ly) owns cell (x0 + lx, y0 + ly) of the plane and solves the three LOWER faces of its
// cell: the x and y faces from the plane in shared memory, the z face by marching (left state, forward differences and previous flux in registers).
// The upper x face comes from lane lx + 1 by shuffle, the upper y face from row ly + 1 through a small double-buffered
// exchange array, the upper z face one plane later: every Riemann problem inside a tile is solved once.  Lane 31 and
// row 7 only supply faces (tiles advance by 31 x 7 cells), which costs 15 % of the x/y solves and nothing in HBM traffic.
//   first stage : R = flux divergence (dt is not known before the whole grid has been swept), max_cells sum_d c_d / dx
//   later stages: U_s = w0 U_0 + w (U_{s-1} - dt/dx R), its primitives and their periodic ghost images (Eq. 9)
#pragma once
#include <cuda.h>

#include <cstdint>

#include "common.cuh"
#include "tma.cuh"
#include "physics.cuh"

namespace idfx {

constexpr int HD_TX = 32, HD_TY = 8;               // threads
constexpr int HD_CX = HD_TX - 1, HD_CY = HD_TY - 1;  // cells a tile completes
constexpr int HD_BW = 36, HD_BH = HD_TY + 3;       // box: columns x0-2-sh .. , rows y0-2 .. y0+8
constexpr int HD_FIELD = HD_BW * HD_BH;            // doubles of one field of a plane
constexpr int HD_PLANE = 5 * HD_FIELD;
constexpr uint32_t HD_PLANE_BYTES = HD_PLANE * 8;
constexpr int HD_NST = 4;
constexpr int HD_THREADS = HD_TX * HD_TY;
constexpr int HD_STRIDE = (HD_PLANE + 15) / 16 * 16;  // doubles between ring stages: TMA destinations are 128-byte aligned
constexpr int HD_RING_BYTES = HD_NST * HD_STRIDE * 8;
constexpr int HD_EXCH_BYTES = 2 * 6 * HD_TY * HD_TX * 8;
constexpr int HD_SMEM_BYTES = HD_RING_BYTES + HD_EXCH_BYTES + 2 * HD_NST * 8 + 128;
constexpr int HD_MINB = 2;  // CTAs per SM

struct HdStageArgs {
  int fV0;        // first field of the stage-input primitives inside the tensor map (0 or 11)
  int chunk;      // z planes per CTA
  double* R[5];
  DevScalars* sc;
  const double* Uin[5];  // U_{s-1}; or, with uin_is_r, the first stage's divergence R_1 (RK2: U_1 = U_0 - dt/dx R_1 is never stored)
  int uin_is_r;
  const double* U0[5];
  double* Uout[5];
  double* Vout[5];
  double w, w0;
};

// block-wide maximum for blocks of HD_THREADS threads; every thread must call it
__device__ __forceinline__ double block_max_hd(double v) {
  __shared__ double red[HD_THREADS / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  double m = red[0];
#pragma unroll
  for (int n = 1; n < HD_THREADS / 32; ++n) m = fmax(m, red[n]);
  return m;
}

// The pointwise arithmetic of the hydrodynamic update, written with explicit roundings: three kernels form the same
// quantities (k_update_hd, k_hd_stage, k_hd_stage_u) and must get the same bits whatever the compiler would contract around
// them, so that the two kinds of cycle (and decomposed against undecomposed runs) stay interchangeable bit for bit.
// a5 of the first stage: U_1 = U_0 - dt/dx R_1
__device__ __forceinline__ double hd_apply(double u0, double dtdx, double r) { return __fma_rn(-dtdx, r, u0); }
// Eq. 9: U_s = w0 U_0 + w (U_{s-1} - dt/dx R)
__device__ __forceinline__ double hd_combine(double w0, double u0, double w, double us, double dtdx, double r) {
  return __fma_rn(w0, u0, __dmul_rn(w, __fma_rn(-dtdx, r, us)));
}
// a2: (rho, v, p) of (rho, m, E)
__device__ __forceinline__ void hd_prims(double gm1, const double u[5], double v[5]) {
  const double ir = __ddiv_rn(1.0, u[0]);
  v[0] = u[0];
  v[1] = __dmul_rn(u[1], ir);
  v[2] = __dmul_rn(u[2], ir);
  v[3] = __dmul_rn(u[3], ir);
  const double v2 = __fma_rn(v[3], v[3], __fma_rn(v[2], v[2], __dmul_rn(v[1], v[1])));
  v[4] = __dmul_rn(gm1, __fma_rn(__dmul_rn(-0.5, u[0]), v2, u[4]));
}

// Lower face of the cell whose stencil (two cells below, one above, along one direction) is q[0..3][5 fields] in the
// sweep's local order (rho, u_n, u_t1, u_t2, p); returns c_face.
template <int SOLVER, int LIM>
__device__ __forceinline__ double hd_face(const double qm2[5], const double qm1[5], const double q0[5], const double qp1[5],
                                          double dx2, double gamma, double F[7]) {
  double WL[7], WR[7];
#pragma unroll
  for (int n = 0; n < 5; ++n) {
    double lo_unused, hi_unused;
    face_values<LIM>(qm1[n], qm1[n] - qm2[n], q0[n] - qm1[n], dx2, lo_unused, WL[n]);
    face_values<LIM>(q0[n], q0[n] - qm1[n], qp1[n] - q0[n], dx2, WR[n], hi_unused);
  }
  WL[5] = WL[6] = WR[5] = WR[6] = 0.0;
  return riemann<SOLVER, false>(WL, WR, 0.0, gamma, F);
}

template <int SOLVER, int LIM, bool FIRST>
__global__ void __launch_bounds__(HD_THREADS, HD_MINB) k_hd_stage(Geom g, HdStageArgs a, const __grid_constant__ CUtensorMap mapV) {
  // dynamic shared memory (HD_SMEM_BYTES, above the 48 KB static limit): the plane ring, the exchange array of the lower
  // y-face fluxes and c_face (double-buffered), the barriers
  extern __shared__ __align__(128) unsigned char hd_smem_raw[];
  // the dynamic region starts after the static one (block_max_hd's scratch): align by hand, TMA wants 128 bytes
  unsigned char* hd_smem = hd_smem_raw + ((128u - (smem_u32(hd_smem_raw) & 127u)) & 127u);
  double (*ring)[HD_STRIDE] = reinterpret_cast<double (*)[HD_STRIDE]>(hd_smem);
  double (*exch)[6][HD_TY][HD_TX] = reinterpret_cast<double (*)[6][HD_TY][HD_TX]>(hd_smem + HD_RING_BYTES);
  uint64_t* full = reinterpret_cast<uint64_t*>(hd_smem + HD_RING_BYTES + HD_EXCH_BYTES);
  uint64_t* empty = full + HD_NST;
  const double dx2 = g.dx * g.dx;
  const int lx = threadIdx.x & 31, ly = threadIdx.x >> 5;
  const int x0 = blockIdx.x * HD_CX, y0 = blockIdx.y * HD_CY;
  const int i = x0 + lx, j = y0 + ly;
  const int s0 = blockIdx.z * a.chunk;
  const int s1 = min(s0 + a.chunk, g.nz);
  const int np = s1 - s0 + 4;  // planes s0-2 .. s1+1
  const bool complete = lx < HD_CX && ly < HD_CY && i < g.nx && j < g.ny;  // this thread owns a cell of the result
  if (threadIdx.x == 0) {
#pragma unroll
    for (int st = 0; st < HD_NST; ++st) {
      mbar_init(&full[st], 1);
      mbar_init(&empty[st], HD_THREADS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  // a box must start on a 16-byte boundary: odd tiles start one column further left
  const int sh = x0 & 1;
  const int cx = IOFF + x0 - 2 - sh, cy = NG + y0 - 2, cz0 = NG + s0 - 2;
  auto issue = [&](int p) {
    uint64_t* bar = &full[p % HD_NST];
    mbar_expect_tx(bar, HD_PLANE_BYTES);
    tma_load_4d(ring[p % HD_NST], &mapV, bar, cx, cy, cz0 + p, a.fV0);
  };
  if (threadIdx.x == 0)
    for (int p = 0; p < min(np, HD_NST); ++p) issue(p);
  auto wait_plane = [&](int p) { mbar_wait(&full[p % HD_NST], (p / HD_NST) & 1); };
  // every thread is done with plane p; thread 0 refills the stage released one plane earlier (everybody has long let go
  // of it, so it does not wait) with plane p - 1 + HD_NST
  auto release_plane = [&](int p) {
    mbar_arrive(&empty[p % HD_NST]);
    const int pr = p - 1;
    if (threadIdx.x == 0 && pr >= 0 && pr + HD_NST < np) {
      mbar_wait(&empty[pr % HD_NST], (pr / HD_NST) & 1);
      issue(pr + HD_NST);
    }
  };
  const int so = (ly + 2) * HD_BW + lx + 2 + sh;  // this thread's cell inside one field of a plane
  auto own = [&](int p, double q[5]) {
    const double* r = ring[p % HD_NST];
#pragma unroll
    for (int n = 0; n < 5; ++n) q[n] = r[n * HD_FIELD + so];
  };

  double dtdx = 0.0;
  if (!FIRST) dtdx = a.sc->dt_used / g.dx;  // published by the first stage's update kernel
  // z marching state in the local order of the z sweep: (rho, vz, vx, vy, p)
  constexpr int ZQ[5] = {0, 3, 1, 2, 4};
  double dm[5], q0[5], WL[7];
  {
    double qm[5], qc[5], t[5];
    wait_plane(0);
    own(0, t);
#pragma unroll
    for (int n = 0; n < 5; ++n) qm[n] = t[ZQ[n]];
    release_plane(0);
    wait_plane(1);
    own(1, t);
#pragma unroll
    for (int n = 0; n < 5; ++n) qc[n] = t[ZQ[n]];
    release_plane(1);
    wait_plane(2);
    own(2, t);
#pragma unroll
    for (int n = 0; n < 5; ++n) {
      q0[n] = t[ZQ[n]];
      dm[n] = q0[n] - qc[n];
      double lo_unused;
      face_values<LIM>(qc[n], qc[n] - qm[n], dm[n], dx2, lo_unused, WL[n]);  // cell s0-1 at its upper face
    }
    WL[5] = WL[6] = 0.0;
  }
  // ghost images of this column in x and y (later stages write the primitives of the result with their images)
  const long long gx = i < NG ? (long long)g.nx : (i >= g.nx - NG ? -(long long)g.nx : 0);
  const long long gy = j < NG ? (long long)g.ny * g.sy : (j >= g.ny - NG ? -(long long)g.ny * g.sy : 0);
  long long c = g.at(min(i, g.nx - 1), min(j, g.ny - 1), s0);
  double Fzp[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, cfzp = 0.0;
  double rxy[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, csxy = 0.0;  // x and y parts of cell s-1
  double smax = 0.0;
  for (int s = s0; s <= s1; ++s, c += g.sz) {
    const int p = s - s0 + 2;  // ring index of plane s; plane s+1 is p + 1
    double qp[5];
    {
      double t[5];
      wait_plane(p + 1);
      own(p + 1, t);
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
          const double uin = a.Uin[n][cu];
          const double us = a.uin_is_r ? hd_apply(u0, dtdx, uin) : uin;
          u[n] = dtdx == 0.0 ? u0 : hd_combine(a.w0, u0, a.w, us, dtdx, rt[n]);  // Eq. 9
        }
        double v[5];
        hd_prims(g.gamma - 1.0, u, v);
        const double vx = v[1], vy = v[2], vz = v[3];
        double pr = v[4];
        if (g.pfloor > 0.0 && pr < g.pfloor) {
          const bool acts = pr < g.pfloor * (1.0 - 1e-9);  // a cell floored before recomputes to the floor within rounding
          pr = g.pfloor;
          if (acts) {
            u[4] = pr / (g.gamma - 1.0) + 0.5 * u[0] * (vx * vx + vy * vy + vz * vz);
            atomicAdd(&a.sc->nfloor, 1ull);
          }
        }
        if (!(u[0] > 0.0) || !(pr > 0.0)) a.sc->flag = 1;
#pragma unroll
        for (int n = 0; n < 5; ++n) a.Uout[n][cu] = u[n];
        v[4] = pr;
        const int k = s - 1;
        const long long gz = k < NG ? (long long)g.nz * g.sz : (k >= g.nz - NG ? -(long long)g.nz * g.sz : 0);
#pragma unroll
        for (int n = 0; n < 5; ++n) a.Vout[n][cu] = v[n];
        if (!g.open && (gx != 0 || gy != 0 || gz != 0)) {
#pragma unroll
          for (int m = 1; m < 8; ++m) {
            const long long off = ((m & 1) ? gx : 0) + ((m & 2) ? gy : 0) + ((m & 4) ? gz : 0);
            const bool ok = (!(m & 1) || gx != 0) && (!(m & 2) || gy != 0) && (!(m & 4) || gz != 0);
            if (ok) {
#pragma unroll
              for (int n = 0; n < 5; ++n) a.Vout[n][cu + off] = v[n];
            }
          }
        }
      }
    }
#pragma unroll
    for (int n = 0; n < 5; ++n) Fzp[n] = F[n];
    cfzp = cfz;
#pragma unroll
    for (int n = 0; n < 7; ++n) WL[n] = WLn[n];
    // ---- x and y faces of plane s (cells s0 .. s1-1 only) ----
    if (s < s1) {
      const double* r = ring[p % HD_NST];
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
      double (*ex)[HD_TY][HD_TX] = exch[s & 1];
#pragma unroll
      for (int n = 0; n < 5; ++n) ex[n][ly][lx] = Fy[n];
      ex[5][ly][lx] = cfy;
      __syncthreads();  // also orders this plane's reads of exch[s & 1] after the writes; the other buffer is free again
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
    release_plane(p);
#pragma unroll
    for (int n = 0; n < 5; ++n) q0[n] = qp[n];
  }
  if (FIRST) {
    const double m = block_max_hd(complete ? smax / g.dx : 0.0);
    if (threadIdx.x == 0) atomicMax(&a.sc->smax_bits, (unsigned long long)__double_as_longlong(m));
  }
}

}  // namespace idfx
