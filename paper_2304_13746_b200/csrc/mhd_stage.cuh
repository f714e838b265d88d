// mhd_stage.cuh — ideal MHD: the three flux sweeps of a stage AND its edge EMFs in ONE kernel (a3 + a4 + a5 + a6, the dt
// reduction a9 in the first stage, the RK combine a8 of the cell-centred state in later stages).
//
// A CTA of 32 x TY threads owns a column of (x, y) tiles and marches along z.  Every z plane of the stage input -- the
// eight cell-centred primitives (rho, v, p, Bc) with their two-cell halo and the three staggered field components -- arrives
// ONCE as two TMA boxes (36 x (TY+3) x 8 fields, 34 x TY x 3 fields) in a shared-memory ring.  Thread (lx, ly) owns cell
// (x0 + lx, y0 + ly) of the plane and solves the three LOWER faces of its cell: x and y from the plane in shared memory,
// z by marching (left state and forward differences carried in registers).  What the neighbours need of a face solve goes
// through a double-buffered exchange area in shared memory: the upper y face of a cell is the lower y face of row ly + 1,
// the upper x face comes from lane lx + 1 by shuffle, the upper z face arrives one plane later.  So every Riemann problem
// inside a tile is solved once and no face flux ever goes to HBM -- not those of (rho, m, E), and not those of B either:
// the same exchange area holds F_d[B_t], the sign of the mass flux and the cell-centred reference EMF of the last two
// planes, from which each thread forms the three edge EMFs on the UPPER edges of its cell (all four faces and cells
// around such an edge belong to threads lx..lx+1, ly..ly+1 and planes s-1..s).  Tiles advance by 31 x (TY-1) cells: lane 31
// and row TY-1 only supply faces to their lower neighbours.
//   all stages  : E_x, E_y, E_z on the edge lattice (three doubles per cell) for the CT update in k_ct_update
//   first stage : R = flux divergence (dt is not known before the whole grid has been swept), max_cells sum_d c_d / dx
//   later stages: U_s = w0 U_0 + w (U_{s-1} - dt/dx R) applied at once (Eq. 9); U_{s-1} and U_0 of the cell are loaded
//                 ahead of the EMF evaluation and used behind it
// Per cell and stage the kernel reads 11 doubles and writes 8 (later stages: reads 21), against 57 (67) for the three
// separate sweeps of round 1 with their x-flux, partial-divergence, face-flux and sign arrays.
#pragma once
#include <cuda.h>

#include <cstdint>

#include "common.cuh"
#include "tma.cuh"
#include "physics.cuh"

namespace idfx {

constexpr int MS_TX = 32, MS_TY = 12;                // threads: 12 warps, 3 per scheduler, 168 registers each
constexpr int MS_CX = MS_TX - 1, MS_CY = MS_TY - 1;  // cells a tile completes
constexpr int MS_BW = 36, MS_BH = MS_TY + 3;         // box: columns x0-2-sh .., rows y0-2 .. y0+TY
constexpr int MS_FIELD = MS_BW * MS_BH;              // doubles of one primitive field of a plane (rho, v, p, Bc: 8 fields)
constexpr int MS_BWB = 34;                           // the staggered field is needed on the threads' own cells only: columns x0-sh ..
constexpr int MS_FIELD_B = MS_BWB * MS_TY;           // doubles of one face-field component of a plane (Bx_f, By_f, Bz_f)
constexpr int MS_PLANE = 8 * MS_FIELD + 3 * MS_FIELD_B;
constexpr uint32_t MS_BYTES_V = 8 * MS_FIELD * 8, MS_BYTES_B = 3 * MS_FIELD_B * 8;
constexpr int MS_NST = 2;                            // ring stages: the plane being solved and the next one
constexpr int MS_THREADS = MS_TX * MS_TY;
constexpr int MS_STRIDE = (MS_PLANE + 15) / 16 * 16;  // doubles between ring stages: TMA destinations are 128-byte aligned
constexpr int MS_RING_BYTES = MS_NST * MS_STRIDE * 8;
// Exchange area: what the neighbouring threads need of this thread's face solves and cell.  Quantities read only in the
// iteration that wrote them are double-buffered (the next iteration writes the other set while slow warps still read);
// those an edge between planes s-1 and s needs of BOTH planes are triple-buffered.
enum { EX_FY = 0,    // 5: F_y of (rho, m, E) in the y sweep's local order
       EX_CFY = 5,   // c_face of the y face
       EX_XBY = 6,   // F_x[B_y]                   (E_z)
       EX_YBX = 7,   // F_y[B_x]                   (E_z)
       EX_ZB = 8,    // 2: F_z[B_x], F_z[B_y]      (E_y, E_x; face s-1/2, solved in the iteration of plane s)
       EX_ECZ = 10,  // z component of the cell-centred reference EMF -(v x Bc) of the stage input (G10)
       EX_ND = 11 };
enum { EL_YBZ = 0,   // F_y[B_z]                   (E_x)
       EL_XBZ = 1,   // F_x[B_z]                   (E_y)
       EL_ECX = 2,   // x and y components of the reference EMF
       EL_ECY = 3,
       EL_ND = 4 };  // followed by the packed donor weights (one int per thread)
constexpr int MS_SLAB = MS_TY * MS_TX;                            // one exchanged quantity of one plane
constexpr int MS_EXS_DOUBLES = EX_ND * MS_SLAB;
constexpr int MS_EXL_DOUBLES = EL_ND * MS_SLAB + MS_SLAB / 2;
constexpr int MS_EXCH_BYTES = (2 * MS_EXS_DOUBLES + 3 * MS_EXL_DOUBLES) * 8;
constexpr int MS_SMEM_BYTES = MS_RING_BYTES + MS_EXCH_BYTES + MS_NST * 8 + 128;
static_assert((8 * MS_FIELD * 8) % 128 == 0, "the face-field box must land on a 128-byte boundary behind the primitives");
static_assert(MS_SMEM_BYTES <= 227 * 1024, "ring + exchange area exceed the shared memory of an SM");

struct MhdStageArgs {
  int fV0;        // first field of the stage-input primitives inside the V tensor map (0 or 11)
  int fB0;        // first field of the stage-input face field inside the B tensor map (3 x buffer)
  int chunk;      // z planes per CTA
  double* R[5];
  double* E[3];   // edge EMFs, lower-edge indexing: E[0](i,j,k) = E_x(i, j-1/2, k-1/2), E[1] = E_y(i-1/2, j, k-1/2), E[2] = E_z(i-1/2, j-1/2, k)
  DevScalars* sc;
  const double* Uin[5];  // U_{s-1}; or, with uin_is_r, the first stage's divergence R_1 (RK2: U_1 = U_0 - dt/dx R_1 is never stored)
  int uin_is_r;
  const double* U0[5];
  double* Uout[5];
  double w, w0;
};

// block-wide maximum for blocks of MS_THREADS threads; every thread must call it
__device__ __forceinline__ double block_max_ms(double v) {
  __shared__ double red[MS_THREADS / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  double m = red[0];
#pragma unroll
  for (int n = 1; n < MS_THREADS / 32; ++n) m = fmax(m, red[n]);
  return m;
}

// Lower face, along a direction with element stride ST inside a plane, of the cell at cell[0]: fields Q0..Q6 of the plane
// in the sweep's local order (rho, u_n, u_t1, u_t2, p, B_t1, B_t2); returns c_face.
template <int SOLVER, int LIM, int ST, int Q0, int Q1, int Q2, int Q3, int Q4, int Q5, int Q6>
__device__ __forceinline__ double ms_face(const double* cell, double Bn, double dx2, double gamma, double F[7]) {
  constexpr int FQ[7] = {Q0, Q1, Q2, Q3, Q4, Q5, Q6};
  double WL[7], WR[7];
#pragma unroll
  for (int n = 0; n < 7; ++n) {
    const double* f = cell + FQ[n] * MS_FIELD;
    const double m2 = f[-2 * ST], m1 = f[-ST], p0 = f[0], p1 = f[ST];
    double drop;
    face_values<LIM>(m1, m1 - m2, p0 - m1, dx2, drop, WL[n]);
    face_values<LIM>(p0, p0 - m1, p1 - p0, dx2, WR[n], drop);
  }
  return riemann<SOLVER, true>(WL, WR, Bn, gamma, F);
}

// Edge EMF in quadrant form (see edge_emf in idfx.cu): onA[r] / onB[k] the EMF carried by the two a-faces (rows r of b) and
// the two b-faces (columns k of a) that meet at the edge, cell[k][r] the cell-centred reference values, wA[r] / wB[k] the
// donor weight of the LOWER column / row for each face (1, 0 or 1/2).
template <int MODE>
__device__ __forceinline__ double ms_edge(const double onA[2], const double onB[2], const double cell[2][2], const double wA[2],
                                          const double wB[2]) {
  const double mean = 0.25 * ((onA[0] + onA[1]) + (onB[0] + onB[1]));
  if (MODE == EMF_ARITH) return mean;
  double side = 0.0;
#pragma unroll
  for (int r = 0; r < 2; ++r) side += wA[r] * (onB[0] - cell[0][r]) + (1.0 - wA[r]) * (onB[1] - cell[1][r]);
#pragma unroll
  for (int k = 0; k < 2; ++k) side += wB[k] * (onA[0] - cell[k][0]) + (1.0 - wB[k]) * (onA[1] - cell[k][1]);
  return mean + 0.25 * side;
}

// MODE: EMF_ARITH, EMF_UCT (upwind-contact) or EMF_UCT0.  OPEN: some direction does not wrap (Geom::open); the periodic box
// is its own instantiation so that none of the open-side bookkeeping is in its instruction stream.
template <int SOLVER, int LIM, int MODE, bool FIRST, bool OPEN>
__global__ void __launch_bounds__(MS_THREADS, 1) k_mhd_stage(Geom g, MhdStageArgs a, const __grid_constant__ CUtensorMap mapV,
                                                              const __grid_constant__ CUtensorMap mapB) {
  extern __shared__ __align__(128) unsigned char ms_smem_raw[];
  // the dynamic region starts after the static one (block_max_ms's scratch): align by hand, TMA wants 128 bytes
  unsigned char* ms_smem = ms_smem_raw + ((128u - (smem_u32(ms_smem_raw) & 127u)) & 127u);
  double (*ring)[MS_STRIDE] = reinterpret_cast<double (*)[MS_STRIDE]>(ms_smem);
  double* exch = reinterpret_cast<double*>(ms_smem + MS_RING_BYTES);
  uint64_t* full = reinterpret_cast<uint64_t*>(ms_smem + MS_RING_BYTES + MS_EXCH_BYTES);
  const double dx2 = g.dx * g.dx;
  const int lx = threadIdx.x & 31, ly = threadIdx.x >> 5;
  // Along an open direction (Geom::open) the tiles start one cell below the box: the ghost cell -1 is nobody's cell, but the
  // edges at index 0 are its UPPER edges, and on a periodic side they belong to cell n-1 of the far end instead.
  const int ox = OPEN ? g.open & 1 : 0, oy = OPEN ? (g.open >> 1) & 1 : 0, oz = OPEN ? (g.open >> 2) & 1 : 0;
  const int x0 = blockIdx.x * MS_CX - ox, y0 = blockIdx.y * MS_CY - oy;
  const int i = x0 + lx, j = y0 + ly;
  const int s0 = blockIdx.z * a.chunk;
  const int s1 = min(s0 + a.chunk, g.nz);
  const int np = s1 - s0 + 4;  // planes s0-2 .. s1+1; plane p of the ring is z plane s0 - 2 + p
  const bool in_tile = ly < MS_CY && j < g.ny && lx < MS_CX && i < g.nx;  // this thread owns the upper edges of its cell
  const bool complete = in_tile && (!OPEN || (i >= 0 && j >= 0));         // and the cell itself
  const bool live_row = j <= g.ny;  // warp-uniform; rows above the upper boundary face (last tile only) have nothing to supply
  if (threadIdx.x == 0) {
#pragma unroll
    for (int st = 0; st < MS_NST; ++st) mbar_init(&full[st], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  // a box must start on a 16-byte boundary: odd tiles start one column further left
  const int sh = x0 & 1;
  const int cx = IOFF + x0 - 2 - sh, cy = NG + y0 - 2, cz0 = NG + s0 - 2;
  auto issue = [&](int p) {
    uint64_t* bar = &full[p % MS_NST];
    double* dst = ring[p % MS_NST];
    mbar_expect_tx(bar, MS_BYTES_V + MS_BYTES_B);
    tma_load_4d(dst, &mapV, bar, cx, cy, cz0 + p, a.fV0);
    tma_load_4d(dst + 8 * MS_FIELD, &mapB, bar, cx + 2, cy + 2, cz0 + p, a.fB0);
  };
  if (threadIdx.x == 0)
    for (int p = 0; p < min(np, MS_NST); ++p) issue(p);
  auto wait_plane = [&](int p) { mbar_wait(&full[p % MS_NST], (p / MS_NST) & 1); };
  // call after a __syncthreads behind the last read of plane p: its ring stage is refilled with plane p + MS_NST
  auto refill = [&](int p) {
    if (threadIdx.x == 0 && p + MS_NST < np) issue(p + MS_NST);
  };
  const int so = (ly + 2) * MS_BW + lx + 2 + sh;        // this thread's cell inside one primitive field of a plane
  const int sb = 8 * MS_FIELD + ly * MS_BWB + lx + sh;  // and inside the first face-field component
  const int se = ly * MS_TX + lx;                       // and inside one slab of the exchange area
  // this thread's cell of plane p in the local order of the z sweep (rho, vz, vx, vy, p, Bcx, Bcy)
  constexpr int ZQ[7] = {0, 3, 1, 2, 4, 5, 6};
  auto own = [&](int p, double q[7]) {
    const double* r = ring[p % MS_NST] + so;
#pragma unroll
    for (int n = 0; n < 7; ++n) q[n] = r[ZQ[n] * MS_FIELD];
  };

  double dtdx = 0.0;
  if (!FIRST) dtdx = a.sc->dt_used / g.dx;  // published by the first stage's update kernel
  // ---- plane s0-2: only its own cells, for the slope of cell s0-1 ----
  double dm[7], WL[7];  // z marching: forward difference q(s) - q(s-1) and the upper face value of cell s-1
  wait_plane(0);
  if (live_row) own(0, dm);  // q(s0-2) for now
  __syncthreads();
  refill(0);
  wait_plane(1);  // every later plane is waited for one iteration ahead, by the z solve
  // periodic image of the upper neighbours (edges are stored under the index of the cell whose LOWER edge they are)
  const long long c_row = g.at(min(i, g.nx - 1), min(j, g.ny - 1), 0);
  const long long up_x = !ox && i + 1 >= g.nx ? 1 - (long long)g.nx : 1;
  const long long up_y = !oy && j + 1 >= g.ny ? (1 - (long long)g.ny) * g.sy : (long long)g.sy;
  double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};  // cell s-1: divergence of its x and y faces minus its lower z flux (global order)
  double csxy = 0.0, cfzp = 0.0;              // and c_x + c_y, c_face of its lower z face
  double smax = 0.0;
  for (int s = s0 - 1; s <= s1; ++s) {
    const int p = s - s0 + 2;                 // ring index of plane s
    const long long c = c_row + (long long)s * g.sz;
    const int it = s - s0 + 1;                // iteration count from 0
    double* ex = exch + (it & 1) * MS_EXS_DOUBLES;                                   // same-plane set of this iteration
    double* el = exch + 2 * MS_EXS_DOUBLES + (it % 3) * MS_EXL_DOUBLES;              // two-plane set of this iteration
    const double* elp = exch + 2 * MS_EXS_DOUBLES + ((it + 2) % 3) * MS_EXL_DOUBLES; // and of the previous one
    int* wts = reinterpret_cast<int*>(el + EL_ND * MS_SLAB);
    const int* wtsp = reinterpret_cast<const int*>(elp + EL_ND * MS_SLAB);
    const double* cell = ring[p % MS_NST] + so;
    const double* face = ring[p % MS_NST] + sb;
    int wcode = 0;  // donor weights of this thread's three faces: 2 bits each, sign + 1
    double dFx[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, cfx2 = 0.0, FyO[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, cfy = 0.0;
    // ---- y and x faces of plane s (the last chunk of an open z direction: also of the ghost plane nz, for the lattice plane nz) ----
    const bool xy = s < s1 || (OPEN && oz && s == g.nz);
    if (xy && live_row) {
      {
        // y: local order (rho, vy, vz, vx, p, Bcz, Bcx), normal field B_y on the lower y face
        double F[7];
        cfy = ms_face<SOLVER, LIM, MS_BW, 0, 2, 3, 1, 4, 7, 5>(cell, face[MS_FIELD_B], dx2, g.gamma, F);
#pragma unroll
        for (int n = 0; n < 5; ++n) {
          ex[(EX_FY + n) * MS_SLAB + se] = F[n];
          FyO[n] = F[n];
        }
        ex[EX_CFY * MS_SLAB + se] = cfy;
        el[EL_YBZ * MS_SLAB + se] = F[5];
        ex[EX_YBX * MS_SLAB + se] = F[6];
        if (MODE == EMF_UCT) wcode |= (F[0] > 0.0 ? 2 : (F[0] < 0.0 ? 0 : 1)) << 2;
      }
      {
        // x: local order (rho, vx, vy, vz, p, Bcy, Bcz) = field order, normal field B_x on the lower x face
        double F[7];
        const double cfx = ms_face<SOLVER, LIM, 1, 0, 1, 2, 3, 4, 6, 7>(cell, face[0], dx2, g.gamma, F);
        ex[EX_XBY * MS_SLAB + se] = F[5];
        el[EL_XBZ * MS_SLAB + se] = F[6];
        if (MODE == EMF_UCT) wcode |= (F[0] > 0.0 ? 2 : (F[0] < 0.0 ? 0 : 1));
        // upper x face from the next lane
#pragma unroll
        for (int n = 0; n < 5; ++n) dFx[n] = __shfl_down_sync(0xffffffffu, F[n], 1) - F[n];
        cfx2 = fmax(cfx, __shfl_down_sync(0xffffffffu, cfx, 1));
      }
      if (MODE != EMF_ARITH) {  // -(v x Bc) of this thread's cell
        const double vx = cell[1 * MS_FIELD], vy = cell[2 * MS_FIELD], vz = cell[3 * MS_FIELD];
        const double bx = cell[5 * MS_FIELD], by = cell[6 * MS_FIELD], bz = cell[7 * MS_FIELD];
        el[EL_ECX * MS_SLAB + se] = vz * by - vy * bz;
        el[EL_ECY * MS_SLAB + se] = vx * bz - vz * bx;
        ex[EX_ECZ * MS_SLAB + se] = vy * bx - vx * by;
      }
    }
    // ---- z face s-1/2 (s = s0-1: only the marching state is set up) ----
    double Fz[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, cfz = 0.0;
    wait_plane(p + 1);
    if (live_row) {
      double q0[7], qp[7];
      own(p, q0);
      own(p + 1, qp);
      if (s < s0) {
#pragma unroll
        for (int n = 0; n < 7; ++n) {
          const double qm = dm[n];
          dm[n] = qp[n] - q0[n];
          double drop;
          face_values<LIM>(q0[n], q0[n] - qm, dm[n], dx2, drop, WL[n]);  // cell s0-1 at its upper face
        }
      } else {
        double WR[7], F[7];
#pragma unroll
        for (int n = 0; n < 7; ++n) {
          const double dp = qp[n] - q0[n];
          double up;
          face_values<LIM>(q0[n], dm[n], dp, dx2, WR[n], up);
          dm[n] = dp;
          qp[n] = up;  // becomes the left state of the next face
        }
        cfz = riemann<SOLVER, true>(WL, WR, face[2 * MS_FIELD_B], g.gamma, F);
#pragma unroll
        for (int n = 0; n < 7; ++n) WL[n] = qp[n];
        ex[(EX_ZB + 0) * MS_SLAB + se] = F[5];
        ex[(EX_ZB + 1) * MS_SLAB + se] = F[6];
        if (MODE == EMF_UCT) wcode |= (F[0] > 0.0 ? 2 : (F[0] < 0.0 ? 0 : 1)) << 4;
        // z sweep: (n, t1, t2) = (z, x, y)
        Fz[0] = F[0]; Fz[3] = F[1]; Fz[1] = F[2]; Fz[2] = F[3]; Fz[4] = F[4];
      }
    }
    if (MODE == EMF_UCT) wts[se] = wcode;
    __syncthreads();  // the exchange set of this plane is complete; nobody reads plane s of the ring any more
    refill(p);
    if (!in_tile || s < s0) continue;  // (no barrier below this line)
    const bool closing = complete && s > s0;
    // ---- close cell s-1: its divergence is complete.  First stage: store it.  Later stages: Eq. 9 at once; the loads of
    // U_{s-1} and U_0 are issued here and used behind the EMF evaluation below, which hides their latency ----
    const long long cu = c - g.sz;
    double rt[5], uin[5], u0[5];
    if (closing) {
#pragma unroll
      for (int n = 0; n < 5; ++n) rt[n] = acc[n] + Fz[n];
      if (FIRST) {
#pragma unroll
        for (int n = 0; n < 5; ++n) a.R[n][cu] = rt[n];
        smax = fmax(smax, csxy + fmax(cfzp, cfz));  // G8
      } else {
#pragma unroll
        for (int n = 0; n < 5; ++n) {
          uin[n] = a.Uin[n][cu];
          u0[n] = a.U0[n][cu];
        }
      }
    }
    auto apply = [&]() {
      if constexpr (!FIRST) {
        if (!closing) return;
#pragma unroll
        for (int n = 0; n < 5; ++n) {
          // RK2 keeps no copy of U_1: it is U_0 - dt/dx R_1, with R_1 in place of U_{s-1} (same expression as k_ct_update's)
          const double us = a.uin_is_r ? u0[n] - dtdx * uin[n] : uin[n];
          a.Uout[n][cu] = dtdx == 0.0 ? u0[n] : a.w0 * u0[n] + a.w * (us - dtdx * rt[n]);  // Eq. 9
        }
      }
    };
    if (!xy) {
      apply();
      break;
    }
    if (!FIRST && (!OPEN || (complete && s < s1))) {  // the same lines of the next plane, on their way to L2
#pragma unroll
      for (int n = 0; n < 5; ++n) {
        prefetch_l2(a.Uin[n] + c);
        prefetch_l2(a.U0[n] + c);
      }
    }
    // ---- cell s: x and y parts of its divergence, minus its lower z flux ----
    if (!OPEN || s < s1) {
      const double* up = ex + se + MS_TX;  // row ly + 1; y sweep: (n, t1, t2) = (y, z, x)
      acc[0] = dFx[0] + (up[(EX_FY + 0) * MS_SLAB] - FyO[0]) - Fz[0];
      acc[2] = dFx[2] + (up[(EX_FY + 1) * MS_SLAB] - FyO[1]) - Fz[2];
      acc[3] = dFx[3] + (up[(EX_FY + 2) * MS_SLAB] - FyO[2]) - Fz[3];
      acc[1] = dFx[1] + (up[(EX_FY + 3) * MS_SLAB] - FyO[3]) - Fz[1];
      acc[4] = dFx[4] + (up[(EX_FY + 4) * MS_SLAB] - FyO[4]) - Fz[4];
      csxy = cfx2 + fmax(cfy, up[EX_CFY * MS_SLAB]);
      cfzp = cfz;
    }
    // ---- edge EMFs on the upper x/y edges of cell (i, j): E_z in plane s, E_x and E_y at s-1/2 ----
    {
      const int e00 = se, e10 = se + 1, e01 = se + MS_TX, e11 = se + MS_TX + 1;  // threads (lx + k, ly + r)
      auto wgt = [](int code, int shift) { return 0.5 * (double)((code >> shift) & 3); };
      double onA[2], onB[2], cl[2][2], wA[2] = {0.5, 0.5}, wB[2] = {0.5, 0.5};
      // E_z(i+1/2, j+1/2, s): a = x, b = y.  x faces of rows j, j+1 carry -F_x[B_y]; y faces of columns i, i+1 carry +F_y[B_x]
      onA[0] = -ex[EX_XBY * MS_SLAB + e10];
      onA[1] = -ex[EX_XBY * MS_SLAB + e11];
      onB[0] = ex[EX_YBX * MS_SLAB + e01];
      onB[1] = ex[EX_YBX * MS_SLAB + e11];
      if (MODE != EMF_ARITH) {
        cl[0][0] = ex[EX_ECZ * MS_SLAB + e00];
        cl[1][0] = ex[EX_ECZ * MS_SLAB + e10];
        cl[0][1] = ex[EX_ECZ * MS_SLAB + e01];
        cl[1][1] = ex[EX_ECZ * MS_SLAB + e11];
      }
      if (MODE == EMF_UCT) {
        wA[0] = wgt(wts[e10], 0);
        wA[1] = wgt(wts[e11], 0);
        wB[0] = wgt(wts[e01], 2);
        wB[1] = wgt(wts[e11], 2);
      }
      if (!OPEN || s < s1) a.E[2][c + up_x + up_y] = ms_edge<MODE>(onA, onB, cl, wA, wB);
      // E_x(i, j+1/2, s-1/2): a = y, b = z.  y faces (j+1/2) of planes s-1, s carry -F_y[B_z]; z faces (s-1/2) of rows j, j+1 carry +F_z[B_y]
      onA[0] = -elp[EL_YBZ * MS_SLAB + e01];
      onA[1] = -el[EL_YBZ * MS_SLAB + e01];
      onB[0] = ex[(EX_ZB + 1) * MS_SLAB + e00];
      onB[1] = ex[(EX_ZB + 1) * MS_SLAB + e01];
      if (MODE != EMF_ARITH) {
        cl[0][0] = elp[EL_ECX * MS_SLAB + e00];   // [column in y][row in z]
        cl[1][0] = elp[EL_ECX * MS_SLAB + e01];
        cl[0][1] = el[EL_ECX * MS_SLAB + e00];
        cl[1][1] = el[EL_ECX * MS_SLAB + e01];
      }
      if (MODE == EMF_UCT) {
        wA[0] = wgt(wtsp[e01], 2);
        wA[1] = wgt(wts[e01], 2);
        wB[0] = wgt(wts[e00], 4);
        wB[1] = wgt(wts[e01], 4);
      }
      if (!OPEN || i >= 0) a.E[0][c + up_y] = ms_edge<MODE>(onA, onB, cl, wA, wB);
      // E_y(i+1/2, j, s-1/2): a = z, b = x.  z faces (s-1/2) of columns i, i+1 carry -F_z[B_x]; x faces (i+1/2) of planes s-1, s carry +F_x[B_z]
      onA[0] = -ex[(EX_ZB + 0) * MS_SLAB + e00];
      onA[1] = -ex[(EX_ZB + 0) * MS_SLAB + e10];
      onB[0] = elp[EL_XBZ * MS_SLAB + e10];
      onB[1] = el[EL_XBZ * MS_SLAB + e10];
      if (MODE != EMF_ARITH) {
        cl[0][0] = elp[EL_ECY * MS_SLAB + e00];   // [column in z][row in x]
        cl[1][0] = el[EL_ECY * MS_SLAB + e00];
        cl[0][1] = elp[EL_ECY * MS_SLAB + e10];
        cl[1][1] = el[EL_ECY * MS_SLAB + e10];
      }
      if (MODE == EMF_UCT) {
        wA[0] = wgt(wts[e00], 4);
        wA[1] = wgt(wts[e10], 4);
        wB[0] = wgt(wtsp[e10], 0);
        wB[1] = wgt(wts[e10], 0);
      }
      if (!OPEN || j >= 0) a.E[1][c + up_x] = ms_edge<MODE>(onA, onB, cl, wA, wB);
    }
    apply();
  }
  if (FIRST) {
    const double m = block_max_ms(complete ? smax / g.dx : 0.0);
    if (threadIdx.x == 0) atomicMax(&a.sc->smax_bits, (unsigned long long)__double_as_longlong(m));
  }
}

}  // namespace idfx
