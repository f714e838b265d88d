// idfx.cu — kernels and C ABI of the idfx CUDA path (sm_100a, fp64).  Interface: include/idfx.h.
//
// Data layout in HBM: structure of arrays; every field is a padded box
// [nz+4][ny+4][pitch] doubles with 2 ghost layers in y and z and, in x, the active cells starting at
// column IOFF = 16 (a 128-byte boundary) with ghost columns 14,15 and nx+16,nx+17; pitch is a multiple of
// 16 doubles.  All fields live in the caller's workspace.
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>  // header-only; ranges cost nothing unless a profiler (nsys, ncu --nvtx) is attached

#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/idfx.h"
#include "common.cuh"
#include "physics.cuh"
#include "hd_stage.cuh"
#include "mhd_stage.cuh"

namespace idfx {

// ---------------------------------------------------------------------------------------------
// copy-in / copy-out between the caller's contiguous arrays and the padded fields
// ---------------------------------------------------------------------------------------------
struct FieldList {
  double* f[14];
  int n;
};

__global__ void k_pack(Geom g, FieldList dst, const double* __restrict__ src) {
  int i, j, k;
  if (!cell_of_thread(g, i, j, k)) return;
  const long long c = g.at(i, j, k);
  const long long s = ((long long)k * g.ny + j) * g.nx + i;
  for (int n = 0; n < dst.n; ++n) dst.f[n][c] = src[n * g.nc + s];
}

__global__ void k_unpack(Geom g, FieldList srcf, double* __restrict__ dst) {
  int i, j, k;
  if (!cell_of_thread(g, i, j, k)) return;
  const long long c = g.at(i, j, k);
  const long long s = ((long long)k * g.ny + j) * g.nx + i;
  for (int n = 0; n < srcf.n; ++n) dst[n * g.nc + s] = srcf.f[n][c];
}

// a1: ghost fill of a list of fields, one thread per ghost cell.  Periodic: every ghost cell copies from its
// wrapped active image, which equals the sequential x, y, z fill of O2 (i).  Outflow (HD only): from the
// nearest active cell, which equals the sequential zero-gradient fill.
// T: unsigned int wherever the count of ghost cells fits (64-bit divisions cost an order of magnitude more).
template <typename T>
__device__ __forceinline__ void fill_ghost_cell(const Geom& g, const FieldList& fl) {
  const T px = (T)(g.nx + 2 * NG), py = (T)(g.ny + 2 * NG);
  const T nZ = (T)(2 * NG) * py * px;             // k in ghost
  const T nY = (T)g.nz * (T)(2 * NG) * px;        // k active, j in ghost
  const T nX = (T)g.nz * (T)g.ny * (T)(2 * NG);
  T t = (T)blockIdx.x * (T)blockDim.x + (T)threadIdx.x;
  int i, j, k;
  if (t < nZ) {
    i = (int)(t % px) - NG;
    const T r = t / px;
    j = (int)(r % py) - NG;
    const int kk = (int)(r / py);
    k = kk < NG ? kk - NG : g.nz + kk - NG;
  } else if ((t -= nZ) < nY) {
    i = (int)(t % px) - NG;
    const T r = t / px;
    const int jj = (int)(r % (T)(2 * NG));
    j = jj < NG ? jj - NG : g.ny + jj - NG;
    k = (int)(r / (T)(2 * NG));
  } else if ((t -= nY) < nX) {
    const int ii = (int)(t % (T)(2 * NG));
    i = ii < NG ? ii - NG : g.nx + ii - NG;
    const T r = t / (T)(2 * NG);
    j = (int)(r % (T)g.ny);
    k = (int)(r / (T)g.ny);
  } else {
    return;
  }
  // the wrapped active image (extents are at least 2 NG, so one box length is enough)
  int is = i < 0 ? i + g.nx : (i >= g.nx ? i - g.nx : i);
  int js = j < 0 ? j + g.ny : (j >= g.ny ? j - g.ny : j);
  int ks = k < 0 ? k + g.nz : (k >= g.nz ? k - g.nz : k);
  if (g.outflow) {  // zero gradient: the nearest active cell
    is = min(max(i, 0), g.nx - 1);
    js = min(max(j, 0), g.ny - 1);
    ks = min(max(k, 0), g.nz - 1);
  }
  const long long d = g.at(i, j, k), s = g.at(is, js, ks);
  // all loads first: a ghost cell is one strided access per field, and the copy is bound by how many are in flight
  double v[14];
#pragma unroll
  for (int n = 0; n < 14; ++n)
    if (n < fl.n) v[n] = fl.f[n][s];
#pragma unroll
  for (int n = 0; n < 14; ++n)
    if (n < fl.n) fl.f[n][d] = v[n];
}

template <typename T>
__global__ void k_fill_ghost(Geom g, FieldList fl) {
  fill_ghost_cell<T>(g, fl);
}

// the same fill after the first stage of a cycle whose stages read the conserved fields (hd_stage_u.cuh): there is no update
// kernel between the stages, so one thread of this launch publishes the dt the reduction of the stage just found
template <typename T>
__global__ void k_fill_ghost_dt(Geom g, FieldList fl, DevScalars* sc, double dt_fixed, double cfl) {
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    bool lands;
    const double dt = first_stage_dt(sc, dt_fixed, cfl, lands);
    publish_dt(sc, dt, lands);
  }
  fill_ghost_cell<T>(g, fl);
}

// a1 one direction and one side at a time ("sequential x -> y -> z exchange", the order that also gets
// edges and corners right): a slab of NG layers normal to direction d that spans the active cells of the directions
// above d and the whole padded extent of the directions below it.
//   SLAB_COPY   ghost slab <- a slab of the same field (periodic image, or with `clamp` the nearest active layer)
//   SLAB_PACK   the NG active layers next to the side -> a contiguous buffer [field][z][y][x of the slab]
//   SLAB_UNPACK a contiguous buffer -> the ghost slab of that side
// Under a domain decomposition the buffer packed on one rank's upper side is unpacked on its upper neighbour's lower side.
enum { SLAB_COPY = 0, SLAB_PACK = 1, SLAB_UNPACK = 2 };

struct SlabGeom {
  int lo[3], ext[3];  // first index and extent of the slab in x, y, z (ext[d] = NG)
  int d, src0, clamp; // SLAB_COPY: first source layer along d, or the one layer every ghost layer copies
  long long count;    // cells of the slab
};

inline SlabGeom slab_geom(const Geom& g, int d, int side, int mode, int clamp) {
  SlabGeom s;
  const int n[3] = {g.nx, g.ny, g.nz};
  for (int q = 0; q < 3; ++q) {
    s.lo[q] = q < d ? -NG : 0;
    s.ext[q] = q < d ? n[q] + 2 * NG : n[q];
  }
  s.ext[d] = NG;
  s.d = d;
  s.clamp = clamp;
  if (mode == SLAB_PACK) {
    s.lo[d] = side ? n[d] - NG : 0;
    s.src0 = 0;
  } else {
    s.lo[d] = side ? n[d] : -NG;
    s.src0 = clamp ? (side ? n[d] - 1 : 0) : (side ? 0 : n[d] - NG);
  }
  s.count = (long long)s.ext[0] * s.ext[1] * s.ext[2];
  return s;
}

template <int MODE>
__global__ void k_slab(Geom g, SlabGeom sg, FieldList fl, double* __restrict__ buf) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= sg.count) return;
  int l[3];
  l[0] = (int)(t % sg.ext[0]);
  const long long r = t / sg.ext[0];
  l[1] = (int)(r % sg.ext[1]);
  l[2] = (int)(r / sg.ext[1]);
  int idx[3] = {sg.lo[0] + l[0], sg.lo[1] + l[1], sg.lo[2] + l[2]};
  const long long cell = g.at(idx[0], idx[1], idx[2]);
  if (MODE == SLAB_COPY) {
    idx[sg.d] = sg.clamp ? sg.src0 : sg.src0 + l[sg.d];
    const long long src = g.at(idx[0], idx[1], idx[2]);
    for (int n = 0; n < fl.n; ++n) fl.f[n][cell] = fl.f[n][src];
  } else if (MODE == SLAB_PACK) {
    for (int n = 0; n < fl.n; ++n) buf[n * sg.count + t] = fl.f[n][cell];
  } else {
    for (int n = 0; n < fl.n; ++n) fl.f[n][cell] = buf[n * sg.count + t];
  }
}

// Pack and unpack in one: the NG active layers next to one side of a sub-box go straight into the ghost layers of the
// opposite side of its neighbour.  The neighbour's fields may live on another GPU of the same process: the stores are then
// peer stores over NVLink (coalesced along x, no staging buffer, one launch per slab instead of two).
__global__ void k_slab_push(Geom gs, SlabGeom from, FieldList fs, Geom gd, SlabGeom to, FieldList fd) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= from.count) return;
  const int l0 = (int)(t % from.ext[0]);
  const long long r = t / from.ext[0];
  const int l1 = (int)(r % from.ext[1]), l2 = (int)(r / from.ext[1]);
  const long long src = gs.at(from.lo[0] + l0, from.lo[1] + l1, from.lo[2] + l2);
  const long long dst = gd.at(to.lo[0] + l0, to.lo[1] + l1, to.lo[2] + l2);
  for (int n = 0; n < fs.n; ++n) fd.f[n][dst] = fs.f[n][src];
}

// ---------------------------------------------------------------------------------------------
// a2: cell-centred B and cons <-> prim
// ---------------------------------------------------------------------------------------------
struct StateArgs {
  double* U[5];
  double* V[11];  // rho, v, p, Bc, Ec = -(v x Bc)
  const double* Bf[3];
  DevScalars* sc;
};

// set_state (O1): V[0..4] hold the primitives; writes Bc into V[5..7] and the conserved state into U.
template <bool MHD>
__global__ void k_cons_from_prim(Geom g, StateArgs a) {
  int i, j, k;
  if (!cell_of_thread(g, i, j, k)) return;
  const long long c = g.at(i, j, k);
  double bx = 0.0, by = 0.0, bz = 0.0;
  if (MHD) {
    // right faces through the periodic image (face ghosts are not filled yet); along an open direction the ghost face,
    // which is filled before this kernel runs
    bx = 0.5 * (a.Bf[0][c] + a.Bf[0][g.at(i + 1 == g.nx && !(g.open & 1) ? 0 : i + 1, j, k)]);
    by = 0.5 * (a.Bf[1][c] + a.Bf[1][g.at(i, j + 1 == g.ny && !(g.open & 2) ? 0 : j + 1, k)]);
    bz = 0.5 * (a.Bf[2][c] + a.Bf[2][g.at(i, j, k + 1 == g.nz && !(g.open & 4) ? 0 : k + 1)]);
    a.V[5][c] = bx;
    a.V[6][c] = by;
    a.V[7][c] = bz;
  }
  const double rho = a.V[0][c], vx = a.V[1][c], vy = a.V[2][c], vz = a.V[3][c], p = a.V[4][c];
  if (MHD && a.V[8]) {  // only PPM keeps -(v x Bc) in memory
    a.V[8][c] = vz * by - vy * bz;
    a.V[9][c] = vx * bz - vz * bx;
    a.V[10][c] = vy * bx - vx * by;
  }
  if (!(rho > 0.0) || !(p > 0.0)) a.sc->flag = 1;
  a.U[0][c] = rho;
  a.U[1][c] = rho * vx;
  a.U[2][c] = rho * vy;
  a.U[3][c] = rho * vz;
  a.U[4][c] = p / (g.gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * (bx * bx + by * by + bz * bz);
}

__device__ __forceinline__ void prim_from_cons(double gm1, double rho, double mx, double my, double mz, double E,
                                               double bx, double by, double bz, double& vx, double& vy, double& vz,
                                               double& p) {
  const double ir = 1.0 / rho;
  vx = mx * ir;
  vy = my * ir;
  vz = mz * ir;
  p = gm1 * (E - 0.5 * rho * (vx * vx + vy * vy + vz * vz) - 0.5 * (bx * bx + by * by + bz * bz));
}

// get_state: primitives from the master state into scratch fields (Bf ghosts are valid whenever this runs).
// Optional pressure floor (off unless idfx_set_option_real sets it; the paper describes none, reading G13/G20): a pressure
// below the floor is raised to it and the total energy rewritten to match.  Returns true when it acted.
__device__ __forceinline__ bool pressure_floor(const Geom& g, DevScalars* sc, double rho, double vx, double vy, double vz,
                                               double bx, double by, double bz, double& p, double& E) {
  if (!(g.pfloor > 0.0) || !(p < g.pfloor)) return false;
  // a cell floored before recomputes to the floor within rounding: it is not floored (or counted) again, so a cycle that
  // changes nothing (idfx_advance_to past t_end) leaves the count alone too
  const bool acts = p < g.pfloor * (1.0 - 1e-9);
  p = g.pfloor;
  if (!acts) return false;
  E = p / (g.gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * (bx * bx + by * by + bz * bz);
  atomicAdd(&sc->nfloor, 1ull);
  return true;
}

// The stage-input primitives V are left untouched so that reading the state never perturbs the run.
template <bool MHD>
__global__ void k_prim_from_cons(Geom g, StateArgs a) {
  int i, j, k;
  if (!cell_of_thread(g, i, j, k)) return;
  const long long c = g.at(i, j, k);
  double bx = 0.0, by = 0.0, bz = 0.0;
  if (MHD) {
    bx = 0.5 * (a.Bf[0][c] + a.Bf[0][c + 1]);
    by = 0.5 * (a.Bf[1][c] + a.Bf[1][c + g.sy]);
    bz = 0.5 * (a.Bf[2][c] + a.Bf[2][c + g.sz]);
  }
  double vx, vy, vz, p;
  const double rho = a.U[0][c];
  if (MHD) {
    prim_from_cons(g.gamma - 1.0, rho, a.U[1][c], a.U[2][c], a.U[3][c], a.U[4][c], bx, by, bz, vx, vy, vz, p);
  } else {  // the bits the stage kernels form (hd_stage.cuh)
    const double u[5] = {rho, a.U[1][c], a.U[2][c], a.U[3][c], a.U[4][c]};
    double v[5];
    hd_prims(g.gamma - 1.0, u, v);
    vx = v[1], vy = v[2], vz = v[3], p = v[4];
  }
  if (g.pfloor > 0.0 && p < g.pfloor) p = g.pfloor;  // a floored cell recomputes to the floor within rounding
  a.V[0][c] = rho;
  a.V[1][c] = vx;
  a.V[2][c] = vy;
  a.V[3][c] = vz;
  a.V[4][c] = p;
}

// ---------------------------------------------------------------------------------------------
// a3 + a4: reconstruct -> Riemann -> flux on the left face of every active cell, one direction.
// q[] are the primitive fields permuted for the sweep direction (rho, u, v, w, p, B_t1, B_t2), bn the
// staggered normal field, sd the stride along the sweep.  Faces in the ghost layers are never computed:
// they are periodic images of these and consumers wrap their indices instead.
// ---------------------------------------------------------------------------------------------
struct FluxArgs {
  const double* q[7];
  const double* bn;
  long long sd;
  double* F[7];  // local ordering (rho, m_n, m_t1, m_t2, E, B_t1, B_t2); F[5], F[6] unused in HD
  double* cf;    // c_face
};

// FMODE 0: fluxes and c_face; 1: c_face only; 2: what the 2D-HLL EMF needs of the face (G21):
// F[0] = alpha+ = max(0, S_R), F[1] = alpha- = max(0, -S_L), F[2], F[3] = the HLL-weighted transverse velocities;
// 3: what the 2D-HLLD EMF needs (G24, hlld_uct_face): F[0] = dirL, F[1] = kL, F[2] = kR, F[3], F[4] = the effective velocities.
template <int SOLVER, int LIM, bool MHD, int FMODE>
__global__ void __launch_bounds__(128) k_flux_face(Geom g, FluxArgs a) {
  int i, j, k;
  if (!cell_of_thread(g, i, j, k)) return;
  const long long c = g.at(i, j, k);
  constexpr int NQ = MHD ? 7 : 5;
  const double dx2 = g.dx * g.dx;
  double WL[7], WR[7];
#pragma unroll
  for (int n = 0; n < NQ; ++n) {
    const double* __restrict__ q = a.q[n];
    const double qm2 = q[c - 2 * a.sd], qm1 = q[c - a.sd], q0 = q[c], qp1 = q[c + a.sd];
    double lo_unused, hi_unused;
    face_values<LIM>(qm1, qm1 - qm2, q0 - qm1, dx2, lo_unused, WL[n]);
    face_values<LIM>(q0, q0 - qm1, qp1 - q0, dx2, WR[n], hi_unused);
  }
  if (!MHD) WL[5] = WL[6] = WR[5] = WR[6] = 0.0;
  const double Bn = MHD ? a.bn[c] : 0.0;  // G3
  if (FMODE == 1) {
    double SL, SR;
    outer_speeds<MHD>(WL, WR, Bn, g.gamma, SL, SR);
    a.cf[c] = fmax(fabs(SL), fabs(SR));
  } else if (FMODE == 2) {
    double SL, SR;
    outer_speeds<MHD>(WL, WR, Bn, g.gamma, SL, SR);
    const double ap = fmax(0.0, SR), am = fmax(0.0, -SL);
    const double inv = 1.0 / (ap + am);
    a.F[0][c] = ap;
    a.F[1][c] = am;
    a.F[2][c] = (ap * WL[2] + am * WR[2]) * inv;
    a.F[3][c] = (ap * WL[3] + am * WR[3]) * inv;
  } else if (FMODE == 3) {
    double dirL, kL, kR, vt1, vt2;
    hlld_uct_face(WL, WR, Bn, g.gamma, dirL, kL, kR, vt1, vt2);
    a.F[0][c] = dirL;
    a.F[1][c] = kL;
    a.F[2][c] = kR;
    a.F[3][c] = vt1;
    a.F[4][c] = vt2;
  } else {
    double F[7];
    a.cf[c] = riemann<SOLVER, MHD>(WL, WR, Bn, g.gamma, F);
#pragma unroll
    for (int n = 0; n < NQ; ++n) a.F[n][c] = F[n];
  }
}

// ---------------------------------------------------------------------------------------------
// PPM (reading G22) outside the tuned sweeps: the same left-face solve with five-cell stencils.  The fields
// carry two ghost layers and PPM reaches three cells back, so positions along the sweep are wrapped (periodic boxes only).
// Along the six cells id-3 .. id+2 there are five interfaces; each is evaluated once and shared by the two parabolas.
// FMODE 0: fluxes (hydro part to F[0..4], field part to F[5..6]), c_face and the sign of the mass flux; 1: c_face only.
// ---------------------------------------------------------------------------------------------
struct FluxPpmArgs {
  const double* q[7];
  const double* bn;
  long long sd;
  int dir;
  double* F[7];
  double* cf;
  signed char* sg;  // null unless the upwind-contact EMF needs it
};

template <int SOLVER, bool MHD, int FMODE>
__global__ void __launch_bounds__(128) k_flux_face_ppm(Geom g, FluxPpmArgs a) {
  int ijk[3];
  if (!cell_of_thread(g, ijk[0], ijk[1], ijk[2])) return;
  const long long c = g.at(ijk[0], ijk[1], ijk[2]);
  const int nd = a.dir == 0 ? g.nx : (a.dir == 1 ? g.ny : g.nz), id = ijk[a.dir];
  long long off[6];
#pragma unroll
  for (int m = 0; m < 6; ++m) {
    int w = id + m - 3;
    w = w < 0 ? w + nd : (w >= nd ? w - nd : w);
    off[m] = c + (long long)(w - id) * a.sd;
  }
  constexpr int NQ = MHD ? 7 : 5;
  double WL[7], WR[7];
#pragma unroll
  for (int n = 0; n < NQ; ++n) {
    const double* __restrict__ q = a.q[n];
    double v[6];
#pragma unroll
    for (int m = 0; m < 6; ++m) v[m] = q[off[m]];
    // interfaces between v[1]|v[2], v[2]|v[3] (the face being solved), v[3]|v[4]
    const double e12 = ppm_edge(v[0], v[1], v[2], v[3]);
    const double e23 = ppm_edge(v[1], v[2], v[3], v[4]);
    const double e34 = ppm_edge(v[2], v[3], v[4], v[5]);
    double unused;
    ppm_limit(v, e12, e23, unused, WL[n]);       // cell id-1 (v[2]) at its upper face
    ppm_limit(v + 1, e23, e34, WR[n], unused);   // cell id (v[3]) at its lower face
  }
  if (!MHD) WL[5] = WL[6] = WR[5] = WR[6] = 0.0;
  const double Bn = MHD ? a.bn[c] : 0.0;  // G3
  if (FMODE == 1) {
    double SL, SR;
    outer_speeds<MHD>(WL, WR, Bn, g.gamma, SL, SR);
    a.cf[c] = fmax(fabs(SL), fabs(SR));
  } else {
    double F[7];
    a.cf[c] = riemann<SOLVER, MHD>(WL, WR, Bn, g.gamma, F);
#pragma unroll
    for (int n = 0; n < NQ; ++n) a.F[n][c] = F[n];
    if (a.sg) a.sg[c] = flux_sign(F[0]);
  }
}

// ---------------------------------------------------------------------------------------------
// a5: flux divergence R = sum_d [F_d(i+1/2) - F_d(i-1/2)] (Eq. 5); a9: block max of sum_d c_d/dx
// ---------------------------------------------------------------------------------------------
struct RhsArgs {
  const double* F[3][5];
  const double* cf[3];
  double* R[5];
  DevScalars* sc;
};

template <bool WANT_R, bool WANT_DT>
__global__ void __launch_bounds__(128) k_rhs(Geom g, RhsArgs a) {
  int i, j, k;
  const bool active = cell_of_thread(g, i, j, k);
  double s = 0.0;
  if (active) {
    const long long c = g.at(i, j, k);
    const long long cp[3] = {g.at(i + 1 == g.nx ? 0 : i + 1, j, k), g.at(i, j + 1 == g.ny ? 0 : j + 1, k),
                             g.at(i, j, k + 1 == g.nz ? 0 : k + 1)};
    if (WANT_R) {
      double r[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        r[0] += a.F[d][0][cp[d]] - a.F[d][0][c];
        r[1 + d] += a.F[d][1][cp[d]] - a.F[d][1][c];
        r[1 + (d + 1) % 3] += a.F[d][2][cp[d]] - a.F[d][2][c];
        r[1 + (d + 2) % 3] += a.F[d][3][cp[d]] - a.F[d][3][c];
        r[4] += a.F[d][4][cp[d]] - a.F[d][4][c];
      }
#pragma unroll
      for (int n = 0; n < 5; ++n) a.R[n][c] = r[n];
    }
    if (WANT_DT) {
#pragma unroll
      for (int d = 0; d < 3; ++d) s += fmax(a.cf[d][c], a.cf[d][cp[d]]);  // G8
      s /= g.dx;
    }
  }
  if (WANT_DT) {
    const double m = block_max_128(s);
    if (threadIdx.x == 0) atomicMax(&a.sc->smax_bits, (unsigned long long)__double_as_longlong(m));
  }
}

// ---------------------------------------------------------------------------------------------
// a6: edge EMFs (O10).  Thread (i,j,k) owns the three lower edges of its cell:
//   E[0] = E_x(i, j-1/2, k-1/2), E[1] = E_y(i-1/2, j, k-1/2), E[2] = E_z(i-1/2, j-1/2, k).
// For component c with (a,b,c) cyclic:  E_c^(a) = -F_a[B_b] = -FB[a][0],  E_c^(b) = +F_b[B_a] = +FB[b][1].
// ---------------------------------------------------------------------------------------------
// read-only load of data no thread of the running kernel writes (ld.global.nc): the compiler may then move it across the
// kernel's stores, which lets the update phase of k_ct_update issue loads of several cells at once.  Used for the flux
// divergence, the face fluxes and signs, the stage-input face field and E^c, the saved face field: none of these
// buffers is ever the destination of the same launch (run_stage)
template <typename T>
__device__ __forceinline__ T ldro(const T* p) {
  return __ldg(p);
}

struct EmfArgs {
  const double* FB[3][2];  // FB[d][0] = F_d[B_t1], FB[d][1] = F_d[B_t2] on the left d-faces
  const signed char* SG[3];  // sign of the mass flux F_d[rho] on the left d-faces
  const double* Ec[3];     // cell-centred reference EMF -(v x Bc) of the stage input, with ghosts (G10)
  const double* Eg[3];     // EMF_UCT_HLL: edge EMFs already evaluated by k_emf_hll2d
};

// E_c on the lower (a-1/2, b-1/2) edge of active cell idx, (a, b, c) cyclic (Gardiner & Stone 2005).
// Written in "quadrant form".  Four faces meet at the edge: the a-faces of rows ib-1 and ib (they carry E^(a) = -F_a[B_b])
// and the b-faces of columns ia-1 and ia (E^(b) = +F_b[B_a]); four cells touch it, (column, row) in {ia-1, ia} x {ib-1, ib}.
//   arithmetic:  E = mean of the four face values
//   E^c:         every face also looks sideways into one of its two cells -- the one its mass flux comes from -- and adds
//                a quarter of (transverse face value on that cell's side of the edge - cell-centred reference value):
//                  a-face of row r, donor column k:  E^(b)[k] - E^ref[k][r]
//                  b-face of column k, donor row r:  E^(a)[r] - E^ref[k][r]
//                which is Gardiner & Stone's (dx/8)(dE/dx at the two quarter points) with the one-sided differences
//                2 (E_face - E_ref) and 2 (E_ref - E_face) written out and summed; a vanishing mass flux weighs both cells 1/2
//   E^0:         the same with both cells weighted 1/2 on every face
// The donor weight of the lower cell is (1 + s)/2 with s the stored sign of the mass flux (+1, -1, 0), so the upwind choice
// is arithmetic on {0, 1/2, 1} rather than a branch.
template <int MODE>
__device__ __forceinline__ double edge_emf(const Geom& g, const EmfArgs& A, const int idx[3], int c) {
  if (MODE == EMF_UCT_HLL) return A.Eg[c][g.at(idx[0], idx[1], idx[2])];
  const int a = (c + 1) % 3, b = (c + 2) % 3;
  const int ext[3] = {g.nx, g.ny, g.nz};
  const long long step[3] = {1, g.sy, g.sz};
  const long long P = g.at(idx[0], idx[1], idx[2]);
  // one step down in a / in b: flux and sign arrays carry no ghosts (their periodic image is taken), cell arrays do
  const long long downA = idx[a] == 0 ? (long long)(ext[a] - 1) * step[a] : -step[a];
  const long long downB = idx[b] == 0 ? (long long)(ext[b] - 1) * step[b] : -step[b];
  const double* __restrict__ fluxA = A.FB[a][0];  // F_a[B_b]
  const double* __restrict__ fluxB = A.FB[b][1];  // F_b[B_a]
  const double onA[2] = {-ldro(fluxA + P + downB), -ldro(fluxA + P)};  // by row:    ib-1, ib
  const double onB[2] = {ldro(fluxB + P + downA), ldro(fluxB + P)};    // by column: ia-1, ia
  const double mean = 0.25 * ((onA[0] + onA[1]) + (onB[0] + onB[1]));
  if (MODE == EMF_ARITH) return mean;
  const double* __restrict__ ref = A.Ec[c];  // -(v x Bc)_c of the stage input, with ghosts (G10)
  double cell[2][2];                         // [column][row]
  cell[1][1] = ldro(ref + P);
  cell[0][1] = ldro(ref + P - step[a]);
  cell[1][0] = ldro(ref + P - step[b]);
  cell[0][0] = ldro(ref + P - step[a] - step[b]);
  double wA[2] = {0.5, 0.5}, wB[2] = {0.5, 0.5};  // weight of the LOWER cell: column ia-1 for the a-faces, row ib-1 for the b-faces
  if (MODE == EMF_UCT) {
    wA[0] = 0.5 + 0.5 * (double)ldro(A.SG[a] + P + downB);
    wA[1] = 0.5 + 0.5 * (double)ldro(A.SG[a] + P);
    wB[0] = 0.5 + 0.5 * (double)ldro(A.SG[b] + P + downA);
    wB[1] = 0.5 + 0.5 * (double)ldro(A.SG[b] + P);
  }
  double side = 0.0;
#pragma unroll
  for (int r = 0; r < 2; ++r)  // a-face of row r
    side += wA[r] * (onB[0] - cell[0][r]) + (1.0 - wA[r]) * (onB[1] - cell[1][r]);
#pragma unroll
  for (int k = 0; k < 2; ++k)  // b-face of column k
    side += wB[k] * (onA[0] - cell[k][0]) + (1.0 - wB[k]) * (onA[1] - cell[k][1]);
  return mean + 0.25 * side;
}

// ---------------------------------------------------------------------------------------------
// 2D-HLL edge EMF (reading G21).  Thread (i, j, k) evaluates the three lower edges of its cell.  At an edge
// along c the induction flux v_a B_b is transported across the edge along a, and v_b B_a along b; each is a one-dimensional
// HLL flux of a staggered field between its two edge-side values:
//   T(q; lo, hi) = [al+ q_lo (v_lo + al-) + al- q_hi (v_hi - al+)] / (al+ + al-)      (= the HLL average of v q, regrouped)
//   E_c = -T(B_b along a) + T(B_a along b)
// with lo / hi the staggered field and the face velocity reconstructed to the edge from either side, and al+- the larger
// one-sided speed of the two faces normal to the transport direction that touch the edge.  Inputs: the face quantities of
// k_flux_face<FMODE 2> (no ghosts: indices wrap) and the staggered field (ghosts filled).
// ---------------------------------------------------------------------------------------------
struct Hll2dArgs {
  // per direction d, on the left d-faces: 2D-HLL: alpha+, alpha-, v_t1 (component d+1), v_t2 (component d+2);
  // 2D-HLLD: dirL, kL, kR, vt1, vt2 of hlld_uct_face
  const double* H[3][5];
  const double* Bf[3];
  double* E[3];
};

// values at the point between samples m1 and p0 of a line of four samples, seen from below and from above (S2 along the line)
template <int LIM>
__device__ __forceinline__ void edge_sides(double m2, double m1, double p0, double p1, double dx2, double& below, double& above) {
  double drop;
  face_values<LIM>(m1, m1 - m2, p0 - m1, dx2, drop, below);
  face_values<LIM>(p0, p0 - m1, p1 - p0, dx2, above, drop);
}

__device__ __forceinline__ double hll_transport(double alp, double alm, double v_lo, double q_lo, double v_hi, double q_hi) {
  return (alp * q_lo * (v_lo + alm) + alm * q_hi * (v_hi - alp)) / (alp + alm);
}

// 2D-HLLD (reading G24): the transport of staggered component q across the edge with the response of the HLLD face solves
// normal to it: plain upwind transport by the reconstructed face velocity on the side the contact points from, plus kL q_lo - kR q_hi
__device__ __forceinline__ double hlld_transport(double dirL, double kL, double kR, double v_lo, double q_lo, double v_hi, double q_hi) {
  return q_lo * (dirL * v_lo + kL) + q_hi * ((1.0 - dirL) * v_hi - kR);
}

template <int LIM, bool HLLD>
__global__ void __launch_bounds__(128) k_emf_hll2d(Geom g, Hll2dArgs h) {
  int cellidx[3];
  if (!cell_of_thread(g, cellidx[0], cellidx[1], cellidx[2])) return;
  const int ext[3] = {g.nx, g.ny, g.nz};
  const long long step[3] = {1, g.sy, g.sz};
  const long long P = g.at(cellidx[0], cellidx[1], cellidx[2]);
  const double dx2 = g.dx * g.dx;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double T[2];  // transport along a = c+1 (of B_b), along b = c+2 (of B_a)
#pragma unroll
    for (int leg = 0; leg < 2; ++leg) {
      const int along = (c + 1 + leg) % 3;   // direction of the transport across the edge
      const int other = (c + 2 - leg) % 3;   // component of the staggered field carried = normal of the faces it lives on
      // periodic images of the face samples at -2, -1, +1 along `along` (ghost-free arrays)
      long long w[4];
#pragma unroll
      for (int m = 0; m < 4; ++m) {
        int t = cellidx[along] + m - 2;
        t = t < 0 ? t + ext[along] : (t >= ext[along] ? t - ext[along] : t);
        w[m] = P + (long long)(t - cellidx[along]) * step[along];
      }
      // velocity component `along` on the `other`-faces: slot 2 of that sweep is component other+1, slot 3 is other+2
      const double* __restrict__ vel = h.H[other][((along - other + 3) % 3 == 1 ? 2 : 3) + (HLLD ? 1 : 0)];
      const double* __restrict__ fld = h.Bf[other];
      double q_lo, q_hi, v_lo, v_hi;
      edge_sides<LIM>(fld[P - 2 * step[along]], fld[P - step[along]], fld[P], fld[P + step[along]], dx2, q_lo, q_hi);
      edge_sides<LIM>(vel[w[0]], vel[w[1]], vel[P], vel[w[3]], dx2, v_lo, v_hi);
      // the two `along`-faces touching the edge are neighbours in `other`
      const int t = cellidx[other] - 1;
      const long long nb = P + (long long)((t < 0 ? t + ext[other] : t) - cellidx[other]) * step[other];
      if (HLLD) {  // the mean response of the two faces
        const double dirL = 0.5 * (h.H[along][0][nb] + h.H[along][0][P]);
        const double kL = 0.5 * (h.H[along][1][nb] + h.H[along][1][P]), kR = 0.5 * (h.H[along][2][nb] + h.H[along][2][P]);
        T[leg] = hlld_transport(dirL, kL, kR, v_lo, q_lo, v_hi, q_hi);
      } else {
        const double alp = fmax(h.H[along][0][nb], h.H[along][0][P]), alm = fmax(h.H[along][1][nb], h.H[along][1][P]);
        T[leg] = hll_transport(alp, alm, v_lo, q_lo, v_hi, q_hi);
      }
    }
    h.E[c][P] = T[1] - T[0];
  }
}

// ---------------------------------------------------------------------------------------------
// a5 (apply) + a7 (CT, Eq. 6) + a8 (RK2 combine, Eq. 9) + a2 (cons->prim of the result).
// Stage 1: Unew = U0 - dt/dx R.  Stage 2: Unew = U0/2 + (U1 - dt/dx R)/2; same for the face field.
// ---------------------------------------------------------------------------------------------
struct UpdateArgs {
  const double* Uin[5];   // state the stage started from (U0 in stage 1, U1 in stage 2)
  const double* U0[5];    // saved state (stage 2 only)
  const double* R[5];
  double* Uout[5];
  const double* Bin[3];   // ghosts filled
  const double* B0[3];    // ghosts filled (stage 2 only)
  double* Bout[3];
  double* V[11];
  DevScalars* sc;
  const double* Ain[3];   // vector-potential form (Eq. 7-8): edge potential of the stage input, the saved one, the result,
  const double* A0[3];
  double* Aout[3];
  const double* Bref[3];  // and the face field the potential is counted from (ghosts filled)
  int store_u;            // first stage: 0 = U_1 is needed for the primitives only (rk2_keeps_no_u1)
  double dt_fixed;        // > 0: use it; otherwise dt = cfl / smax (first stage; later stages read sc->dt_used)
  double cfl;
  double w, w0;           // Eq. 9: U_s = w U* + w0 U_0 (stages >= 2)
};

// Hydrodynamics: apply the flux divergence, RK2 combine, cons->prim.  (MHD uses k_ct_update below.)
template <bool STAGE2>
__global__ void __launch_bounds__(128, 16) k_update_hd(Geom g, UpdateArgs a) {  // 32 registers: full occupancy for a pure stream
  int i, j, k;
  if (!cell_of_thread(g, i, j, k)) return;
  const long long c = g.at(i, j, k);
  double dt;
  if (STAGE2) {
    dt = a.sc->dt_used;
  } else {
    bool lands;
    dt = first_stage_dt(a.sc, a.dt_fixed, a.cfl, lands);
    if (blockIdx.x == 0 && threadIdx.x == 0) publish_dt(a.sc, dt, lands);
  }
  const double dtdx = dt / g.dx;
  double u[5];
#pragma unroll
  for (int n = 0; n < 5; ++n) {
    // (the pointwise arithmetic of hd_stage.cuh: the stage kernels form the same quantities and must get the same bits)
    if (STAGE2) u[n] = dt == 0.0 ? a.U0[n][c] : hd_combine(a.w0, a.U0[n][c], a.w, a.Uin[n][c], dtdx, a.R[n][c]);
    else u[n] = hd_apply(a.Uin[n][c], dtdx, a.R[n][c]);
    if (STAGE2 || a.store_u) a.Uout[n][c] = u[n];
  }
  double v[5];
  hd_prims(g.gamma - 1.0, u, v);
  double vx = v[1], vy = v[2], vz = v[3], p = v[4];
  if (pressure_floor(g, a.sc, u[0], vx, vy, vz, 0.0, 0.0, 0.0, p, u[4])) a.Uout[4][c] = u[4];
  if (!(u[0] > 0.0) || !(p > 0.0)) a.sc->flag = 1;
  a.V[0][c] = u[0];
  a.V[1][c] = vx;
  a.V[2][c] = vy;
  a.V[3][c] = vz;
  a.V[4][c] = p;
}

// ---------------------------------------------------------------------------------------------
// a6 + a5 (apply) + a7 + a8 + a2 + a1 fused for MHD: one CTA owns a TX x TY x TZ tile of cells.
// Phase 1 evaluates every edge EMF of the tile's edge lattice once (upper lattice planes are recomputed by the
// neighbouring tile: 45 % more edge evaluations with the 32 x 4 x 8 tile, no DRAM cost) into shared memory; phase 2 is k_update with the
// edges read from shared memory, so the edge EMFs never travel to HBM; the result's ghost images (V and the new
// face field) are written by the owners of the boundary cells, which replaces the separate ghost-fill pass.
// ---------------------------------------------------------------------------------------------
constexpr int CT_TX = 32, CT_TY = 4, CT_TZ = 8;
constexpr int CT_ZSPLIT = 2;  // threads per (i, j) column of the tile in the update phase
constexpr int CT_THREADS = CT_TX * CT_TY * CT_ZSPLIT;
constexpr int CT_MINB = 4;    // CTAs per SM
constexpr int CT_LX = CT_TX + 1, CT_LY = CT_TY + 1, CT_LZ = CT_TZ + 1;

// UDONE: the conserved state was already combined by the stage kernel (stages >= 2); only read it back for the primitives.
// VP: vector-potential form (Eq. 7-8): the lattice holds the new potential A = w (A_in - dt E) + w0 A_0 instead of E
// and the face field is B_ref + curl A, so its divergence is one rounding of the face values at any time.
// NCU: the conserved fields this launch reads are not written by it (the host checks the buffers, launch_ct_v), so
// they too can be loaded read-only.
template <int MODE, bool STAGE2, bool UDONE, bool VP, bool NCU>
__global__ void __launch_bounds__(CT_THREADS, CT_MINB) k_ct_update(Geom g, EmfArgs ea, UpdateArgs a) {
  __shared__ double sE[3][CT_LZ][CT_LY][CT_LX];
  const int i0 = blockIdx.x * CT_TX, j0 = blockIdx.y * CT_TY, k0 = blockIdx.z * CT_TZ;
  double dt;
  if (STAGE2) {
    dt = a.sc->dt_used;
  } else {
    bool lands;
    dt = first_stage_dt(a.sc, a.dt_fixed, a.cfl, lands);
    if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && threadIdx.x == 0) publish_dt(a.sc, dt, lands);
  }
  const bool idle = STAGE2 && dt == 0.0;  // a cycle at t_end (idfx_advance_to ran past it): hand U_0 on unchanged
  // ---- phase 1: edge lattice ----
#pragma unroll 1
  for (int p = threadIdx.x; p < CT_LZ * CT_LY * CT_LX; p += CT_THREADS) {
    const int li = p % CT_LX, lj = (p / CT_LX) % CT_LY, lk = p / (CT_LX * CT_LY);
    const int I = i0 + li, J = j0 + lj, K = k0 + lk;
    if (I > g.nx || J > g.ny || K > g.nz) continue;
    // periodic image of lattice index n is index 0; along an open direction the lattice keeps its own plane n
    const int idx[3] = {I == g.nx && !(g.open & 1) ? 0 : I, J == g.ny && !(g.open & 2) ? 0 : J, K == g.nz && !(g.open & 4) ? 0 : K};
    const bool on[3] = {li < CT_TX, lj < CT_TY, lk < CT_TZ};
    const bool owned = on[0] && on[1] && on[2] && I < g.nx && J < g.ny && K < g.nz;
    const long long P = g.at(idx[0], idx[1], idx[2]);
#pragma unroll
    for (int comp = 0; comp < 3; ++comp) {
      if (!on[comp]) continue;
      double e = edge_emf<MODE>(g, ea, idx, comp);
      if (VP) {
        e = a.Ain[comp][P] - dt * e;  // Eq. 7
        if (STAGE2) e = idle ? a.A0[comp][P] : a.w0 * a.A0[comp][P] + a.w * e;
        if (owned) a.Aout[comp][P] = e;
      }
      sE[comp][lk][lj][li] = e;
    }
  }
  __syncthreads();
  // ---- phase 2: one (i, j) column of TZ cells per thread ----
  const int li = threadIdx.x % CT_TX, lj = (threadIdx.x / CT_TX) % CT_TY, lz = threadIdx.x / (CT_TX * CT_TY);
  const int i = i0 + li, j = j0 + lj;
  if (i >= g.nx || j >= g.ny) return;
  const double dtdx = dt / g.dx;
  const long long st[3] = {1, g.sy, g.sz};
  // ghost images of this column in x and y (none with an open side: a fill pass follows then)
  const long long gx = g.open ? 0 : (i < NG ? (long long)g.nx : (i >= g.nx - NG ? -(long long)g.nx : 0));
  const long long gy = g.open ? 0 : (j < NG ? (long long)g.ny * g.sy : (j >= g.ny - NG ? -(long long)g.ny * g.sy : 0));
  const int nd[3] = {g.nx, g.ny, g.nz};
#pragma unroll
  for (int lkk = 0; lkk < CT_TZ / CT_ZSPLIT; ++lkk) {
    const int lk = lz * (CT_TZ / CT_ZSPLIT) + lkk;
    const int k = k0 + lk;
    if (k >= g.nz) break;
    const long long c = g.at(i, j, k);
    double u[5];
#pragma unroll
    for (int n = 0; n < 5; ++n) {
      // the result may be written over the stage input or over U_0 (Euler, RK3): plain loads then
      if (UDONE) {
        u[n] = NCU ? ldro(a.Uout[n] + c) : a.Uout[n][c];
      } else {
        const double uin = NCU ? ldro(a.Uin[n] + c) : a.Uin[n][c];
        const double us = uin - dtdx * ldro(a.R[n] + c);
        if (STAGE2) {
          const double u0 = NCU ? ldro(a.U0[n] + c) : a.U0[n][c];
          u[n] = idle ? u0 : a.w0 * u0 + a.w * us;
        } else {
          u[n] = us;
        }
        if (STAGE2 || a.store_u) a.Uout[n][c] = u[n];
      }
    }
    const double ex00 = sE[0][lk][lj][li], ex10 = sE[0][lk][lj + 1][li];
    const double ex01 = sE[0][lk + 1][lj][li], ex11 = sE[0][lk + 1][lj + 1][li];
    const double ey00 = sE[1][lk][lj][li], ey10 = sE[1][lk][lj][li + 1];
    const double ey01 = sE[1][lk + 1][lj][li], ey11 = sE[1][lk + 1][lj][li + 1];
    const double ez00 = sE[2][lk][lj][li], ez10 = sE[2][lk][lj][li + 1];
    const double ez01 = sE[2][lk][lj + 1][li], ez11 = sE[2][lk][lj + 1][li + 1];
    // O11, left faces then right faces
    const double curlL[3] = {(ez01 - ez00) - (ey01 - ey00), (ex01 - ex00) - (ez10 - ez00), (ey10 - ey00) - (ex10 - ex00)};
    const double curlR[3] = {(ez11 - ez10) - (ey11 - ey10), (ex11 - ex10) - (ez11 - ez01), (ey11 - ey01) - (ex11 - ex01)};
    double v[11];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      double bl, br;
      if (VP) {
        bl = ldro(a.Bref[d] + c) + curlL[d] / g.dx;  // Eq. 8
        br = ldro(a.Bref[d] + c + st[d]) + curlR[d] / g.dx;
      } else {
        bl = ldro(a.Bin[d] + c) - dtdx * curlL[d];  // Eq. 6
        br = ldro(a.Bin[d] + c + st[d]) - dtdx * curlR[d];
        if (STAGE2) {
          const double b0l = ldro(a.B0[d] + c), b0r = ldro(a.B0[d] + c + st[d]);
          bl = idle ? b0l : a.w0 * b0l + a.w * bl;
          br = idle ? b0r : a.w0 * b0r + a.w * br;
        }
      }
      // outflow (G23): the upper boundary face is not part of the state, it copies the last active face
      if (((g.outflow >> (2 * d + 1)) & 1) && (d == 0 ? i : (d == 1 ? j : k)) == nd[d] - 1) br = bl;
      v[5 + d] = 0.5 * (bl + br);
      a.Bout[d][c] = bl;
      // images of the new face value
      const long long gz = g.open ? 0 : (k < NG ? (long long)g.nz * g.sz : (k >= g.nz - NG ? -(long long)g.nz * g.sz : 0));
#pragma unroll
      for (int m = 1; m < 8; ++m) {
        const long long off = ((m & 1) ? gx : 0) + ((m & 2) ? gy : 0) + ((m & 4) ? gz : 0);
        const bool ok = (!(m & 1) || gx != 0) && (!(m & 2) || gy != 0) && (!(m & 4) || gz != 0);
        if (ok) a.Bout[d][c + off] = bl;
      }
    }
    prim_from_cons(g.gamma - 1.0, u[0], u[1], u[2], u[3], u[4], v[5], v[6], v[7], v[1], v[2], v[3], v[4]);
    if (pressure_floor(g, a.sc, u[0], v[1], v[2], v[3], v[5], v[6], v[7], v[4], u[4])) a.Uout[4][c] = u[4];
    v[0] = u[0];
    v[8] = v[3] * v[6] - v[2] * v[7];
    v[9] = v[1] * v[7] - v[3] * v[5];
    v[10] = v[2] * v[5] - v[1] * v[6];
    if (!(u[0] > 0.0) || !(v[4] > 0.0)) a.sc->flag = 1;
    const long long gz = g.open ? 0 : (k < NG ? (long long)g.nz * g.sz : (k >= g.nz - NG ? -(long long)g.nz * g.sz : 0));
    const bool want_ec = a.V[8] != nullptr;  // only the PPM path (edge_emf above) reads the reference EMF back
#pragma unroll
    for (int n = 0; n < 11; ++n)
      if (n < 8 || want_ec) a.V[n][c] = v[n];
    if (gx != 0 || gy != 0 || gz != 0) {
#pragma unroll
      for (int m = 1; m < 8; ++m) {
        const long long off = ((m & 1) ? gx : 0) + ((m & 2) ? gy : 0) + ((m & 4) ? gz : 0);
        const bool ok = (!(m & 1) || gx != 0) && (!(m & 2) || gy != 0) && (!(m & 4) || gz != 0);
        if (ok) {
#pragma unroll
          for (int n = 0; n < 11; ++n)
            if (n < 8 || want_ec) a.V[n][c + off] = v[n];
        }
      }
    }
  }
}

// First launch of every cycle: commits the time reached by the previous one and resets the dt reduction.
__global__ void k_cycle_begin(DevScalars* sc) {
  if (threadIdx.x == 0) {
    sc->t = sc->t_next;
    sc->smax_bits = 0ull;
  }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
thread_local char g_err[512] = "";

void set_err(const char* fmt, const char* a = "", const char* b = "") { snprintf(g_err, sizeof(g_err), fmt, a, b); }

}  // namespace idfx

#include "host.cuh"

using namespace idfx;

#define CK(call)                                                          \
  do {                                                                    \
    cudaError_t e_ = (call);                                              \
    if (e_ != cudaSuccess) {                                              \
      set_err("CUDA error: %s at %s", cudaGetErrorString(e_), #call);     \
      return IDFX_ERR_CUDA;                                               \
    }                                                                     \
  } while (0)

namespace {


typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 4D tensor maps (x, y, z, field) over groups of equally spaced padded fields; one box = one z plane of a tile with its halo.
int make_tensor_maps(idfx_ctx* c) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    set_err("cuTensorMapEncodeTiled is not available from this driver");
    return IDFX_ERR_CUDA;
  }
  EncodeTiledFn enc = (EncodeTiledFn)fn;
  const Geom& g = c->g;
  const cuuint64_t py = g.ny + 2 * NG, pz = g.nz + 2 * NG;
  const cuuint64_t strides[3] = {(cuuint64_t)g.sy * 8, (cuuint64_t)g.sz * 8, (cuuint64_t)g.np * 8};
  const cuuint32_t es[4] = {1, 1, 1, 1};
  if (!c->mhd) {
    const cuuint64_t dimV[4] = {(cuuint64_t)g.sy, py, pz, (cuuint64_t)(2 * c->nv())};
    const cuuint32_t box[4] = {(cuuint32_t)HD_BW, (cuuint32_t)HD_BH, 1u, 5u};
    CUresult r = enc(&c->mapHD, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, c->field(c->f_v()), dimV, strides, box, es,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    const cuuint64_t dimU[4] = {(cuuint64_t)g.sy, py, pz, 5}, dimUU[4] = {(cuuint64_t)g.sy, py, pz, 10};
    CUresult ru = enc(&c->mapHU, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, c->field(F_UA), dimUU, strides, box, es,
                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    CUresult rr = enc(&c->mapHR, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, c->field(c->f_r()), dimU, strides, box, es,
                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS || ru != CUDA_SUCCESS || rr != CUDA_SUCCESS) {
      set_err("cuTensorMapEncodeTiled failed");
      return IDFX_ERR_CUDA;
    }
    return IDFX_OK;
  }
  {
    const cuuint64_t dimV[4] = {(cuuint64_t)g.sy, py, pz, (cuuint64_t)(2 * c->nv())}, dimB[4] = {(cuuint64_t)g.sy, py, pz, 9};
    const cuuint32_t boxV[4] = {(cuuint32_t)MS_BW, (cuuint32_t)MS_BH, 1u, 8u}, boxB[4] = {(cuuint32_t)MS_BWB, (cuuint32_t)MS_TY, 1u, 3u};
    CUresult r1 = enc(&c->mapMV, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, c->field(c->f_v()), dimV, strides, boxV, es,
                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    CUresult r2 = enc(&c->mapMB, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, c->field(F_BA), dimB, strides, boxB, es,
                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r1 != CUDA_SUCCESS || r2 != CUDA_SUCCESS) {
      set_err("cuTensorMapEncodeTiled failed");
      return IDFX_ERR_CUDA;
    }
  }
  return IDFX_OK;
}

void drop_graphs(idfx_ctx* c) {
  for (int k = 0; k < idfx_ctx::N_GRAPHS; ++k) {
    if (c->graph[k]) cudaGraphExecDestroy(c->graph[k]);
    c->graph[k] = nullptr;
  }
}

// Every ABI call runs on the device that holds the workspace, whatever device is current in the calling thread, and
// leaves the caller's current device as it found it.
struct DeviceScope {
  int prev = -1;
  explicit DeviceScope(int dev) {
    if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) cudaSetDevice(dev);
    else prev = -1;
  }
  ~DeviceScope() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

int check_bound(const idfx_ctx* c) {
  if (!c) {
    set_err("null context");
    return IDFX_ERR_INVALID_ARG;
  }
  if (!c->bound) {
    set_err("context has no workspace: call idfx_bind first");
    return IDFX_ERR_NOT_BOUND;
  }
  return IDFX_OK;
}

// ---- standalone dt with PPM (idfx_compute_dt; the other reconstructions run their first-stage kernel for its reduction):
// signal speeds on every face, then the per-cell sum and the max ----
void launch_speed(idfx_ctx* c, int d, const double* const Bf[3]) {
  const int ib = (d + 1) % 3, ie = (d + 2) % 3;
  const long long st[3] = {1, c->g.sy, c->g.sz};
  FluxPpmArgs pa;
  pa.q[0] = c->vfield(0);
  pa.q[1] = c->vfield(1 + d);
  pa.q[2] = c->vfield(1 + ib);
  pa.q[3] = c->vfield(1 + ie);
  pa.q[4] = c->vfield(4);
  pa.q[5] = c->vfield(5 + ib);
  pa.q[6] = c->vfield(5 + ie);
  for (int n = 0; n < 7; ++n) pa.F[n] = nullptr;
  pa.bn = c->mhd ? Bf[d] : nullptr;
  pa.sd = st[d];
  pa.dir = d;
  pa.cf = c->field(c->f_r() + d);  // scratch: R is dead between cycles
  pa.sg = nullptr;
  LaunchScope ls(c, K_FLUX_X + d);
  const unsigned nb = blocks_for(c->g.nc, 128);
  if (c->mhd) k_flux_face_ppm<SOLVER_HLL, true, 1><<<nb, 128, 0, c->stream>>>(c->g, pa);
  else k_flux_face_ppm<SOLVER_HLL, false, 1><<<nb, 128, 0, c->stream>>>(c->g, pa);
}

void launch_dtmax(idfx_ctx* c) {
  RhsArgs a;
  for (int d = 0; d < 3; ++d) {
    for (int n = 0; n < 5; ++n) a.F[d][n] = nullptr;
    a.cf[d] = c->field(c->f_r() + d);
  }
  for (int n = 0; n < 5; ++n) a.R[n] = nullptr;
  a.sc = c->sc;
  LaunchScope ls(c, K_RHS);
  k_rhs<false, true><<<blocks_for(c->g.nc, 128), 128, 0, c->stream>>>(c->g, a);
}

// ---- PPM: face fluxes of the three directions into their own fields, then divergence and dt (k_rhs) ----
template <int SOLVER, bool MHD>
void launch_ppm_s(idfx_ctx* c, const double* const Bf[3], bool want_dt) {
  const Geom& g = c->g;
  const long long st[3] = {1, g.sy, g.sz};
  const unsigned nb = blocks_for(g.nc, 128);
  RhsArgs r;
  for (int d = 0; d < 3; ++d) {
    const int ib = (d + 1) % 3, ie = (d + 2) % 3;
    FluxPpmArgs a;
    a.q[0] = c->vfield(0);
    a.q[1] = c->vfield(1 + d);
    a.q[2] = c->vfield(1 + ib);
    a.q[3] = c->vfield(1 + ie);
    a.q[4] = c->vfield(4);
    a.q[5] = c->vfield(5 + ib);
    a.q[6] = c->vfield(5 + ie);
    a.bn = MHD ? Bf[d] : nullptr;
    a.sd = st[d];
    a.dir = d;
    for (int n = 0; n < 5; ++n) {
      a.F[n] = c->field(c->f_gen() + 5 * d + n);
      r.F[d][n] = a.F[n];
    }
    a.F[5] = c->field(c->f_fb() + 2 * d);
    a.F[6] = c->field(c->f_fb() + 2 * d + 1);
    a.cf = c->field(c->f_gen() + 15 + d);
    r.cf[d] = a.cf;
    a.sg = c->emf == EMF_UCT ? c->sgn(d) : nullptr;
    LaunchScope ls(c, K_FLUX_X + d);
    k_flux_face_ppm<SOLVER, MHD, 0><<<nb, 128, 0, c->stream>>>(g, a);
  }
  for (int n = 0; n < 5; ++n) r.R[n] = c->field(c->f_r() + n);
  r.sc = c->sc;
  LaunchScope ls(c, K_RHS);
  if (want_dt) k_rhs<true, true><<<nb, 128, 0, c->stream>>>(g, r);
  else k_rhs<true, false><<<nb, 128, 0, c->stream>>>(g, r);
}

void launch_ppm(idfx_ctx* c, const double* const Bf[3], bool want_dt) {
  if (c->mhd) {
    if (c->solver == SOLVER_HLL) launch_ppm_s<SOLVER_HLL, true>(c, Bf, want_dt);
    else if (c->solver == SOLVER_RUSANOV) launch_ppm_s<SOLVER_RUSANOV, true>(c, Bf, want_dt);
    else if (c->solver == SOLVER_HLLD) launch_ppm_s<SOLVER_HLLD, true>(c, Bf, want_dt);
    else launch_ppm_s<SOLVER_ROE, true>(c, Bf, want_dt);
  } else {
    if (c->solver == SOLVER_HLL) launch_ppm_s<SOLVER_HLL, false>(c, Bf, want_dt);
    else if (c->solver == SOLVER_RUSANOV) launch_ppm_s<SOLVER_RUSANOV, false>(c, Bf, want_dt);
    else if (c->solver == SOLVER_HLLC) launch_ppm_s<SOLVER_HLLC, false>(c, Bf, want_dt);
    else launch_ppm_s<SOLVER_ROE, false>(c, Bf, want_dt);
  }
}

EmfArgs emf_args(idfx_ctx* c) {
  EmfArgs a;
  for (int d = 0; d < 3; ++d) {
    a.FB[d][0] = c->field(c->f_fb() + 2 * d);
    a.FB[d][1] = c->field(c->f_fb() + 2 * d + 1);
    a.SG[d] = c->sgn(d);
    a.Ec[d] = c->nv() > 8 ? c->vfield(8 + d) : nullptr;
    // edge EMFs already evaluated: by k_emf_hll2d (2D-HLL), or by the one-kernel stage (mhd_stage.cuh)
    a.Eg[d] = c->emf2d() ? c->field(c->f_eg() + d) : (c->fused ? c->field(c->f_fb() + d) : nullptr);
  }
  return a;
}

// 2D-HLL EMF: face quantities of the three directions, then the edge EMFs (two passes over the stage input)
template <int LIM>
void launch_hll2d_l(idfx_ctx* c, const double* const Bf[3]) {
  const bool hlld = c->emf == EMF_UCT_HLLD;
  const int nq = hlld ? 5 : 4;  // face quantities per direction
  const Geom& g = c->g;
  const long long st[3] = {1, g.sy, g.sz};
  const unsigned nb = blocks_for(g.nc, 128);
  Hll2dArgs h;
  for (int d = 0; d < 3; ++d) {
    const int ib = (d + 1) % 3, ie = (d + 2) % 3;
    FluxArgs a;
    a.q[0] = c->vfield(0);
    a.q[1] = c->vfield(1 + d);
    a.q[2] = c->vfield(1 + ib);
    a.q[3] = c->vfield(1 + ie);
    a.q[4] = c->vfield(4);
    a.q[5] = c->vfield(5 + ib);
    a.q[6] = c->vfield(5 + ie);
    a.bn = Bf[d];
    a.sd = st[d];
    for (int n = 0; n < 7; ++n) a.F[n] = nullptr;
    for (int m = 0; m < nq; ++m) {
      a.F[m] = c->field(c->f_h2d() + nq * d + m);
      h.H[d][m] = a.F[m];
    }
    a.cf = nullptr;
    h.Bf[d] = Bf[d];
    h.E[d] = c->field(c->f_eg() + d);
    LaunchScope ls(c, K_EMF);
    if (hlld) k_flux_face<SOLVER_HLL, LIM, true, 3><<<nb, 128, 0, c->stream>>>(g, a);
    else k_flux_face<SOLVER_HLL, LIM, true, 2><<<nb, 128, 0, c->stream>>>(g, a);
  }
  LaunchScope ls(c, K_EMF);
  if (hlld) k_emf_hll2d<LIM, true><<<nb, 128, 0, c->stream>>>(g, h);
  else k_emf_hll2d<LIM, false><<<nb, 128, 0, c->stream>>>(g, h);
}

void launch_hll2d(idfx_ctx* c, const double* const Bf[3]) {
  switch (c->limiter) {
    case LIM_FLAT: launch_hll2d_l<LIM_FLAT>(c, Bf); break;
    case LIM_MINMOD: launch_hll2d_l<LIM_MINMOD>(c, Bf); break;
    case LIM_LIMO3: launch_hll2d_l<LIM_LIMO3>(c, Bf); break;
    default: launch_hll2d_l<LIM_VANLEER>(c, Bf);
  }
}

// a1 of a list of fields; publish: also the dt of the running cycle (k_fill_ghost_dt)
void launch_fill_list(idfx_ctx* c, const FieldList& fl, bool publish) {
  const Geom& g = c->g;
  const long long px = g.nx + 2 * NG, py = g.ny + 2 * NG;
  const long long nt = 2LL * NG * py * px + (long long)g.nz * 2 * NG * px + (long long)g.nz * g.ny * 2 * NG;
  const unsigned nb = blocks_for(nt, 128);
  LaunchScope ls(c, K_FILL);
  if (nt + 128 < (1LL << 31)) {
    if (publish) k_fill_ghost_dt<unsigned int><<<nb, 128, 0, c->stream>>>(g, fl, c->sc, c->cyc_dt_fixed, c->cyc_cfl);
    else k_fill_ghost<unsigned int><<<nb, 128, 0, c->stream>>>(g, fl);
  } else {
    if (publish) k_fill_ghost_dt<long long><<<nb, 128, 0, c->stream>>>(g, fl, c->sc, c->cyc_dt_fixed, c->cyc_cfl);
    else k_fill_ghost<long long><<<nb, 128, 0, c->stream>>>(g, fl);
  }
}

// ghost layers of five consecutive fields
void launch_fill_five(idfx_ctx* c, int first_field, bool publish) {
  FieldList fl;
  fl.n = 5;
  for (int n = 0; n < 5; ++n) fl.f[n] = c->field(first_field + n);
  launch_fill_list(c, fl, publish);
}

void launch_fill(idfx_ctx* c, int which_b) {
  FieldList fl;
  fl.n = 0;
  for (int n = 0; n < c->nv(); ++n) fl.f[fl.n++] = c->vfield(n);
  if (c->mhd)
    for (int d = 0; d < 3; ++d) fl.f[fl.n++] = c->bbuf(which_b, d);
  launch_fill_list(c, fl, false);
}

template <int MODE, bool VP, bool NCU>
void launch_ct_n(idfx_ctx* c, dim3 grid, const EmfArgs& ea, const UpdateArgs& a, bool stage2, bool udone) {
  if (udone) k_ct_update<MODE, true, true, VP, NCU><<<grid, CT_THREADS, 0, c->stream>>>(c->g, ea, a);
  else if (stage2) k_ct_update<MODE, true, false, VP, NCU><<<grid, CT_THREADS, 0, c->stream>>>(c->g, ea, a);
  else k_ct_update<MODE, false, false, VP, NCU><<<grid, CT_THREADS, 0, c->stream>>>(c->g, ea, a);
}

template <int MODE, bool VP>
void launch_ct_v(idfx_ctx* c, dim3 grid, const EmfArgs& ea, const UpdateArgs& a, bool stage2, bool udone) {
  // read-only loads of the conserved fields only when this launch writes none of the buffers it reads them from: the
  // stage input and U_0 differ from the destination, and the pressure floor (which rewrites E in place) is off
  bool ncu;
  if (udone) ncu = !(c->g.pfloor > 0.0);
  else ncu = a.Uin[0] != a.Uout[0] && (!stage2 || a.U0[0] != a.Uout[0]);
  if (ncu) launch_ct_n<MODE, VP, true>(c, grid, ea, a, stage2, udone);
  else launch_ct_n<MODE, VP, false>(c, grid, ea, a, stage2, udone);
}

template <int MODE>
void launch_ct(idfx_ctx* c, dim3 grid, const EmfArgs& ea, const UpdateArgs& a, bool stage2, bool udone) {
  if (c->vp) launch_ct_v<MODE, true>(c, grid, ea, a, stage2, udone);
  else launch_ct_v<MODE, false>(c, grid, ea, a, stage2, udone);
}

// ---- hydrodynamics: the whole stage in one kernel (hd_stage.cuh; instantiated in stage_inst.cu) ----
template <int SOLVER>
HdKernel hd_kernel_s(int limiter, bool first) {
  switch (limiter) {
    case LIM_FLAT: return hd_kernel_sl<SOLVER, LIM_FLAT>(first);
    case LIM_MINMOD: return hd_kernel_sl<SOLVER, LIM_MINMOD>(first);
    case LIM_LIMO3: return hd_kernel_sl<SOLVER, LIM_LIMO3>(first);
    default: return hd_kernel_sl<SOLVER, LIM_VANLEER>(first);
  }
}

HdKernel hd_kernel(const idfx_ctx* c, bool first) {
  switch (c->solver) {
    case SOLVER_HLL: return hd_kernel_s<SOLVER_HLL>(c->limiter, first);
    case SOLVER_RUSANOV: return hd_kernel_s<SOLVER_RUSANOV>(c->limiter, first);
    case SOLVER_HLLC: return hd_kernel_s<SOLVER_HLLC>(c->limiter, first);
    default: return hd_kernel_s<SOLVER_ROE>(c->limiter, first);
  }
}

template <int SOLVER>
HdKernelU hd_kernel_u_s(int limiter, bool first) {
  switch (limiter) {
    case LIM_FLAT: return hd_kernel_u_sl<SOLVER, LIM_FLAT>(first);
    case LIM_MINMOD: return hd_kernel_u_sl<SOLVER, LIM_MINMOD>(first);
    case LIM_LIMO3: return hd_kernel_u_sl<SOLVER, LIM_LIMO3>(first);
    default: return hd_kernel_u_sl<SOLVER, LIM_VANLEER>(first);
  }
}

HdKernelU hd_kernel_u(const idfx_ctx* c, bool first) {
  switch (c->solver) {
    case SOLVER_HLL: return hd_kernel_u_s<SOLVER_HLL>(c->limiter, first);
    case SOLVER_RUSANOV: return hd_kernel_u_s<SOLVER_RUSANOV>(c->limiter, first);
    case SOLVER_HLLC: return hd_kernel_u_s<SOLVER_HLLC>(c->limiter, first);
    default: return hd_kernel_u_s<SOLVER_ROE>(c->limiter, first);
  }
}

// RK2 without a stored U_1 (one-kernel stages, no pressure floor): the first stage's update kernel keeps U_1 in registers
// for the primitives only, and the second stage rebuilds it from U_0 and R_1, which it reads instead of U_1
bool rk2_keeps_no_u1(const idfx_ctx* c) { return c->fused && c->nstages == 2 && !(c->g.pfloor > 0.0); }

void launch_hd_stage(idfx_ctx* c, bool first, double w, double w0, int uin, int uout) {
  const Geom& g = c->g;
  HdStageArgs a;
  a.fV0 = c->vcur ? c->nv() : 0;
  const long long per_chunk = (long long)((g.nx + HD_CX - 1) / HD_CX) * ((g.ny + HD_CY - 1) / HD_CY);
  long long nch = (148 * 2 * 8 + per_chunk - 1) / per_chunk;  // about 8 waves of 2 CTAs per SM
  const long long maxch = g.nz / 16 > 0 ? g.nz / 16 : 1;
  nch = nch < 1 ? 1 : (nch > maxch ? maxch : nch);
  a.chunk = (int)((g.nz + nch - 1) / nch);
  for (int n = 0; n < 5; ++n) {
    a.R[n] = c->field(c->f_r() + n);
    a.Uin[n] = c->field((rk2_keeps_no_u1(c) ? c->f_r() : uin) + n);
    a.U0[n] = c->field(c->f_u() + n);
    a.Uout[n] = c->field(uout + n);
    a.Vout[n] = c->vfield_out(n);
  }
  a.uin_is_r = rk2_keeps_no_u1(c) ? 1 : 0;
  a.sc = c->sc;
  a.w = w;
  a.w0 = w0;
  dim3 grid((g.nx + HD_CX - 1) / HD_CX, (g.ny + HD_CY - 1) / HD_CY, (unsigned)((g.nz + a.chunk - 1) / a.chunk));
  LaunchScope ls(c, K_HD);
  hd_kernel(c, first)<<<grid, HD_THREADS, HD_SMEM_BYTES, c->stream>>>(g, a, c->mapHD);
}

// Hydrodynamic RK2 on a periodic box without pressure floor and without neighbours: the stages read the conserved fields
// (hd_stage_u.cuh).  The first cycle after set_state still reconstructs from the caller's primitives as given.
bool hd_ufed(const idfx_ctx* c) {
  return c->fused && !c->mhd && c->nstages == 2 && !(c->g.pfloor > 0.0) && !c->g.open && !c->exch && !c->v_given;
}

void launch_hd_stage_u(idfx_ctx* c, bool first, double w, double w0) {
  const Geom& g = c->g;
  HdStageArgs a;
  a.fV0 = c->ucur ? 5 : 0;  // U_0 inside the map over both conserved buffers
  const long long per_chunk = (long long)((g.nx + HD_CX - 1) / HD_CX) * ((g.ny + HD_CY - 1) / HD_CY);
  long long nch = (148 * 2 * 8 + per_chunk - 1) / per_chunk;  // about 8 waves of 2 CTAs per SM
  const long long maxch = g.nz / 16 > 0 ? g.nz / 16 : 1;
  nch = nch < 1 ? 1 : (nch > maxch ? maxch : nch);
  a.chunk = (int)((g.nz + nch - 1) / nch);
  for (int n = 0; n < 5; ++n) {
    a.R[n] = c->field(c->f_r() + n);
    a.Uin[n] = c->field(c->f_r() + n);
    a.U0[n] = c->field(c->f_u() + n);
    a.Uout[n] = c->field(c->f_ub() + n);
    a.Vout[n] = nullptr;
  }
  a.uin_is_r = 1;
  a.sc = c->sc;
  a.w = w;
  a.w0 = w0;
  dim3 grid((g.nx + HD_CX - 1) / HD_CX, (g.ny + HD_CY - 1) / HD_CY, (unsigned)((g.nz + a.chunk - 1) / a.chunk));
  LaunchScope ls(c, K_HD);
  hd_kernel_u(c, first)<<<grid, HD_THREADS, HDU_SMEM_BYTES, c->stream>>>(g, a, c->mapHU, c->mapHR);
}

// ---- MHD: the three sweeps and the edge EMFs of a stage in one kernel (mhd_stage.cuh; instantiated in stage_inst.cu) ----
template <int SOLVER>
MhdKernel mhd_kernel_s(int limiter, bool first, int mode, bool open) {
  switch (limiter) {
    case LIM_FLAT: return mhd_kernel_sl<SOLVER, LIM_FLAT>(first, mode, open);
    case LIM_MINMOD: return mhd_kernel_sl<SOLVER, LIM_MINMOD>(first, mode, open);
    case LIM_LIMO3: return mhd_kernel_sl<SOLVER, LIM_LIMO3>(first, mode, open);
    default: return mhd_kernel_sl<SOLVER, LIM_VANLEER>(first, mode, open);
  }
}

// mode: the edge EMF the kernel evaluates (arithmetic, E^c, E^0); the 2D-HLL EMF comes from its own kernels afterwards
MhdKernel mhd_kernel(const idfx_ctx* c, bool first, int mode, bool open) {
  switch (c->solver) {
    case SOLVER_HLL: return mhd_kernel_s<SOLVER_HLL>(c->limiter, first, mode, open);
    case SOLVER_RUSANOV: return mhd_kernel_s<SOLVER_RUSANOV>(c->limiter, first, mode, open);
    case SOLVER_HLLD: return mhd_kernel_s<SOLVER_HLLD>(c->limiter, first, mode, open);
    default: return mhd_kernel_s<SOLVER_ROE>(c->limiter, first, mode, open);
  }
}

void launch_mhd_stage(idfx_ctx* c, bool first, double w, double w0, int uin, int uout, int bin) {
  const Geom& g = c->g;
  MhdStageArgs a;
  a.fV0 = c->vcur ? c->nv() : 0;
  a.fB0 = 3 * bin;
  // along an open direction the tiles start at cell -1 (mhd_stage.cuh)
  const int tx = (g.nx + (g.open & 1) + MS_CX - 1) / MS_CX, ty = (g.ny + ((g.open >> 1) & 1) + MS_CY - 1) / MS_CY;
  // z planes per CTA: one CTA per SM runs at a time, so the launch takes ceil(CTAs / SMs) rounds of (chunk + 1) plane
  // iterations (every chunk re-solves the plane below it for its lowest edges); take the chunk count with the shortest
  // launch among those with at least two rounds (measured: finer granularity balances better than the model says: 128^3
  // with 120 CTAs in one round 1.01 ms, 420 CTAs in three rounds 0.94 ms); a box too small for two rounds is cut into
  // chunks as short as four planes so that its CTAs spread over the SMs (32^3: 0.22 -> 0.09 ms per cycle).
  const long long per_chunk = (long long)tx * ty;
  const long long maxch = g.nz / 4 > 0 ? g.nz / 4 : 1;
  long long nch = 1, best = -1;
  for (int pass = 0; pass < 2 && best < 0; ++pass)
    for (long long k = 1; k <= maxch; ++k) {
      const long long chunk = (g.nz + k - 1) / k, ctas = per_chunk * ((g.nz + chunk - 1) / chunk);
      const long long rounds = (ctas + c->sms - 1) / c->sms, cost = rounds * (chunk + 1);
      if ((rounds >= 2 || pass == 1) && (best < 0 || cost < best)) {
        best = cost;
        nch = k;
      }
    }
  a.chunk = (int)((g.nz + nch - 1) / nch);
  for (int n = 0; n < 5; ++n) {
    a.R[n] = c->field(c->f_r() + n);
    a.Uin[n] = c->field((rk2_keeps_no_u1(c) ? c->f_r() : uin) + n);
    a.U0[n] = c->field(c->f_u() + n);
    a.Uout[n] = c->field(uout + n);
  }
  a.uin_is_r = rk2_keeps_no_u1(c) ? 1 : 0;
  for (int d = 0; d < 3; ++d) a.E[d] = c->field(c->f_fb() + d);  // the edge lattice lives in the first three face-flux slots
  a.sc = c->sc;
  a.w = w;
  a.w0 = w0;
  dim3 grid(tx, ty, (unsigned)((g.nz + a.chunk - 1) / a.chunk));
  LaunchScope ls(c, K_MHD);
  mhd_kernel(c, first, c->emf2d() ? EMF_ARITH : c->emf, g.open != 0)<<<grid, MS_THREADS, MS_SMEM_BYTES, c->stream>>>(g, a, c->mapMV,
                                                                                                                 c->mapMB);
}

// ---- one cycle, in pieces: cycle_begin, then per stage stage_flux -> stage_update (-> ghost fill), then cycle_end.
// idfx_step / idfx_advance run them back to back (run_cycle); a domain-decomposed run drives them through the staged ABI
// with its halo exchange and the reduction of dt in between.
// Conserved fields: U_0 lives in one of the two conserved buffers (idfx_ctx::f_u) for the whole cycle, the intermediate
// stages in the other (f_ub), the last stage writes the result back over U_0 -- except in the hydrodynamic cycle fed with
// the conserved fields (hd_stage_u.cuh), whose second stage still reads the halo of U_0 in neighbouring tiles while it
// writes: its result goes to the other buffer and the two swap roles.  Face field: three buffers rotate, never writing the saved one (b0) nor the stage input.
struct StagePlan {
  bool combine, last;
  int uin, uout, bin, b0, bout;
  double w, w0;
};

StagePlan plan_stage(const idfx_ctx* c, int s) {
  static const double W[3][3] = {{1.0, 0.0, 0.0}, {1.0, 0.5, 0.0}, {1.0, 0.25, 2.0 / 3.0}};      // Tab. 1
  static const double W0[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.5, 0.0}, {0.0, 0.75, 1.0 / 3.0}};
  StagePlan p;
  p.combine = s > 0;
  p.last = s == c->nstages - 1;
  p.uin = s == 0 ? c->f_u() : c->f_ub();
  p.uout = p.last ? c->f_u() : c->f_ub();
  p.w = W[c->nstages - 1][s];
  p.w0 = W0[c->nstages - 1][s];
  p.b0 = c->cyc_b0;
  p.bin = c->cyc_bin;
  const int b1 = (p.b0 + 1) % 3, b2 = (p.b0 + 2) % 3;
  p.bout = p.bin == b1 ? b2 : b1;
  return p;
}

// dt_fixed > 0: that dt; otherwise dt = cfl / max found by stage 1, shortened to land on t_end (never leaves the device)
// NVTX range per cycle piece: "idfx cycle" > "stage s flux" / "stage s update"; under CUDA-graph replay
// only the capture shows them, run with IDFX_GRAPH=0 for a per-stage timeline
struct NvtxScope {
  explicit NvtxScope(const char* name) { nvtxRangePushA(name); }
  ~NvtxScope() { nvtxRangePop(); }
};

int ensure_v(idfx_ctx* c);

// Before every cycle, outside any graph capture: decides which kind of cycle runs and brings the fields it reads up to date.
int prepare_cycle(idfx_ctx* c) {
  c->cyc_ufed = hd_ufed(c);
  if (c->cyc_ufed) {
    if (!c->ug_valid) {  // the cycle before wrote U without its ghost layers
      launch_fill_five(c, c->f_u(), false);
      c->ug_valid = true;
    }
    return IDFX_OK;
  }
  return ensure_v(c);
}

// the flags a finished cycle leaves (cycle_end, or the replay of its graph)
void after_cycle(idfx_ctx* c) {
  if (c->cyc_ufed) c->ucur ^= 1;
  c->v_stale = c->cyc_ufed;
  c->ug_valid = c->cyc_ufed;
  c->v_given = false;
}

void cycle_begin(idfx_ctx* c, double dt_fixed, double cfl) {
  NvtxScope range("idfx cycle_begin");
  c->cyc_dt_fixed = dt_fixed;
  c->cyc_cfl = cfl;
  c->cyc_b0 = c->cyc_bin = c->bcur;
  LaunchScope ls(c, K_STATE);
  k_cycle_begin<<<1, 32, 0, c->stream>>>(c->sc);
}

// a3 - a6 of stage s: reconstruct -> Riemann -> flux divergence (-> edge EMFs); stage 0 also reduces max sum_d c_d / dx
void stage_flux(idfx_ctx* c, int s) {
  static const char* const names[3] = {"idfx stage 1 flux+emf", "idfx stage 2 flux+emf", "idfx stage 3 flux+emf"};
  NvtxScope range(names[s]);
  const StagePlan p = plan_stage(c, s);
  if (c->cyc_ufed) {
    launch_hd_stage_u(c, !p.combine, p.w, p.w0);
    return;
  }
  const double* Bf[3] = {c->bbuf(p.bin, 0), c->bbuf(p.bin, 1), c->bbuf(p.bin, 2)};
  if (!c->fused) launch_ppm(c, Bf, s == 0 && !(c->cyc_dt_fixed > 0.0));  // PPM: generic face-flux kernels, divergence and dt in k_rhs
  else if (c->mhd) launch_mhd_stage(c, !p.combine, p.w, p.w0, p.uin, p.uout, p.bin);
  else launch_hd_stage(c, !p.combine, p.w, p.w0, p.uin, p.uout);
}

// a7, a8, a2 of stage s (and the ghost images or the local ghost fill a1 of its result); rotates the buffers
void stage_update(idfx_ctx* c, int s) {
  static const char* const names[3] = {"idfx stage 1 ct+update", "idfx stage 2 ct+update", "idfx stage 3 ct+update"};
  NvtxScope range(names[s]);
  const StagePlan p = plan_stage(c, s);
  const Geom& g = c->g;
  c->cyc_bin = p.bout;
  if (c->cyc_ufed) {
    // a1 of what the stage wrote: R_1 (and the dt of the cycle, now that the whole box has been reduced), or the result
    if (!p.combine) launch_fill_five(c, c->f_r(), true);
    else launch_fill_five(c, c->f_ub(), false);
    return;
  }
  if (c->fused && !c->mhd && p.combine) {
    // the HD stage kernel wrote U_s, its primitives and (periodic box) their ghost images into the other primitive buffer
    c->vcur ^= 1;
    if (g.open && !c->exch) launch_fill(c, p.bout);
    return;
  }
  UpdateArgs a;
  for (int n = 0; n < 5; ++n) {
    a.Uin[n] = c->field(p.uin + n);
    a.U0[n] = c->field(c->f_u() + n);
    a.R[n] = c->field(c->f_r() + n);
    a.Uout[n] = c->field(p.uout + n);
  }
  for (int d = 0; d < 3; ++d) {
    a.Bin[d] = c->bbuf(p.bin, d);
    a.B0[d] = c->bbuf(p.b0, d);
    a.Bout[d] = c->bbuf(p.bout, d);
    a.Ain[d] = c->vp ? c->abuf(p.bin, d) : nullptr;
    a.A0[d] = c->vp ? c->abuf(p.b0, d) : nullptr;
    a.Aout[d] = c->vp ? c->abuf(p.bout, d) : nullptr;
    a.Bref[d] = c->vp ? c->field(c->f_bref() + d) : nullptr;
  }
  a.sc = c->sc;
  a.dt_fixed = c->cyc_dt_fixed;
  a.cfl = c->cyc_cfl;
  a.w = p.w;
  a.w0 = p.w0;
  a.store_u = !(s == 0 && rk2_keeps_no_u1(c));
  if (c->mhd) {
    // CT + RK combine + cons->prim + ghost images in one kernel; V is double-buffered because neighbouring tiles still
    // read the stage-input primitives while this tile writes the result's
    const EmfArgs ea = emf_args(c);
    // -(v x Bc) is stored for PPM only: the one-kernel stage forms it itself
    for (int n = 0; n < 11; ++n) a.V[n] = n < c->nv() ? c->vfield_out(n) : nullptr;
    dim3 grid((g.nx + CT_TX - 1) / CT_TX, (g.ny + CT_TY - 1) / CT_TY, (g.nz + CT_TZ - 1) / CT_TZ);
    const bool udone = p.combine && c->fused;  // the one-kernel stage applied the divergence itself
    if (c->emf2d()) {
      const double* Bf[3] = {c->bbuf(p.bin, 0), c->bbuf(p.bin, 1), c->bbuf(p.bin, 2)};
      launch_hll2d(c, Bf);
    }
    {
      LaunchScope ls(c, K_UPDATE);
      if (c->fused || c->emf2d()) launch_ct<EMF_UCT_HLL>(c, grid, ea, a, p.combine, udone);  // lattice read from memory
      else if (c->emf == EMF_UCT) launch_ct<EMF_UCT>(c, grid, ea, a, p.combine, udone);
      else if (c->emf == EMF_UCT0) launch_ct<EMF_UCT0>(c, grid, ea, a, p.combine, udone);
      else launch_ct<EMF_ARITH>(c, grid, ea, a, p.combine, udone);
    }
    c->vcur ^= 1;
    if (g.open && !c->exch) launch_fill(c, p.bout);  // no images were written
  } else {
    for (int n = 0; n < 11; ++n) a.V[n] = n < c->nv() ? c->vfield(n) : nullptr;
    {
      LaunchScope ls(c, K_UPDATE);
      if (p.combine) k_update_hd<true><<<blocks_for(g.nc, 128), 128, 0, c->stream>>>(g, a);
      else k_update_hd<false><<<blocks_for(g.nc, 128), 128, 0, c->stream>>>(g, a);
    }
    if (!c->exch) launch_fill(c, p.bout);
  }
}

void cycle_end(idfx_ctx* c) {
  c->bcur = c->cyc_bin;
  after_cycle(c);
}

int run_cycle(idfx_ctx* c, double dt_fixed, double cfl) {
  cycle_begin(c, dt_fixed, cfl);
  for (int s = 0; s < c->nstages; ++s) {
    stage_flux(c, s);
    stage_update(c, s);
  }
  cycle_end(c);
  CK(cudaGetLastError());
  return IDFX_OK;
}

int copy3d(idfx_ctx* c, double* field, const double* contig_in, double* contig_out, cudaMemcpyKind kind) {
  const Geom& g = c->g;
  cudaMemcpy3DParms p;
  memset(&p, 0, sizeof(p));
  cudaPitchedPtr pad = make_cudaPitchedPtr((void*)(field + g.at(0, 0, 0)), (size_t)g.sy * 8, g.nx, g.ny + 2 * NG);
  p.extent = make_cudaExtent((size_t)g.nx * 8, g.ny, g.nz);
  p.kind = kind;
  if (contig_in) {
    p.srcPtr = make_cudaPitchedPtr((void*)contig_in, (size_t)g.nx * 8, g.nx, g.ny);
    p.dstPtr = pad;
  } else {
    p.srcPtr = pad;
    p.dstPtr = make_cudaPitchedPtr((void*)contig_out, (size_t)g.nx * 8, g.nx, g.ny);
  }
  CK(cudaMemcpy3DAsync(&p, c->stream));
  return IDFX_OK;
}

// t = 0, no target time, no cycles counted; the sticky error flag and the dt scalars are left alone
int reset_clock(idfx_ctx* c) {
  DevScalars h;
  memset(&h, 0, sizeof(h));
  h.t_end = INFINITY;
  const size_t off = offsetof(DevScalars, t);
  // pageable source: staged before the call returns
  CK(cudaMemcpyAsync((char*)c->sc + off, (const char*)&h + off, sizeof(h) - off, cudaMemcpyHostToDevice, c->stream));
  return IDFX_OK;
}

// after the primitives (V[0..4]) and the face field (current buffer, active part) are in place
int finish_set_state(idfx_ctx* c) {
  StateArgs a;
  for (int n = 0; n < 5; ++n) a.U[n] = c->field(c->f_u() + n);
  for (int n = 0; n < 11; ++n) a.V[n] = n < c->nv() ? c->vfield(n) : nullptr;
  for (int d = 0; d < 3; ++d) a.Bf[d] = c->bbuf(c->bcur, d);
  a.sc = c->sc;
  const unsigned nb = blocks_for(c->g.nc, 128);
  // open sides: Bc of the last cell needs the ghost face beyond it (its caller has filled the face ghosts when they come
  // from a neighbour; zero-gradient ones are filled here)
  if (c->mhd && c->g.open && !c->exch) launch_fill(c, c->bcur);
  { LaunchScope ls(c, K_STATE);
  if (c->mhd) k_cons_from_prim<true><<<nb, 128, 0, c->stream>>>(c->g, a);
  else k_cons_from_prim<false><<<nb, 128, 0, c->stream>>>(c->g, a);
  }
  c->cyc_bin = c->bcur;
  if (!c->exch) launch_fill(c, c->bcur);
  c->v_given = true;  // the next cycle reconstructs from exactly these primitives
  c->v_stale = false;
  c->ug_valid = false;
  CK(cudaGetLastError());
  if (c->vp) {  // G19: the potential is counted from this state on
    const size_t fb = (size_t)c->g.np * sizeof(double);
    CK(cudaMemsetAsync(c->field(c->f_aa()), 0, 9 * fb, c->stream));
    CK(cudaMemcpyAsync(c->field(c->f_bref()), c->bbuf(c->bcur, 0), 3 * fb, cudaMemcpyDeviceToDevice, c->stream));
  }
  return reset_clock(c);
}

int refresh_prims(idfx_ctx* c) {
  StateArgs a;
  for (int n = 0; n < 5; ++n) a.U[n] = c->field(c->f_u() + n);
  for (int n = 0; n < 11; ++n) a.V[n] = nullptr;
  for (int n = 0; n < 5; ++n) a.V[n] = c->field(c->f_r() + n);  // scratch: R is dead between cycles
  for (int d = 0; d < 3; ++d) a.Bf[d] = c->bbuf(c->bcur, d);
  a.sc = c->sc;
  const unsigned nb = blocks_for(c->g.nc, 128);
  { LaunchScope ls(c, K_STATE);
  if (c->mhd) k_prim_from_cons<true><<<nb, 128, 0, c->stream>>>(c->g, a);
  else k_prim_from_cons<false><<<nb, 128, 0, c->stream>>>(c->g, a);
  }
  CK(cudaGetLastError());
  return IDFX_OK;
}

// Hydrodynamic cycles fed with the conserved fields leave the primitive buffer behind: bring it (and its ghost layers) up to
// date before anything reads it (a cycle of the other kind after an option changed)
int ensure_v(idfx_ctx* c) {
  if (!c->v_stale) return IDFX_OK;
  StateArgs a;
  for (int n = 0; n < 5; ++n) a.U[n] = c->field(c->f_u() + n);
  for (int n = 0; n < 11; ++n) a.V[n] = n < 5 ? c->vfield(n) : nullptr;
  for (int d = 0; d < 3; ++d) a.Bf[d] = nullptr;
  a.sc = c->sc;
  {
    LaunchScope ls(c, K_STATE);
    k_prim_from_cons<false><<<blocks_for(c->g.nc, 128), 128, 0, c->stream>>>(c->g, a);
  }
  launch_fill(c, c->bcur);
  c->v_stale = false;
  CK(cudaGetLastError());
  return IDFX_OK;
}

}  // namespace

// =============================================================================================
// C ABI
// =============================================================================================
extern "C" {

const char* idfx_last_error(void) { return g_err; }

idfx_ctx* idfx_create(int nx, int ny, int nz, double dx, double gamma, int solver, int limiter, int emf_mode) {
  if (nx < 4 || ny < 4 || nz < 4) {
    set_err("idfx_create: nx, ny, nz must be >= 4");
    return nullptr;
  }
  if (!(dx > 0.0) || !(gamma > 1.0)) {
    set_err("idfx_create: need dx > 0 and gamma > 1");
    return nullptr;
  }
  if (solver < 0 || solver > 4 || limiter < 0 || limiter > 4 || emf_mode < 0 || emf_mode > 5) {
    set_err("idfx_create: unknown solver, limiter or emf_mode");
    return nullptr;
  }
  if (limiter == LIM_PPM && (emf_mode == EMF_UCT_HLL || emf_mode == EMF_UCT_HLLD)) {
    set_err("idfx_create: unsupported combination (the 2D-HLL / HLLD EMFs reconstruct with three-cell stencils, not PPM)");
    return nullptr;
  }
  if (emf_mode == EMF_UCT_HLLD && solver != SOLVER_HLLD) {
    set_err("idfx_create: unsupported combination (the 2D-HLLD EMF takes its coefficients from HLLD face solves)");
    return nullptr;
  }
  const bool mhd = emf_mode != EMF_NONE;
  if ((mhd && solver == SOLVER_HLLC) || (!mhd && solver == SOLVER_HLLD)) {
    set_err("idfx_create: unsupported combination (HLLC is HD-only, HLLD is MHD-only)");
    return nullptr;
  }
  idfx_ctx* c = new (std::nothrow) idfx_ctx;
  if (!c) return nullptr;
  Geom& g = c->g;
  g.nx = nx;
  g.ny = ny;
  g.nz = nz;
  g.dx = dx;
  g.gamma = gamma;
  g.pfloor = 0.0;
  g.outflow = 0;
  g.open = 0;
  g.sy = ((nx + IOFF + NG + 15) / 16) * 16;
  g.sz = (long long)g.sy * (ny + 2 * NG);
  g.np = ((g.sz * (nz + 2 * NG) + 31) / 32) * 32;
  g.nc = (long long)nx * ny * nz;
  c->solver = solver;
  c->limiter = limiter;
  c->emf = emf_mode;
  c->mhd = mhd;
  return c;
}

size_t idfx_workspace_bytes(const idfx_ctx* c) {
  if (!c) return 0;
  return (size_t)c->nfields() * (size_t)c->g.np * sizeof(double) + 256;
}

int idfx_bind(idfx_ctx* c, void* d_workspace, size_t bytes, void* cuda_stream) {
  if (!c || !d_workspace) {
    set_err("idfx_bind: null argument");
    return IDFX_ERR_INVALID_ARG;
  }
  if (bytes < idfx_workspace_bytes(c) || ((size_t)d_workspace & 255) != 0) {
    set_err("idfx_bind: workspace too small or not 256-byte aligned");
    return IDFX_ERR_INVALID_ARG;
  }
  cudaPointerAttributes attr;
  if (cudaPointerGetAttributes(&attr, d_workspace) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
    cudaGetLastError();
    set_err("idfx_bind: the workspace is not device memory");
    return IDFX_ERR_INVALID_ARG;
  }
  c->device = attr.device;
  DeviceScope on_device(c->device);
  if (cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess || c->sms < 1) c->sms = 148;
  c->ws = (double*)d_workspace;
  c->ws_bytes = bytes;
  c->stream = (cudaStream_t)cuda_stream;
  c->sc = (DevScalars*)(c->ws + (size_t)c->nfields() * (size_t)c->g.np);
  c->bcur = 0;
  c->vcur = 0;
  c->ucur = 0;
  c->v_given = true;
  c->v_stale = c->ug_valid = c->cyc_ufed = false;
  c->launches = 0;
  CK(cudaMemsetAsync(d_workspace, 0, idfx_workspace_bytes(c), c->stream));
  if (int rc = reset_clock(c)) return rc;
  drop_graphs(c);
  const char* genv = getenv("IDFX_GRAPH");
  // the legacy default stream cannot be captured: graphs only on a stream of the caller's own
  c->use_graph = !(genv && genv[0] == '0') && c->stream != nullptr && c->stream != cudaStreamLegacy &&
                 c->stream != cudaStreamPerThread;
  const char* benv = getenv("IDFX_ADVANCE_BATCH");
  c->fixed_batch = benv ? atoi(benv) : 0;
  c->fused = c->limiter != LIM_PPM;  // PPM (five-cell stencils) runs through k_flux_face_ppm / k_rhs
  if (c->fused) {
    int rc = make_tensor_maps(c);
    if (rc) return rc;
  }
  if (c->fused && !c->mhd)
    for (int first = 0; first < 2; ++first)
    {
      CK(cudaFuncSetAttribute((const void*)hd_kernel(c, first != 0), cudaFuncAttributeMaxDynamicSharedMemorySize, HD_SMEM_BYTES));
      CK(cudaFuncSetAttribute((const void*)hd_kernel_u(c, first != 0), cudaFuncAttributeMaxDynamicSharedMemorySize, HDU_SMEM_BYTES));
    }
  if (c->fused && c->mhd)
    for (int v = 0; v < 4; ++v)  // first / later stage x periodic / open (the boundary option may still change after bind)
      CK(cudaFuncSetAttribute((const void*)mhd_kernel(c, (v & 1) != 0, c->emf2d() ? EMF_ARITH : c->emf, (v & 2) != 0),
                              cudaFuncAttributeMaxDynamicSharedMemorySize, MS_SMEM_BYTES));
  c->bound = true;
  return IDFX_OK;
}

int idfx_set_state(idfx_ctx* c, const double* d_prim, const double* d_bface) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!d_prim || (c->mhd && !d_bface)) {
    set_err("idfx_set_state: null state pointer");
    return IDFX_ERR_INVALID_ARG;
  }
  const unsigned nb = blocks_for(c->g.nc, 128);
  FieldList fl;
  fl.n = 5;
  for (int n = 0; n < 5; ++n) fl.f[n] = c->vfield(n);
  { LaunchScope ls(c, K_STATE);
  k_pack<<<nb, 128, 0, c->stream>>>(c->g, fl, d_prim);
  }
  if (c->mhd) {
    fl.n = 3;
    for (int d = 0; d < 3; ++d) fl.f[d] = c->bbuf(c->bcur, d);
    { LaunchScope ls(c, K_STATE);
    k_pack<<<nb, 128, 0, c->stream>>>(c->g, fl, d_bface);
    }
  }
  c->cyc_bin = c->bcur;
  if (c->exch) return IDFX_OK;  // the caller exchanges the face ghosts, then calls idfx_set_state_finish
  return finish_set_state(c);
}

int idfx_set_state_finish(idfx_ctx* c) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!c->exch) {
    set_err("idfx_set_state_finish: only with exchanged directions (idfx_set_state is complete otherwise)");
    return IDFX_ERR_INVALID_ARG;
  }
  return finish_set_state(c);
}

int idfx_set_state_host(idfx_ctx* c, const double* h_prim, const double* h_bface) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!h_prim || (c->mhd && !h_bface)) {
    set_err("idfx_set_state_host: null state pointer");
    return IDFX_ERR_INVALID_ARG;
  }
  for (int n = 0; n < 5; ++n)
    if ((rc = copy3d(c, c->vfield(n), h_prim + (size_t)n * c->g.nc, nullptr, cudaMemcpyHostToDevice))) return rc;
  if (c->mhd)
    for (int d = 0; d < 3; ++d)
      if ((rc = copy3d(c, c->bbuf(c->bcur, d), h_bface + (size_t)d * c->g.nc, nullptr, cudaMemcpyHostToDevice)))
        return rc;
  c->cyc_bin = c->bcur;
  if (!c->exch && (rc = finish_set_state(c))) return rc;
  CK(cudaStreamSynchronize(c->stream));  // the caller may reuse its host buffers as soon as this returns
  return IDFX_OK;
}

int idfx_get_state(idfx_ctx* c, double* d_prim, double* d_bface) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!d_prim) {
    set_err("idfx_get_state: null output");
    return IDFX_ERR_INVALID_ARG;
  }
  if ((rc = refresh_prims(c))) return rc;
  const unsigned nb = blocks_for(c->g.nc, 128);
  FieldList fl;
  fl.n = 5;
  for (int n = 0; n < 5; ++n) fl.f[n] = c->field(c->f_r() + n);
  { LaunchScope ls(c, K_STATE);
  k_unpack<<<nb, 128, 0, c->stream>>>(c->g, fl, d_prim);
  }
  if (c->mhd && d_bface) {
    fl.n = 3;
    for (int d = 0; d < 3; ++d) fl.f[d] = c->bbuf(c->bcur, d);
    { LaunchScope ls(c, K_STATE);
    k_unpack<<<nb, 128, 0, c->stream>>>(c->g, fl, d_bface);
    }
  }
  CK(cudaGetLastError());
  return IDFX_OK;
}

int idfx_get_state_host(idfx_ctx* c, double* h_prim, double* h_bface) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!h_prim) {
    set_err("idfx_get_state_host: null output");
    return IDFX_ERR_INVALID_ARG;
  }
  if ((rc = refresh_prims(c))) return rc;
  for (int n = 0; n < 5; ++n)
    if ((rc = copy3d(c, c->field(c->f_r() + n), nullptr, h_prim + (size_t)n * c->g.nc, cudaMemcpyDeviceToHost))) return rc;
  if (c->mhd && h_bface)
    for (int d = 0; d < 3; ++d)
      if ((rc = copy3d(c, c->bbuf(c->bcur, d), nullptr, h_bface + (size_t)d * c->g.nc, cudaMemcpyDeviceToHost)))
        return rc;
  CK(cudaStreamSynchronize(c->stream));
  return IDFX_OK;
}

int idfx_get_conserved(idfx_ctx* c, double* d_cons, double* d_bface) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!d_cons) {
    set_err("idfx_get_conserved: null output");
    return IDFX_ERR_INVALID_ARG;
  }
  const unsigned nb = blocks_for(c->g.nc, 128);
  FieldList fl;
  fl.n = 5;
  for (int n = 0; n < 5; ++n) fl.f[n] = c->field(c->f_u() + n);
  { LaunchScope ls(c, K_STATE);
  k_unpack<<<nb, 128, 0, c->stream>>>(c->g, fl, d_cons);
  }
  if (c->mhd && d_bface) {
    fl.n = 3;
    for (int d = 0; d < 3; ++d) fl.f[d] = c->bbuf(c->bcur, d);
    { LaunchScope ls(c, K_STATE);
    k_unpack<<<nb, 128, 0, c->stream>>>(c->g, fl, d_bface);
    }
  }
  CK(cudaGetLastError());
  return IDFX_OK;
}

int idfx_compute_dt(idfx_ctx* c, double cfl, double* h_dt_out) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!h_dt_out || !(cfl > 0.0) || !(cfl < 1.0)) {
    set_err("idfx_compute_dt: need 0 < cfl < 1 and a non-null output");
    return IDFX_ERR_INVALID_ARG;
  }
  CK(cudaMemsetAsync(&c->sc->smax_bits, 0, sizeof(unsigned long long), c->stream));
  if (c->fused) {
    // the first-stage kernel itself, run for its reduction only (its divergence and EMFs land in scratch that is dead
    // between cycles): the same arithmetic, tile for tile, as the dt a cycle would take, on any kind of boundary
    if (c->mhd) launch_mhd_stage(c, true, 1.0, 0.0, c->f_u(), c->f_ub(), c->bcur);
    else if (c->v_stale) launch_hd_stage_u(c, true, 1.0, 0.0);  // the conserved fields (with ghosts) are what is current
    else launch_hd_stage(c, true, 1.0, 0.0, c->f_u(), c->f_ub());
  } else {
    const double* Bf[3] = {c->bbuf(c->bcur, 0), c->bbuf(c->bcur, 1), c->bbuf(c->bcur, 2)};
    for (int d = 0; d < 3; ++d) launch_speed(c, d, Bf);
    launch_dtmax(c);
  }
  CK(cudaGetLastError());
  unsigned long long bits = 0;
  CK(cudaMemcpyAsync(&bits, &c->sc->smax_bits, sizeof(bits), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  double smax;
  memcpy(&smax, &bits, sizeof(smax));
  *h_dt_out = cfl / smax;
  return IDFX_OK;
}

int idfx_step(idfx_ctx* c, double dt) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!(dt > 0.0)) {
    set_err("idfx_step: dt must be > 0");
    return IDFX_ERR_INVALID_ARG;
  }
  if (c->exch) {
    set_err("idfx_step: with exchanged directions the cycle is driven through idfx_cycle_begin / idfx_stage_* / idfx_halo_*");
    return IDFX_ERR_UNSUPPORTED;
  }
  if ((rc = prepare_cycle(c))) return rc;
  return run_cycle(c, dt, 0.0);
}

// nsteps cycles with the CFL step, replayed from CUDA graphs where possible
static int advance_cycles(idfx_ctx* c, int nsteps, double cfl) {
  int rc;
  if (c->exch) {
    set_err("idfx_advance: with exchanged directions the cycle is driven through idfx_cycle_begin / idfx_stage_* / idfx_halo_*");
    return IDFX_ERR_UNSUPPORTED;
  }
  if (c->graph_cfl != cfl) {
    drop_graphs(c);
    c->graph_cfl = cfl;
  }
  for (int s = 0; s < nsteps; ++s) {
    if ((rc = prepare_cycle(c))) return rc;
    if (!c->use_graph || c->prof_on) {
      if ((rc = run_cycle(c, 0.0, cfl))) return rc;
      continue;
    }
    // the cycle is a fixed sequence of kernels whose arguments depend only on the buffer rotation state: capture it
    // once per state, then replay (dt and the clock never leave the device, so nothing else varies)
    // (a cycle fed with the conserved fields rotates only those; the other kind never runs with them swapped unless such
    // cycles came before it, and then its graphs are captured anew)
    const int key = c->cyc_ufed ? 6 + c->ucur : c->bcur * 2 + c->vcur;
    if (c->graph[key] && c->graph_ucur[key] != c->ucur) {
      cudaGraphExecDestroy(c->graph[key]);
      c->graph[key] = nullptr;
    }
    if (!c->graph[key]) {
      const int b = c->bcur, v = c->vcur, u = c->ucur;
      const bool vg = c->v_given, vs = c->v_stale, ug = c->ug_valid;
      c->graph_ucur[key] = u;
      const long long l0 = c->launches;
      cudaGraph_t gr = nullptr;
      CK(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
      rc = run_cycle(c, 0.0, cfl);
      cudaError_t e = cudaStreamEndCapture(c->stream, &gr);
      if (rc || e != cudaSuccess || !gr) {
        set_err("CUDA graph capture of the cycle failed: %s", cudaGetErrorString(e));
        return IDFX_ERR_CUDA;
      }
      CK(cudaGraphInstantiate(&c->graph[key], gr, 0));
      cudaGraphDestroy(gr);
      c->graph_launches[key] = c->launches - l0;
      c->launches = l0;  // nothing ran during capture
      c->graph_bnext[key] = c->bcur;
      c->graph_vnext[key] = c->vcur;
      c->bcur = b;
      c->vcur = v;
      c->ucur = u;
      c->v_given = vg;
      c->v_stale = vs;
      c->ug_valid = ug;
    }
    CK(cudaGraphLaunch(c->graph[key], c->stream));
    c->launches += c->graph_launches[key];
    c->bcur = c->graph_bnext[key];  // as run_cycle leaves them
    c->vcur = c->graph_vnext[key];
    after_cycle(c);
  }
  return IDFX_OK;
}

static int read_scalars(idfx_ctx* c, DevScalars* h) {
  CK(cudaMemcpyAsync(h, c->sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  return IDFX_OK;
}

int idfx_advance(idfx_ctx* c, int nsteps, double cfl) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (nsteps < 0 || !(cfl > 0.0) || !(cfl < 1.0)) {
    set_err("idfx_advance: need nsteps >= 0 and 0 < cfl < 1");
    return IDFX_ERR_INVALID_ARG;
  }
  return advance_cycles(c, nsteps, cfl);
}

int idfx_advance_to(idfx_ctx* c, double t_end, double cfl, int max_steps, int* h_nsteps_out, double* h_t_out) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (max_steps < 0 || !(cfl > 0.0) || !(cfl < 1.0) || !(t_end == t_end)) {
    set_err("idfx_advance_to: need max_steps >= 0, 0 < cfl < 1 and a t_end that is not NaN");
    return IDFX_ERR_INVALID_ARG;
  }
  DevScalars h;
  if ((rc = read_scalars(c, &h))) return rc;
  const long long n0 = h.ncycles;
  CK(cudaMemcpyAsync(&c->sc->t_end, &t_end, sizeof(double), cudaMemcpyHostToDevice, c->stream));
  long long done = 0;
  double dt_last = 0.0;
  while (h.t_next < t_end && done < max_steps) {
    // batch size: most of the cycles the last dt says are left, at least one, never past max_steps
    long long batch = dt_last > 0.0 ? (long long)(0.9 * (t_end - h.t_next) / dt_last) : 1;
    batch = batch < 1 ? 1 : (batch > 64 ? 64 : batch);
    if (c->fixed_batch > 0) batch = c->fixed_batch;
    if (batch > max_steps - done) batch = max_steps - done;
    if ((rc = advance_cycles(c, (int)batch, cfl))) break;
    if ((rc = read_scalars(c, &h))) break;
    if (h.flag) break;  // unphysical state: idfx_status reports it
    done = h.ncycles - n0;
    dt_last = h.dt_used;
    if (!(dt_last > 0.0) && h.t_next < t_end) break;  // cannot progress (dt = 0 or NaN)
  }
  const double inf = INFINITY;
  cudaMemcpyAsync(&c->sc->t_end, &inf, sizeof(double), cudaMemcpyHostToDevice, c->stream);
  if (h_nsteps_out) *h_nsteps_out = (int)done;
  if (h_t_out) *h_t_out = h.t_next;
  return rc;
}

int idfx_time(idfx_ctx* c, double* h_t_out) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!h_t_out) return IDFX_ERR_INVALID_ARG;
  DevScalars h;
  if ((rc = read_scalars(c, &h))) return rc;
  *h_t_out = h.t_next;
  return IDFX_OK;
}

int idfx_set_option(idfx_ctx* c, int option, int value) {
  if (!c) {
    set_err("null context");
    return IDFX_ERR_INVALID_ARG;
  }
  if (option == 0 /* IDFX_OPT_INTEGRATOR */ && value >= 1 && value <= 3) {
    if (value != c->nstages) drop_graphs(c);
    c->nstages = value;
    return IDFX_OK;
  }
  if (option == 3 /* IDFX_OPT_BOUNDARY */ && (value == 0 || value == 1)) {
    if (value == 1 && (c->limiter == LIM_PPM || c->emf2d() || c->vp)) {
      set_err("idfx_set_option: outflow boundaries need a three-cell reconstruction, a face-flux EMF and the face form of CT");
      return IDFX_ERR_UNSUPPORTED;
    }
    drop_graphs(c);
    c->g.outflow = value ? 0x3f : 0;
    c->g.open = (value ? 7 : 0) | c->exch;
    return IDFX_OK;
  }
  if (option == 5 /* IDFX_OPT_OUTFLOW_SIDES */ && value >= 0 && value <= 0x3f) {
    if (!c->exch) {
      set_err("idfx_set_option: per-side walls are for sub-boxes of a decomposed box (IDFX_OPT_EXCHANGE_DIRS first)");
      return IDFX_ERR_INVALID_ARG;
    }
    drop_graphs(c);
    c->g.outflow = value;
    return IDFX_OK;
  }
  if (option == 4 /* IDFX_OPT_EXCHANGE_DIRS */ && value >= 0 && value <= 7) {
    if (c->bound) {
      set_err("idfx_set_option: the exchanged directions must be chosen before idfx_bind");
      return IDFX_ERR_INVALID_ARG;
    }
    if (value && (c->limiter == LIM_PPM || c->emf2d() || c->vp)) {
      set_err("idfx_set_option: halo exchange needs a three-cell reconstruction, a face-flux EMF and the face form of CT");
      return IDFX_ERR_UNSUPPORTED;
    }
    c->exch = value;
    c->g.open = (c->g.outflow ? 7 : 0) | value;
    return IDFX_OK;
  }
  if (option == 1 /* IDFX_OPT_CT_FORM */ && (value == 0 || value == 1)) {
    if (c->bound) {
      set_err("idfx_set_option: the CT form must be chosen before idfx_bind");
      return IDFX_ERR_INVALID_ARG;
    }
    if (value == 1 && (!c->mhd || c->g.open)) {
      set_err("idfx_set_option: the vector-potential form needs a magnetic field and a periodic box");
      return IDFX_ERR_UNSUPPORTED;
    }
    c->vp = value == 1;
    return IDFX_OK;
  }
  set_err("idfx_set_option: unknown option or value");
  return IDFX_ERR_INVALID_ARG;
}

int idfx_set_option_real(idfx_ctx* c, int option, double value) {
  if (!c) {
    set_err("null context");
    return IDFX_ERR_INVALID_ARG;
  }
  if (option == 2 /* IDFX_OPT_PRESSURE_FLOOR */ && value >= 0.0) {
    if (value != c->g.pfloor) drop_graphs(c);  // kernel arguments are baked into the captured cycles
    c->g.pfloor = value;
    return IDFX_OK;
  }
  set_err("idfx_set_option_real: unknown option or value");
  return IDFX_ERR_INVALID_ARG;
}

int idfx_floor_count(idfx_ctx* c, long long* h_count_out) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!h_count_out) return IDFX_ERR_INVALID_ARG;
  DevScalars h;
  if ((rc = read_scalars(c, &h))) return rc;
  *h_count_out = (long long)h.nfloor;
  return IDFX_OK;
}

int idfx_get_potential(idfx_ctx* c, double* d_pot) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!c->vp || !d_pot) {
    set_err("idfx_get_potential: needs IDFX_CT_POTENTIAL and a non-null output");
    return IDFX_ERR_INVALID_ARG;
  }
  FieldList fl;
  fl.n = 3;
  for (int d = 0; d < 3; ++d) fl.f[d] = c->abuf(c->bcur, d);
  { LaunchScope ls(c, K_STATE);
  k_unpack<<<blocks_for(c->g.nc, 128), 128, 0, c->stream>>>(c->g, fl, d_pot);
  }
  CK(cudaGetLastError());
  return IDFX_OK;
}

// ---- the cycle in pieces, and the halo slabs (domain decomposition) ----
int idfx_cycle_begin(idfx_ctx* c, double dt, double cfl) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!(dt > 0.0) && (!(cfl > 0.0) || !(cfl < 1.0))) {
    set_err("idfx_cycle_begin: need dt > 0, or dt <= 0 and 0 < cfl < 1");
    return IDFX_ERR_INVALID_ARG;
  }
  if ((rc = prepare_cycle(c))) return rc;
  cycle_begin(c, dt > 0.0 ? dt : 0.0, cfl);
  CK(cudaGetLastError());
  return IDFX_OK;
}

static int check_stage(idfx_ctx* c, int stage, const char* who) {
  if (stage < 0 || stage >= c->nstages) {
    set_err("%s: no such stage", who);
    return IDFX_ERR_INVALID_ARG;
  }
  return IDFX_OK;
}

int idfx_stage_flux(idfx_ctx* c, int stage) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if ((rc = check_stage(c, stage, "idfx_stage_flux"))) return rc;
  stage_flux(c, stage);
  CK(cudaGetLastError());
  return IDFX_OK;
}

int idfx_stage_update(idfx_ctx* c, int stage) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if ((rc = check_stage(c, stage, "idfx_stage_update"))) return rc;
  stage_update(c, stage);
  CK(cudaGetLastError());
  return IDFX_OK;
}

int idfx_cycle_end(idfx_ctx* c) {
  int rc = check_bound(c);
  if (rc) return rc;
  cycle_end(c);
  return IDFX_OK;
}

size_t idfx_dt_reduce_offset(const idfx_ctx* c) {
  if (!c || !c->bound) return 0;
  return (size_t)((const char*)&c->sc->smax_bits - (const char*)c->ws);
}

// the fields a halo slab carries: the primitives of the stage input (with Bc) and its face field
static FieldList halo_fields(const idfx_ctx* c) {
  FieldList fl;
  fl.n = 0;
  for (int n = 0; n < c->nv(); ++n) fl.f[fl.n++] = c->vfield(n);
  if (c->mhd)
    for (int d = 0; d < 3; ++d) fl.f[fl.n++] = c->bbuf(c->cyc_bin, d);
  return fl;
}

long long idfx_halo_count(const idfx_ctx* c, int dir) {
  if (!c || !c->bound || dir < 0 || dir > 2) return 0;
  return (long long)halo_fields(c).n * slab_geom(c->g, dir, 0, SLAB_PACK, 0).count;
}

static int halo_op(idfx_ctx* c, int dir, int side, int mode, int clamp, double* d_buf, const char* who) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (dir < 0 || dir > 2 || side < 0 || side > 1 || (mode != SLAB_COPY && !d_buf)) {
    set_err("%s: need 0 <= dir <= 2, side 0 (lower) or 1 (upper) and a device buffer", who);
    return IDFX_ERR_INVALID_ARG;
  }
  if ((rc = ensure_v(c))) return rc;  // the slabs are cut from the primitive buffer
  const SlabGeom sg = slab_geom(c->g, dir, side, mode, clamp);
  const FieldList fl = halo_fields(c);
  const unsigned nb = blocks_for(sg.count, 128);
  LaunchScope ls(c, K_FILL);
  if (mode == SLAB_COPY) k_slab<SLAB_COPY><<<nb, 128, 0, c->stream>>>(c->g, sg, fl, nullptr);
  else if (mode == SLAB_PACK) k_slab<SLAB_PACK><<<nb, 128, 0, c->stream>>>(c->g, sg, fl, d_buf);
  else k_slab<SLAB_UNPACK><<<nb, 128, 0, c->stream>>>(c->g, sg, fl, d_buf);
  CK(cudaGetLastError());
  return IDFX_OK;
}

int idfx_halo_pack(idfx_ctx* c, int dir, int side, double* d_buf) { return halo_op(c, dir, side, SLAB_PACK, 0, d_buf, "idfx_halo_pack"); }
int idfx_halo_unpack(idfx_ctx* c, int dir, int side, const double* d_buf) {
  return halo_op(c, dir, side, SLAB_UNPACK, 0, const_cast<double*>(d_buf), "idfx_halo_unpack");
}
int idfx_halo_fill(idfx_ctx* c, int dir, int side, int zero_gradient) {
  return halo_op(c, dir, side, SLAB_COPY, zero_gradient ? 1 : 0, nullptr, "idfx_halo_fill");
}

int idfx_halo_push(idfx_ctx* c, int dir, int side, idfx_ctx* nb) {
  int rc = check_bound(c);
  if (rc) return rc;
  if ((rc = check_bound(nb))) return rc;
  DeviceScope on_device(c->device);
  if (dir < 0 || dir > 2 || side < 0 || side > 1) {
    set_err("idfx_halo_push: need 0 <= dir <= 2 and side 0 (lower) or 1 (upper)");
    return IDFX_ERR_INVALID_ARG;
  }
  if ((rc = ensure_v(c))) return rc;  // the slab is cut from the primitive buffer
  const SlabGeom from = slab_geom(c->g, dir, side, SLAB_PACK, 0), to = slab_geom(nb->g, dir, 1 - side, SLAB_UNPACK, 0);
  const FieldList fs = halo_fields(c), fd = halo_fields(nb);
  if (from.ext[0] != to.ext[0] || from.ext[1] != to.ext[1] || from.ext[2] != to.ext[2] || fs.n != fd.n) {
    set_err("idfx_halo_push: the two sub-boxes do not share the face they meet at (extents or scheme differ)");
    return IDFX_ERR_INVALID_ARG;
  }
  if (nb->device != c->device) {  // peer stores: once per pair of devices
    int can = 0;
    CK(cudaDeviceCanAccessPeer(&can, c->device, nb->device));
    if (!can) {
      set_err("idfx_halo_push: device of the neighbour is not peer-accessible (use idfx_halo_pack / unpack and a transport)");
      return IDFX_ERR_UNSUPPORTED;
    }
    const cudaError_t e = cudaDeviceEnablePeerAccess(nb->device, 0);
    if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) CK(e);
    cudaGetLastError();
  }
  LaunchScope ls(c, K_FILL);
  k_slab_push<<<blocks_for(from.count, 128), 128, 0, c->stream>>>(c->g, from, fs, nb->g, to, fd);
  CK(cudaGetLastError());
  return IDFX_OK;
}

int idfx_last_dt(idfx_ctx* c, double* h_dt_out) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (!h_dt_out) return IDFX_ERR_INVALID_ARG;
  CK(cudaMemcpyAsync(h_dt_out, &c->sc->dt_used, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  return IDFX_OK;
}

int idfx_status(idfx_ctx* c) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  int flag = 0;
  CK(cudaMemcpyAsync(&flag, &c->sc->flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  if (flag) {
    set_err("unphysical state (rho <= 0, p <= 0 or NaN) met on the device");
    return IDFX_ERR_UNPHYSICAL;
  }
  return IDFX_OK;
}

long long idfx_launch_count(const idfx_ctx* c) { return c ? c->launches : 0; }

int idfx_profile_enable(idfx_ctx* c, int on) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  prof_drain(c);
  for (int k = 0; k < K_COUNT; ++k) {
    c->prof_ms[k] = 0.0;
    c->prof_n[k] = 0;
  }
  c->prof_on = on != 0;
  return IDFX_OK;
}

int idfx_profile_read(idfx_ctx* c, int kernel_id, double* h_ms_total, long long* h_launches) {
  int rc = check_bound(c);
  if (rc) return rc;
  DeviceScope on_device(c->device);
  if (kernel_id < 0 || kernel_id >= K_COUNT || !h_ms_total || !h_launches) {
    set_err("idfx_profile_read: bad kernel id or null output");
    return IDFX_ERR_INVALID_ARG;
  }
  prof_drain(c);
  *h_ms_total = c->prof_ms[kernel_id];
  *h_launches = c->prof_n[kernel_id];
  return IDFX_OK;
}

const char* idfx_profile_kernel_name(int kernel_id) {
  return (kernel_id >= 0 && kernel_id < K_COUNT) ? kKernelNames[kernel_id] : nullptr;
}

void idfx_destroy(idfx_ctx* c) {
  if (!c) return;
  DeviceScope on_device(c->device);
  prof_drain(c);
  drop_graphs(c);
  for (cudaEvent_t e : c->prof_free) cudaEventDestroy(e);
  delete c;
}

}  // extern "C"
