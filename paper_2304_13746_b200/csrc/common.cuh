// common.cuh — geometry of the padded fields and the device scalars shared by all kernels of the idfx CUDA path.
#pragma once
#include <cuda_runtime.h>

namespace idfx {

constexpr int NG = 2;
constexpr int IOFF = 16;

struct Geom {
  int nx, ny, nz;
  int sy;         // row pitch in doubles
  long long sz;   // plane stride in doubles
  long long np;   // padded field size in doubles
  long long nc;   // nx*ny*nz
  double dx, gamma;
  int outflow;    // bit 2 d + side set: that side (0 lower, 1 upper) of direction d is an outflow wall with zero-gradient ghosts;
                  // 0: none (periodic box, or a sub-box inside a decomposed one); 0x3f: all six sides
  int open;       // bit d set: the kernels do not wrap periodically along direction d -- the edge lattice keeps its plane of
                  // index n, nobody writes periodic ghost images, and the ghost layers are filled by a separate pass
                  // (zero-gradient copies for outflow, the neighbour's cells under a domain decomposition).  0: periodic box
  double pfloor;  // > 0: pressures below it are raised to it in cons->prim and E is rewritten (idfx_set_option_real); 0: none (G13)
  __host__ __device__ __forceinline__ long long at(int i, int j, int k) const {
    return (long long)(k + NG) * sz + (long long)(j + NG) * sy + (i + IOFF);
  }
};

// flat thread index -> active cell
__device__ __forceinline__ bool cell_of_thread(const Geom& g, int& i, int& j, int& k) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= g.nc) return false;
  i = (int)(t % g.nx);
  const long long r = t / g.nx;
  j = (int)(r % g.ny);
  k = (int)(r / g.ny);
  return true;
}

struct DevScalars {
  unsigned long long smax_bits;  // bit pattern of max_cells sum_d c_d/dx (positive doubles order like integers)
  double dt_used;                // dt of the running cycle, written by the update kernel of its first stage
  int flag;
  int pad_;
  double t;                      // time at the start of the running cycle (committed by k_cycle_begin)
  double t_next;                 // time at its end
  double t_end;                  // +inf, or the target of idfx_advance_to: a step that would pass it lands on it
  long long ncycles;             // cycles with dt > 0 since set_state
  unsigned long long nfloor;     // cells raised to the pressure floor since set_state
};

// dt of the cycle as the first stage's update kernel sees it (every thread evaluates the same expression):
// the fixed step, or Eq. 10 from the reduced maximum, shortened to land on t_end.
__device__ __forceinline__ double first_stage_dt(const DevScalars* sc, double dt_fixed, double cfl, bool& lands) {
  double dt = dt_fixed;
  lands = false;
  if (!(dt > 0.0)) {
    dt = cfl / __longlong_as_double((long long)sc->smax_bits);
    const double remaining = sc->t_end - sc->t;
    lands = dt >= remaining;
    if (lands) dt = remaining;
  }
  return dt;
}

// thread 0 of block 0 of that kernel publishes it
__device__ __forceinline__ void publish_dt(DevScalars* sc, double dt, bool lands) {
  sc->dt_used = dt;
  sc->t_next = lands ? sc->t_end : sc->t + dt;
  if (dt > 0.0) sc->ncycles += 1;
}

// pulls a line into L1 ahead of its use; costs no register
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// sign of a face mass flux as one byte (+1, -1, 0): all the upwind-contact EMF needs of it (G10)
__device__ __forceinline__ signed char flux_sign(double f) { return f > 0.0 ? 1 : (f < 0.0 ? -1 : 0); }

// block-wide maximum for blocks of exactly 128 threads; every thread must call it
__device__ __forceinline__ double block_max_128(double v) {
  __shared__ double red[4];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  return fmax(fmax(red[0], red[1]), fmax(red[2], red[3]));
}

}  // namespace idfx
