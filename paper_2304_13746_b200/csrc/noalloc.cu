// noalloc.cu — the one entry point of libidfx.so that allocates nothing (include/idfx_noalloc.h): the CFL step of Eq. 10
// of a periodic box given as contiguous device arrays, with the scratch memory of the standalone-dt path
// (one c_face per cell and direction, the reduction word) in a file-scope __device__ array instead of a caller's workspace.
// Nothing else in the library uses this file, and it changes no other code path.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/idfx_noalloc.h"
#include "common.cuh"
#include "physics.cuh"

namespace {

using namespace idfx;

// [0, 32): the reduction word (bit pattern of max_cells sum_d c_d / dx) and padding to 256 bytes; then c_face[3][cells].
// In HOST code this name is only a stand-in for the symbol: the device address comes from cudaGetSymbolAddress (scratch_of).
constexpr size_t kHead = 32;  // doubles
static __device__ __align__(256) double g_scratch[kHead + 3 * (size_t)IDFX_NOALLOC_MAX_CELLS];

thread_local char g_msg[256] = "";

struct Box {
  int nx, ny, nz;
  long long nc;
  double dx, gamma;
};

__device__ __forceinline__ int wrap(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

// c_face (reading G5: Davis speeds of the limited face states) on the three lower faces of every cell; thread 0 clears the
// reduction word for the kernel that follows on the same stream
template <int LIM, bool MHD>
__global__ void __launch_bounds__(128) k_noalloc_speed(Box b, const double* __restrict__ prim, const double* __restrict__ bf,
                                                      double* __restrict__ scratch) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t == 0) *reinterpret_cast<unsigned long long*>(scratch) = 0ull;
  if (t >= b.nc) return;
  const int n[3] = {b.nx, b.ny, b.nz};
  int idx[3];
  idx[0] = (int)(t % b.nx);
  idx[1] = (int)((t / b.nx) % b.ny);
  idx[2] = (int)(t / ((long long)b.nx * b.ny));
  const double dx2 = b.dx * b.dx;
  auto at = [&](const int p[3]) { return ((long long)p[2] * b.ny + p[1]) * b.nx + p[0]; };
  // cell-centred field component m of cell p: mean of its two bounding faces (reading G1)
  auto bc = [&](int m, const int p[3]) {
    int q[3] = {p[0], p[1], p[2]};
    const double lo = bf[m * b.nc + at(q)];
    q[m] = wrap(q[m] + 1, n[m]);
    return 0.5 * (lo + bf[m * b.nc + at(q)]);
  };
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const int tb = (d + 1) % 3, te = (d + 2) % 3;
    double W[4][7];  // cells id-2 .. id+1 along d in the sweep's local order (rho, u_n, u_t1, u_t2, p, B_t1, B_t2)
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      int p[3] = {idx[0], idx[1], idx[2]};
      p[d] = wrap(idx[d] + m - 2, n[d]);
      const long long c = at(p);
      W[m][0] = prim[c];
      W[m][1] = prim[(1 + d) * b.nc + c];
      W[m][2] = prim[(1 + tb) * b.nc + c];
      W[m][3] = prim[(1 + te) * b.nc + c];
      W[m][4] = prim[4 * b.nc + c];
      W[m][5] = MHD ? bc(tb, p) : 0.0;
      W[m][6] = MHD ? bc(te, p) : 0.0;
    }
    double WL[7], WR[7];
#pragma unroll
    for (int v = 0; v < 7; ++v) {
      double drop;
      face_values<LIM>(W[1][v], W[1][v] - W[0][v], W[2][v] - W[1][v], dx2, drop, WL[v]);
      face_values<LIM>(W[2][v], W[2][v] - W[1][v], W[3][v] - W[2][v], dx2, WR[v], drop);
    }
    const double Bn = MHD ? bf[d * b.nc + t] : 0.0;  // reading G3: the staggered value on both sides
    double SL, SR;
    outer_speeds<MHD>(WL, WR, Bn, b.gamma, SL, SR);
    scratch[kHead + d * (size_t)IDFX_NOALLOC_MAX_CELLS + t] = fmax(fabs(SL), fabs(SR));
  }
}

// per cell sum_d max(c_face of its two d-faces) / dx (reading G8); warp shuffle -> block -> atomicMax on the ordered bits
__global__ void __launch_bounds__(128) k_noalloc_max(Box b, double* __restrict__ scratch) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double s = 0.0;
  if (t < b.nc) {
    const int n[3] = {b.nx, b.ny, b.nz};
    const long long st[3] = {1, b.nx, (long long)b.nx * b.ny};
    const int idx[3] = {(int)(t % b.nx), (int)((t / b.nx) % b.ny), (int)(t / ((long long)b.nx * b.ny))};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double* cf = scratch + kHead + d * (size_t)IDFX_NOALLOC_MAX_CELLS;
      const long long up = idx[d] + 1 == n[d] ? t - (long long)(n[d] - 1) * st[d] : t + st[d];
      s += fmax(cf[t], cf[up]);
    }
    s /= b.dx;
  }
  const double m = block_max_128(s);
  if (threadIdx.x == 0) atomicMax(reinterpret_cast<unsigned long long*>(scratch), (unsigned long long)__double_as_longlong(m));
}

__global__ void k_noalloc_finish(const double* __restrict__ scratch, double cfl, double* __restrict__ dt_out) {
  if (blockIdx.x == 0 && threadIdx.x == 0)
    *dt_out = cfl / __longlong_as_double((long long)*reinterpret_cast<const unsigned long long*>(scratch));
}

// Device address of g_scratch on the current device: looked up once per device, with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_lock;
double* g_addr[kMaxDevices] = {nullptr};

int scratch_of(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
    snprintf(g_msg, sizeof(g_msg), "idfx_noalloc_compute_dt: no usable current device (%s)", cudaGetErrorString(e));
    return -4;
  }
  std::lock_guard<std::mutex> guard(g_lock);
  if (!g_addr[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_scratch);
    if (e != cudaSuccess || !p) {
      snprintf(g_msg, sizeof(g_msg), "idfx_noalloc_compute_dt: cudaGetSymbolAddress failed on device %d (%s)", dev,
               cudaGetErrorString(e));
      return -4;
    }
    g_addr[dev] = p;
  }
  *out = g_addr[dev];
  return 0;
}

template <int LIM>
void launch_speed(const Box& b, const double* prim, const double* bf, double* scratch, cudaStream_t st) {
  const unsigned nb = (unsigned)((b.nc + 127) / 128);
  if (bf) k_noalloc_speed<LIM, true><<<nb, 128, 0, st>>>(b, prim, bf, scratch);
  else k_noalloc_speed<LIM, false><<<nb, 128, 0, st>>>(b, prim, bf, scratch);
}

}  // namespace

extern "C" const char* idfx_noalloc_last_error(void) { return g_msg; }

extern "C" int idfx_noalloc_compute_dt(int nx, int ny, int nz, double dx, double gamma, int limiter, const double* d_prim,
                                       const double* d_bface, double cfl, void* cuda_stream, double* d_dt_out) {
  if (nx < 4 || ny < 4 || nz < 4 || !(dx > 0.0) || !(gamma > 1.0) || !(cfl > 0.0) || !(cfl < 1.0) || !d_prim || !d_dt_out) {
    snprintf(g_msg, sizeof(g_msg), "idfx_noalloc_compute_dt: need nx, ny, nz >= 4, dx > 0, gamma > 1, 0 < cfl < 1 and non-null pointers");
    return -1;
  }
  if (limiter < LIM_FLAT || limiter > LIM_LIMO3) {
    snprintf(g_msg, sizeof(g_msg), "idfx_noalloc_compute_dt: limiter must be flat, minmod, van Leer or LimO3 (0..3)");
    return -1;
  }
  const long long nc = (long long)nx * ny * nz;
  if (nc > (long long)IDFX_NOALLOC_MAX_CELLS) {
    snprintf(g_msg, sizeof(g_msg),
             "idfx_noalloc_compute_dt: %lld cells exceed the static scratch (IDFX_NOALLOC_MAX_CELLS = %d); use a context and "
             "idfx_compute_dt", nc, IDFX_NOALLOC_MAX_CELLS);
    return -1;
  }
  double* scratch = nullptr;
  if (int rc = scratch_of(&scratch)) return rc;
  const Box b = {nx, ny, nz, nc, dx, gamma};
  cudaStream_t st = (cudaStream_t)cuda_stream;
  switch (limiter) {
    case LIM_FLAT: launch_speed<LIM_FLAT>(b, d_prim, d_bface, scratch, st); break;
    case LIM_MINMOD: launch_speed<LIM_MINMOD>(b, d_prim, d_bface, scratch, st); break;
    case LIM_LIMO3: launch_speed<LIM_LIMO3>(b, d_prim, d_bface, scratch, st); break;
    default: launch_speed<LIM_VANLEER>(b, d_prim, d_bface, scratch, st);
  }
  k_noalloc_max<<<(unsigned)((nc + 127) / 128), 128, 0, st>>>(b, scratch);
  k_noalloc_finish<<<1, 32, 0, st>>>(scratch, cfl, d_dt_out);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(g_msg, sizeof(g_msg), "idfx_noalloc_compute_dt: launch failed (%s)", cudaGetErrorString(e));
    return -4;
  }
  return 0;
}
