/* idfx_noalloc.h — one entry point of libidfx.so that allocates nothing.
 *
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it) and
 * have no idfx context with its workspace at hand: the CFL time step of Eq. 10 of a periodic box given as
 * plain contiguous device arrays.  It is the standalone-dt path of idfx_compute_dt (one signal speed per face from the
 * limited face states, reading G5; per cell the larger of its two faces per direction, reading G8; the maximum over the
 * box), with its scratch memory -- one c_face per cell and direction and the 8-byte reduction word -- in a file-scope
 * `static __device__` array of the library instead of the caller's workspace.
 *
 * LIMIT: nx * ny * nz <= IDFX_NOALLOC_MAX_CELLS (64^3).  The array is 3 * IDFX_NOALLOC_MAX_CELLS doubles + 256 bytes
 * = 6.0 MiB, and every GPU that loads the library holds it until the process exits.  Larger boxes are refused with
 * IDFX_ERR_INVALID_ARG (-1) and a message (idfx_noalloc_last_error): use a context and idfx_compute_dt for those.
 *
 * SHARING: every call on a device uses the same array.  Nothing in it survives a call (the reduction word is cleared at the
 * start of every call, the c_face values are all rewritten before they are read), but two calls whose kernels overlap on the
 * GPU -- different streams, or different host threads on different streams -- RACE on it.  Calls on one stream are ordered.
 *
 * The call enqueues three kernels on `cuda_stream` of the CURRENT device, does not synchronise, and calls no cudaMalloc,
 * cudaFree or allocating library routine (the first call on a device looks up the array's device address with
 * cudaGetSymbolAddress, which allocates nothing).
 */
#ifndef IDFX_NOALLOC_H
#define IDFX_NOALLOC_H

#ifdef __cplusplus
extern "C" {
#endif

#define IDFX_NOALLOC_MAX_CELLS 262144 /* 64^3 */

/* d_prim  [5][nz][ny][nx]: rho, vx, vy, vz, p (device, read only)
 * d_bface [3][nz][ny][nx]: face field, component d on the LEFT d-face of cell (i,j,k); NULL = hydrodynamics
 * limiter: IDFX_LIMITER_FLAT / MINMOD / VANLEER / LIMO3 (0..3) as in idfx.h; PPM is refused
 * d_dt_out: one double (device, written): cfl / max_cells sum_d c_d / dx
 * Needs nx, ny, nz >= 4, dx > 0, gamma > 1, 0 < cfl < 1.  Returns IDFX_OK (0), IDFX_ERR_INVALID_ARG (-1) or IDFX_ERR_CUDA (-4). */
int idfx_noalloc_compute_dt(int nx, int ny, int nz, double dx, double gamma, int limiter, const double* d_prim,
                            const double* d_bface, double cfl, void* cuda_stream, double* d_dt_out);

/* Message of the last failed idfx_noalloc_compute_dt in this thread. */
const char* idfx_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
