/* idfx.h — C ABI of the B200-native (sm_100a) Godunov HD / ideal-MHD step of IDEFIX
 * (Lesur et al., arXiv 2304.13746).  Citations "PAPER.md:<line>" refer to the paper text; "O<n>" / "G<n>"
 * to the written-out formulas and readings in DESIGN.md (same numbering as SURVEY.md §8(c)).
 *
 * What one context is: a uniform periodic Cartesian box of nx*ny*nz cells with spacing dx in all three
 * directions, gamma-law gas, advanced by the explicit multi-stage cycle of PAPER.md:130-145 (Eq. 9, Tab. 1; RK2 unless
 * idfx_set_option selects Euler or RK3):
 *   cycle:  dt = cfl / max_cells sum_d c_max,d/dx                  (Eq. 10 without eta)
 *           U1 = S_dt(U0);  U = U0/2 + S_dt(U1)/2                  (Eq. 9, w2 = w2^0 = 1/2)
 *   S_dt:   periodic ghost fill -> cell-centred B and cons->prim -> PLM reconstruction of primitives to faces
 *            -> Riemann solver per face -> flux divergence (Eq. 5)
 *           -> edge EMFs -> constrained-transport update of the face-centred B (Eq. 6).
 * Every step of that path runs in CUDA kernels of this library; there is no CPU fallback.
 *
 * Conventions
 *   - All arithmetic is IEEE fp64.  No floors are applied (G13) unless IDFX_OPT_PRESSURE_FLOOR is set: rho <= 0, p <= 0
 *     or NaN met in the cons->prim conversion raises a sticky device flag reported as IDFX_ERR_UNPHYSICAL.
 *   - Array layout: structure of arrays, [var][nz][ny][nx] contiguous, x fastest, no padding.
 *       prim  : [5] = rho, vx, vy, vz, p           cons : [5] = rho, mx, my, mz, E
 *       bface : [3]; bface[d][k][j][i] is B_d on the LEFT d-face of cell (i,j,k), i.e. B_x at (i-1/2, j, k).
 *               Periodic, so face n coincides with face 0 and every component has nx*ny*nz entries.
 *     The caller must supply a discretely divergence-free bface; the library never cleans it, and its
 *     CT update keeps the discrete divergence at round-off.
 *   - E = p/(gamma-1) + rho v^2/2 + Bc^2/2 with Bc the mean of the two bounding faces (G1).
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers (pageable or pinned).
 *   - Ownership: the caller owns every buffer it passes, including the workspace (allocate it with
 *     whatever owns device memory in the application, e.g. a torch tensor).  The context owns no large
 *     device allocation; it owns CUDA graphs, TMA descriptors and a few hundred bytes of host memory.
 *   - All work is enqueued on the stream given to idfx_bind (a cudaStream_t cast to void*, NULL = legacy
 *     default stream).  Only idfx_compute_dt, idfx_last_dt, idfx_status, idfx_advance_to, idfx_time, idfx_floor_count,
 *     idfx_set_state_host and idfx_get_state_host synchronise with the host (the host-buffer calls return when the copy is done,
 *     so the caller may reuse or free its buffers immediately).
 *   - Errors: every int-returning call returns IDFX_OK or a negative code; nothing throws or aborts.
 *     idfx_last_error() gives a thread-local message for the last failure.
 */
#ifndef IDFX_H
#define IDFX_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct idfx_ctx idfx_ctx;

/* Riemann solvers, here listed by number; the paper orders them from most to least diffusive:
 * Rusanov (local Lax-Friedrichs), HLL, HLLC / HLLD, Roe.  HLLC is hydrodynamics-only; in MHD it is replaced by HLLD. */
enum { IDFX_SOLVER_HLL = 0, IDFX_SOLVER_HLLC = 1, IDFX_SOLVER_HLLD = 2, IDFX_SOLVER_ROE = 3, IDFX_SOLVER_RUSANOV = 4 };
/* Reconstruction: flat (1st order), PLM with minmod or van Leer (harmonic mean, G2) slopes, and the compact
 * third-order LimO3 of Cada & Torrilhon 2009 (same 3-cell stencil and 2 ghost layers; constants in reading G18). */
enum { IDFX_LIMITER_FLAT = 0, IDFX_LIMITER_MINMOD = 1, IDFX_LIMITER_VANLEER = 2, IDFX_LIMITER_LIMO3 = 3,
       /* piecewise parabolic with the extremum-preserving limiter (Colella & Woodward 1984, Colella & Sekora
        * 2008; reading G22): five-cell stencils, evaluated outside the tuned sweeps (one kernel per direction plus a
        * divergence pass; +18 workspace fields); periodic boxes only, not with IDFX_EMF_UCT_HLL */
       IDFX_LIMITER_PPM = 4 };
/* EMF reconstruction: arithmetic average of the face fluxes, the E^0 and E^c (upwind-contact)
 * schemes of Gardiner & Stone 2005, and the 2D HLL Riemann solver at the edges after Mignone & Del Zanna 2021 (reading G21;
 * consistent in the plane-parallel limit with the HLL face solver) and its HLLD counterpart (reading G24: the same two
 * transports with the response coefficients of the HLLD face solves; plane-parallel limit = the 1D HLLD flux; with
 * IDFX_SOLVER_HLLD only).  IDFX_EMF_NONE selects hydrodynamics (no magnetic field at all). */
enum { IDFX_EMF_NONE = 0, IDFX_EMF_ARITHMETIC = 1, IDFX_EMF_UCT_CONTACT = 2, IDFX_EMF_UCT_0 = 3, IDFX_EMF_UCT_HLL = 4,
       IDFX_EMF_UCT_HLLD = 5 };
enum {
  IDFX_OK = 0,
  IDFX_ERR_INVALID_ARG = -1,
  IDFX_ERR_UNSUPPORTED = -2, /* solver / emf_mode combination that does not exist (HLLC+MHD, HLLD+HD) */
  IDFX_ERR_NOT_BOUND = -3,   /* call needs idfx_bind first */
  IDFX_ERR_CUDA = -4,        /* a CUDA runtime call failed; see idfx_last_error() */
  IDFX_ERR_UNPHYSICAL = -5   /* sticky: rho <= 0 or p <= 0 or NaN was met on the device */
};

/* Creates a context.  Requirements: nx, ny, nz >= 4; dx > 0; gamma > 1; valid enums; HD (emf_mode NONE)
 * with RUSANOV/HLL/HLLC/ROE, MHD with RUSANOV/HLL/HLLD/ROE.  Returns NULL on error (idfx_last_error() says why).
 * Host-only: touches no device memory. */
idfx_ctx* idfx_create(int nx, int ny, int nz, double dx, double gamma, int solver, int limiter, int emf_mode);

/* Options beyond the arguments of idfx_create.
 *   IDFX_OPT_INTEGRATOR: number of stages of the explicit integrator of Tab. 1: 1 = Euler,
 *     2 = RK2 (default), 3 = RK3 (w2 = 1/4, w2^0 = 3/4, w3 = 2/3, w3^0 = 1/3).  May be changed at any time between cycles.
 *   IDFX_OPT_CT_FORM: IDFX_CT_FACE (default) evolves the face field with Eq. 6; IDFX_CT_POTENTIAL evolves the
 *     edge-centred vector potential, dA/dt = -E, and sets B = B_ref + curl A after every stage (Eq. 7-8),
 *     so that round-off cannot accumulate in div B.  B_ref is the face field given to idfx_set_state and A counts from
 *     zero there (reading G19: a periodic A cannot carry a mean field).  MHD only; must be chosen BEFORE
 *     idfx_workspace_bytes / idfx_bind (it needs 12 more fields).
 *   IDFX_OPT_BOUNDARY: IDFX_BOUNDARY_PERIODIC (default) or IDFX_BOUNDARY_OUTFLOW: zero-gradient ghost cells on all six
 *     sides (the paper's non-periodic tests).  With a magnetic field (reading G23) the staggered
 *     components are zero-gradient as well: every ghost face copies the nearest face of the state along its line, the
 *     upper boundary face (index n, not part of the state) included.  Needs a three-cell reconstruction (not PPM), a
 *     face-flux EMF (not IDFX_EMF_UCT_HLL) and IDFX_CT_FACE (IDFX_ERR_UNSUPPORTED otherwise); set it before idfx_set_state.
 *   IDFX_OPT_EXCHANGE_DIRS: bit d set = the ghost layers of direction d (0 = x, 1 = y, 2 = z) are the cells of a
 *     neighbouring sub-box of a domain decomposition and arrive through idfx_halo_unpack.  The context
 *     then never wraps periodically along d, and the CALLER drives every cycle through the staged calls below.  Same
 *     restrictions as outflow; must be chosen BEFORE idfx_bind.
 *   IDFX_OPT_OUTFLOW_SIDES: for a sub-box of a decomposed box with outflow boundaries: bit 2 d + side (side 0 lower,
 *     1 upper) set = that side of the sub-box is a wall of the whole box (its ghosts are then filled with
 *     idfx_halo_fill(d, side, 1) by the caller).  Every direction of such a run must be exchanged or walled. */
enum { IDFX_OPT_INTEGRATOR = 0, IDFX_OPT_CT_FORM = 1, IDFX_OPT_PRESSURE_FLOOR = 2, IDFX_OPT_BOUNDARY = 3, IDFX_OPT_EXCHANGE_DIRS = 4,
       IDFX_OPT_OUTFLOW_SIDES = 5 };
enum { IDFX_CT_FACE = 0, IDFX_CT_POTENTIAL = 1 };
enum { IDFX_BOUNDARY_PERIODIC = 0, IDFX_BOUNDARY_OUTFLOW = 1 };
int idfx_set_option(idfx_ctx* ctx, int option, int value);
/* Real-valued options.  IDFX_OPT_PRESSURE_FLOOR (default 0 = none, reading G13): when > 0, a pressure below it met in
 * the cons->prim conversion is raised to it and the total energy of the cell is rewritten to match (energy is then no
 * longer conserved in that cell; idfx_floor_count says how often this happened since idfx_set_state).  The paper describes
 * no such fix, but without one its own 3D Orszag-Tang run with HLLD meets p < 0 before t = 1 (DESIGN.md,
 * reading G20).  May be changed between cycles. */
int idfx_set_option_real(idfx_ctx* ctx, int option, double value);
int idfx_floor_count(idfx_ctx* ctx, long long* h_count_out); /* synchronises */

/* Device bytes the caller must supply to idfx_bind (internal padded state, stage buffers, divergence, edge EMFs): 43 padded
 * fields of (nx + 18 rounded up to 16) * (ny + 4) * (nz + 4) doubles for MHD, 25 for hydrodynamics, more with PPM, the
 * vector-potential form (choose it first) or the 2D EMFs; DESIGN.md section 6.  No call touches memory outside it. */
size_t idfx_workspace_bytes(const idfx_ctx* ctx);

/* Binds a caller-owned device workspace (>= idfx_workspace_bytes, 256-byte aligned) and a stream.
 * Zeroes the workspace on that stream.  Must precede every call below.  The stream and every device pointer passed to
 * later calls must belong to the device that holds the workspace; the calls themselves may be made with any device
 * current in the calling thread (the library switches to the workspace's device and restores the caller's). */
int idfx_bind(idfx_ctx* ctx, void* d_workspace, size_t bytes, void* cuda_stream);

/* Copy-in of the state (O1): Bc from faces, then conserved variables from the primitives.
 * d_bface may be NULL only when emf_mode is NONE (it is ignored then). */
int idfx_set_state(idfx_ctx* ctx, const double* d_prim, const double* d_bface);
int idfx_set_state_host(idfx_ctx* ctx, const double* h_prim, const double* h_bface); /* synchronises */

/* Copy-out: primitives re-derived from the conserved state and the face field; bface bit-exact. */
int idfx_get_state(idfx_ctx* ctx, double* d_prim, double* d_bface);
int idfx_get_state_host(idfx_ctx* ctx, double* h_prim, double* h_bface); /* synchronises */
/* Copy-out of the master state as it is stored: conserved cell variables and face B. */
int idfx_get_conserved(idfx_ctx* ctx, double* d_cons, double* d_bface);

/* dt of Eq. 10 on the CURRENT state (O9): cfl / max_cells [ sum_d c_d / dx ], with c_d of a
 * cell the larger c_face of its two d-faces (G8) and c_face = max(|S_L|,|S_R|) of the Davis estimate (G5).
 * 0 < cfl < 1.  Writes *h_dt_out; synchronises. */
int idfx_compute_dt(idfx_ctx* ctx, double cfl, double* h_dt_out);

/* One cycle of the integrator (RK2 by default) with the given dt > 0 (O12). */
int idfx_step(idfx_ctx* ctx, double dt);

/* nsteps cycles, each with dt evaluated on the state at the start of that cycle (G9); dt never leaves the
 * device.  Equivalent to nsteps x { idfx_compute_dt; idfx_step }.  When the bound stream is not the default stream the
 * cycle (9 kernels for RK2 MHD) is captured once per buffer-rotation state into a CUDA graph and replayed
 * (IDFX_GRAPH=0 in the environment disables this). */
int idfx_advance(idfx_ctx* ctx, int nsteps, double cfl);

/* Cycles with the CFL step until the time t_end (time counts from 0 at idfx_set_state; the paper's runs are "to t = ...",
 * PAPER.md:346): a step that would reach or pass t_end is shortened on the device to land on it exactly.  Stops early
 * after max_steps cycles.  Cycles are enqueued in batches and the device clock is read back between batches
 * (synchronises); a cycle enqueued past t_end leaves the state bit-for-bit unchanged.  Writes the number of cycles
 * taken by this call and the time reached (either may be NULL). */
int idfx_advance_to(idfx_ctx* ctx, double t_end, double cfl, int max_steps, int* h_nsteps_out, double* h_t_out);

/* Time reached since idfx_set_state (synchronises). */
int idfx_time(idfx_ctx* ctx, double* h_t_out);

/* IDFX_CT_POTENTIAL only: the edge potential accumulated since idfx_set_state, d_pot[c][k][j][i] = A_c on the lower
 * edges of cell (i,j,k): A_x at (i, j-1/2, k-1/2), A_y at (i-1/2, j, k-1/2), A_z at (i-1/2, j-1/2, k). */
int idfx_get_potential(idfx_ctx* ctx, double* d_pot);

/* ---- The cycle in pieces, for a domain decomposition over several contexts (one per GPU) -------
 * One sub-box per context, IDFX_OPT_EXCHANGE_DIRS set.  Per cycle, identically on every sub-box:
 *     idfx_cycle_begin(dt <= 0, cfl)
 *     for s in 0 .. stages-1:
 *         idfx_stage_flux(s)                  reconstruct -> Riemann -> divergence -> edge EMFs; s = 0 also reduces the
 *                                             sub-box's max_cells sum_d c_d/dx into 8 bytes of the workspace
 *         [s = 0: max over all sub-boxes of those 8 bytes, written back in place: Eq. 10's "entire integration volume"]
 *         idfx_stage_update(s)                CT, RK combine, cons -> prim of the stage result (no ghost layer is written)
 *         for d in x, y, z (this order fills edges and corners):
 *             exchanged d:  idfx_halo_pack(d, side) on both sides -> the neighbours -> idfx_halo_unpack(d, side)
 *             otherwise:    idfx_halo_fill(d, side, zero_gradient) on both sides
 *     idfx_cycle_end()
 * A slab carries the primitives (with Bc) and the face field of the stage result: idfx_halo_count(d) doubles, layout
 * [field][z][y][x] of the two layers, spanning the ghost layers of the directions below d.  What one sub-box packs on its
 * upper side is what its upper neighbour unpacks on its lower side.  Setting the state: idfx_set_state (copy-in only),
 * the same ghost sequence (the face field must reach the ghosts before Bc is formed), idfx_set_state_finish, the ghost
 * sequence again.  Every sub-box then computes bit for bit what the undecomposed box computes (tests/test_gpu_decomp.py).
 * The staged calls also work without exchanged directions (they are what idfx_step runs).
 * idfx_dt_reduce_offset: byte offset inside the bound workspace of the 8-byte reduction word; it holds a non-negative
 * double, so an elementwise MAX of doubles over the sub-boxes is the reduction.  All on the bound stream, none synchronises. */
int       idfx_cycle_begin(idfx_ctx* ctx, double dt, double cfl);   /* dt > 0: fixed step; else the CFL step */
int       idfx_stage_flux(idfx_ctx* ctx, int stage);
int       idfx_stage_update(idfx_ctx* ctx, int stage);
int       idfx_cycle_end(idfx_ctx* ctx);
size_t    idfx_dt_reduce_offset(const idfx_ctx* ctx);
int       idfx_set_state_finish(idfx_ctx* ctx);
long long idfx_halo_count(const idfx_ctx* ctx, int dir);
int       idfx_halo_pack(idfx_ctx* ctx, int dir, int side, double* d_buf);          /* side 0: lower, 1: upper */
int       idfx_halo_unpack(idfx_ctx* ctx, int dir, int side, const double* d_buf);
int       idfx_halo_fill(idfx_ctx* ctx, int dir, int side, int zero_gradient);      /* periodic image, or the nearest layer */
/* Pack and unpack in one launch when the neighbour is a context of the SAME process: the two active layers next to `side`
 * of ctx are written straight into the ghost layers of the opposite side of `neighbour` (peer stores over NVLink when it is
 * bound on another, peer-accessible device; IDFX_ERR_UNSUPPORTED when it is not).  Enqueued on ctx's stream: the caller
 * orders it after the neighbour's last use of those ghost layers and before its next one. */
int       idfx_halo_push(idfx_ctx* ctx, int dir, int side, idfx_ctx* neighbour);

/* dt used by the most recent cycle (synchronises). */
int idfx_last_dt(idfx_ctx* ctx, double* h_dt_out);

/* Synchronises; IDFX_OK, IDFX_ERR_UNPHYSICAL (sticky device flag) or IDFX_ERR_CUDA. */
int idfx_status(idfx_ctx* ctx);

/* Number of kernels of this library launched on behalf of ctx since idfx_bind (graph replays included). */
long long idfx_launch_count(const idfx_ctx* ctx);

/* Per-kernel timing for the roofline report.  While enabled, every kernel launch of ctx is bracketed by a
 * CUDA-event pair on the bound stream.  idfx_profile_enable(ctx, 1) clears the accumulators and starts,
 * (ctx, 0) stops.  idfx_profile_read synchronises and returns the summed device time in milliseconds and
 * the number of launches of kernel class kernel_id; idfx_profile_kernel_name gives the class names
 * ("flux_x", "flux_y", "flux_z", "rhs_dtmax", "edge_emf", "ct_update_prim", "ghost_fill", "state_io", "hd_stage"), NULL past
 * the end. */
int idfx_profile_enable(idfx_ctx* ctx, int on);
int idfx_profile_read(idfx_ctx* ctx, int kernel_id, double* h_ms_total, long long* h_launches);
const char* idfx_profile_kernel_name(int kernel_id);

const char* idfx_last_error(void);
void idfx_destroy(idfx_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* IDFX_H */
