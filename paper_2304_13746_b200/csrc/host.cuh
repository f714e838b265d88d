// host.cuh — host-side context of the idfx CUDA path, shared by the translation units of libidfx.so:
// idfx.cu (C ABI, state kernels, fused CT/update kernel) and stage_inst.cu (the one-kernel stages, compiled once per
// Riemann solver and reconstruction so that the code generated for one combination does not depend on the others).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <vector>

#include "../../include/idfx.h"
#include "common.cuh"
#include "physics.cuh"
#include "hd_stage.cuh"
#include "hd_stage_u.cuh"
#include "mhd_stage.cuh"

namespace idfx {

// field slots in the workspace
enum {
  F_UA = 0,    // 5 + 5: conserved state at the start of the cycle (and its result), and the stage-1 state (RK3) or the
  F_UB = 5,    //        result of a hydrodynamic cycle fed with the conserved fields; idfx_ctx::f_u / f_ub say which is which
  F_BA = 10,   // 3 x 3: face-field buffers that rotate between B0 / B1 / result
  F_BB = 13,
  F_BC = 16,
  // then, at offsets that depend on what the context needs (idfx_ctx::f_v .. f_count; hydrodynamics has no face field,
  // only PPM reads -(v x Bc), face fluxes of B and sign bytes back from memory):
  //   V, V2  2 x nv(): primitives, cell-centred B (MHD) and Ec = -(v x Bc) (PPM) of the stage input, double-buffered
  //          (the update kernels read the stage input of neighbouring tiles while writing the result)
  //   R      5: flux divergence
  //   FB     nfb(): the edge EMFs E_x, E_y, E_z of the one-kernel MHD stage in the first three; PPM: face fluxes of B, [d][0..1]
  //   SG     nsg(): 1 slot holding three byte fields, the sign of the face mass flux per direction (PPM with E^c only)
  // optional groups, appended in this order when present (idfx_ctx::f_aa, f_bref, f_h2d, f_eg):
  //   vector-potential form (idfx_set_option(IDFX_OPT_CT_FORM, IDFX_CT_POTENTIAL)): 3 x 3 edge-potential buffers rotating
  //   like the face-field buffers, and the 3 face fields given to set_state (ghosts filled);
  //   2D-HLL EMF: 3 x 4 face quantities of k_flux_face<FMODE 2> and the 3 edge EMFs
  //   PPM: 3 x 5 face fluxes of (rho, m, E) and the 3 c_face fields of k_flux_face_ppm
  N_VP = 12,
  N_H2D = 15,
  N_H2D_D = 18,   // 2D-HLLD EMF: 3 x 5 face quantities and the 3 edge EMFs
  N_GEN = 18
};

}  // namespace idfx

using namespace idfx;  // internal header: the context below is written in the library's own names

// kernel classes for idfx_profile_* (order = idfx_profile_kernel_name)
enum { K_FLUX_X = 0, K_FLUX_Y, K_FLUX_Z, K_RHS, K_EMF, K_UPDATE, K_FILL, K_STATE, K_HD, K_MHD, K_COUNT };
static const char* const kKernelNames[K_COUNT] = {"flux_x", "flux_y", "flux_z", "rhs_dtmax", "edge_emf",
                                                  "ct_update_prim", "ghost_fill", "state_io", "hd_stage", "mhd_stage"};

struct idfx_ctx {
  idfx::Geom g;
  int solver, limiter, emf;
  bool mhd;
  double* ws = nullptr;
  size_t ws_bytes = 0;
  cudaStream_t stream = nullptr;
  int device = -1;  // the device that holds the workspace (idfx_bind); every call runs there
  int sms = 148;    // its SM count
  bool bound = false;
  idfx::DevScalars* sc = nullptr;
  int nstages = 2;  // Tab. 1: 1 Euler, 2 RK2, 3 RK3
  bool vp = false;  // Eq. 7-8 instead of Eq. 6
  int fixed_batch = 0;  // IDFX_ADVANCE_BATCH: cycles per batch of idfx_advance_to (tests: forces cycles past t_end)
  int nbf() const { return mhd ? 9 : 0; }
  int nv() const { return mhd ? (limiter == LIM_PPM ? 11 : 8) : 5; }
  int nfb() const { return limiter == LIM_PPM ? 6 : (mhd ? 3 : 0); }
  int nsg() const { return limiter == LIM_PPM ? 1 : 0; }
  int f_v() const { return F_BA + nbf(); }
  int f_v2() const { return f_v() + nv(); }
  int f_r() const { return f_v2() + nv(); }
  int f_fb() const { return f_r() + 5; }
  int f_sg() const { return f_fb() + nfb(); }
  int f_count() const { return f_sg() + nsg(); }
  int f_aa() const { return f_count(); }
  int f_bref() const { return f_count() + 9; }
  int f_h2d() const { return f_count() + (vp ? N_VP : 0); }
  bool emf2d() const { return emf == EMF_UCT_HLL || emf == EMF_UCT_HLLD; }  // edge EMFs from their own kernels (k_emf_hll2d)
  int f_eg() const { return f_h2d() + (emf == EMF_UCT_HLLD ? 15 : 12); }
  int f_gen() const { return f_h2d() + (emf == EMF_UCT_HLL ? N_H2D : (emf == EMF_UCT_HLLD ? N_H2D_D : 0)); }
  int nfields() const { return f_gen() + (limiter == LIM_PPM ? N_GEN : 0); }
  double* abuf(int which, int d) const { return field(f_aa() + 3 * which + d); }
  int exch = 0;  // bit d set: the ghost layers of direction d come from a neighbouring sub-box (idfx_halo_*), the caller
                 // drives the cycle through the staged calls
  // the running cycle (cycle_begin .. cycle_end)
  double cyc_dt_fixed = 0.0, cyc_cfl = 0.0;
  int cyc_b0 = 0, cyc_bin = 0;  // saved face buffer; face buffer of the next stage's input (= bcur between cycles)
  int bcur = 0;  // which of the three face-field buffers holds the current state
  int vcur = 0;  // which primitive buffer holds the stage input
  // one captured CUDA graph per buffer rotation state (3 face-field rotations x 2 primitive buffers) and one for the
  // hydrodynamic cycle fed with the conserved fields per role of the two conserved buffers
  static constexpr int N_GRAPHS = 8;
  int graph_bnext[N_GRAPHS] = {0}, graph_vnext[N_GRAPHS] = {0};  // rotation state a replayed cycle leaves
  int graph_ucur[N_GRAPHS] = {0};                                // conserved-buffer roles a graph was captured with
  cudaGraphExec_t graph[N_GRAPHS] = {nullptr};
  long long graph_launches[N_GRAPHS] = {0};
  double graph_cfl = 0.0;
  bool use_graph = true;
  bool fused = false;              // one kernel per stage (hd_stage.cuh, mhd_stage.cuh): every reconstruction but PPM
  CUtensorMap mapHD;               // HD: 36 x 11 x 1 x 5 boxes over the primitive fields
  CUtensorMap mapHU, mapHR;        // the same boxes over U_A and over R (hd_stage_u.cuh)
  // hydrodynamic RK2 cycles fed with the conserved fields (hd_stage_u.cuh) never write the primitive buffers:
  bool v_given = true;    // V holds the caller's primitives (set_state): the next cycle reconstructs from exactly those
  bool v_stale = false;   // V is older than U_A
  bool ug_valid = false;  // the ghost layers of U_A hold its periodic images
  bool cyc_ufed = false;  // the running cycle is of that kind
  int ucur = 0;           // which conserved buffer holds the state (only those cycles swap them)
  int f_u() const { return ucur ? F_UB : F_UA; }
  int f_ub() const { return ucur ? F_UA : F_UB; }
  CUtensorMap mapMV, mapMB;        // MHD: 36 x (TY+3) x 1 x 8 boxes over the primitives, 34 x TY x 1 x 3 over the face-field buffers
  long long launches = 0;
  // optional per-kernel timing with CUDA events on the bound stream (idfx_profile_*)
  bool prof_on = false;
  struct ProfRec { cudaEvent_t a, b; int id; };
  std::vector<ProfRec> prof_pending;
  std::vector<cudaEvent_t> prof_free;
  double prof_ms[K_COUNT] = {0};
  long long prof_n[K_COUNT] = {0};
  double* field(int slot) const { return ws + (size_t)slot * (size_t)g.np; }
  double* bbuf(int which, int d) const { return field(F_BA + 3 * which + d); }
  signed char* sgn(int d) const { return (signed char*)field(f_sg()) + (size_t)d * (size_t)g.np; }
  double* vfield(int n) const { return field((vcur ? f_v2() : f_v()) + n); }
  double* vfield_out(int n) const { return field((vcur ? f_v() : f_v2()) + n); }
};

namespace idfx {
inline cudaEvent_t prof_event(idfx_ctx* c) {
  if (!c->prof_free.empty()) {
    cudaEvent_t e = c->prof_free.back();
    c->prof_free.pop_back();
    return e;
  }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}
inline void prof_drain(idfx_ctx* c) {
  for (auto& r : c->prof_pending) {
    float ms = 0.f;
    cudaEventSynchronize(r.b);
    cudaEventElapsedTime(&ms, r.a, r.b);
    c->prof_ms[r.id] += ms;
    c->prof_n[r.id] += 1;
    c->prof_free.push_back(r.a);
    c->prof_free.push_back(r.b);
  }
  c->prof_pending.clear();
}
// brackets one kernel launch: counts it and, when profiling is on, times it with an event pair
struct LaunchScope {
  idfx_ctx* c;
  int id;
  cudaEvent_t a = nullptr;
  LaunchScope(idfx_ctx* c_, int id_) : c(c_), id(id_) {
    if (c->prof_on) {
      a = prof_event(c);
      cudaEventRecord(a, c->stream);
    }
  }
  ~LaunchScope() {
    c->launches++;
    if (c->prof_on) {
      cudaEvent_t b = prof_event(c);
      cudaEventRecord(b, c->stream);
      c->prof_pending.push_back({a, b, id});
      if (c->prof_pending.size() >= 4096) prof_drain(c);
    }
  }
};

inline unsigned blocks_for(long long n, int bs) { return (unsigned)((n + bs - 1) / bs); }

// Hydrodynamics: the whole stage in one kernel (hd_stage.cuh); defined and explicitly instantiated in stage_inst.cu.
typedef void (*HdKernel)(Geom, HdStageArgs, const CUtensorMap);
template <int SOLVER, int LIM>
HdKernel hd_kernel_sl(bool first);

typedef void (*HdKernelU)(Geom, HdStageArgs, const CUtensorMap, const CUtensorMap);
template <int SOLVER, int LIM>
HdKernelU hd_kernel_u_sl(bool first);

// MHD: the three sweeps and the edge EMFs of a stage in one kernel (mhd_stage.cuh), same translation units.
typedef void (*MhdKernel)(Geom, MhdStageArgs, const CUtensorMap, const CUtensorMap);
template <int SOLVER, int LIM>
MhdKernel mhd_kernel_sl(bool first, int emf_mode, bool open);

}  // namespace idfx
