// stage_inst.cu — the one-kernel stages (hd_stage.cuh, hd_stage_u.cuh, mhd_stage.cuh) of one (Riemann solver, reconstruction) pair.
// build.py compiles this file once per pair (-DIDFX_INST_SOLVER=s -DIDFX_INST_LIM=l), each into its own object: the
// register allocation of these kernels sits at the edge of their occupancy target (168 registers for 384 threads) and
// was found to change with the other kernels of the translation unit and with nvcc's -split-compile partitioning, i.e.
// with unrelated edits and with the core count of the build machine.  One pair per object, no split compile: the same
// code everywhere.
#include "host.cuh"

#ifndef IDFX_INST_SOLVER
#error "compile with -DIDFX_INST_SOLVER=<0..4> -DIDFX_INST_LIM=<0..3> (paper_2304_13746_b200/build.py)"
#endif

namespace idfx {

template <int SOLVER, int LIM>
HdKernel hd_kernel_sl(bool first) {
  return first ? (HdKernel)k_hd_stage<SOLVER, LIM, true> : (HdKernel)k_hd_stage<SOLVER, LIM, false>;
}

template <int SOLVER, int LIM>
HdKernelU hd_kernel_u_sl(bool first) {
  return first ? (HdKernelU)k_hd_stage_u<SOLVER, LIM, true> : (HdKernelU)k_hd_stage_u<SOLVER, LIM, false>;
}

template <int SOLVER, int LIM, int MODE>
MhdKernel mhd_kernel_m(bool first, bool open) {
  if (open) return first ? (MhdKernel)k_mhd_stage<SOLVER, LIM, MODE, true, true> : (MhdKernel)k_mhd_stage<SOLVER, LIM, MODE, false, true>;
  return first ? (MhdKernel)k_mhd_stage<SOLVER, LIM, MODE, true, false> : (MhdKernel)k_mhd_stage<SOLVER, LIM, MODE, false, false>;
}

template <int SOLVER, int LIM>
MhdKernel mhd_kernel_sl(bool first, int emf_mode, bool open) {
  switch (emf_mode) {
    case EMF_UCT: return mhd_kernel_m<SOLVER, LIM, EMF_UCT>(first, open);
    case EMF_UCT0: return mhd_kernel_m<SOLVER, LIM, EMF_UCT0>(first, open);
    default: return mhd_kernel_m<SOLVER, LIM, EMF_ARITH>(first, open);
  }
}

// MHD: every solver but HLLC; hydrodynamics: every solver but HLLD (idfx_create refuses the other combinations)
#if IDFX_INST_SOLVER != 1
template MhdKernel mhd_kernel_sl<IDFX_INST_SOLVER, IDFX_INST_LIM>(bool, int, bool);
#endif
#if IDFX_INST_SOLVER != 2
template HdKernel hd_kernel_sl<IDFX_INST_SOLVER, IDFX_INST_LIM>(bool);
template HdKernelU hd_kernel_u_sl<IDFX_INST_SOLVER, IDFX_INST_LIM>(bool);
#endif

}  // namespace idfx
