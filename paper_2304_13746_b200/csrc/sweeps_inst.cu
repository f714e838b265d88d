// sweeps_inst.cu — the flux sweeps of one (Riemann solver, reconstruction) pair: x sweep (shuffle windows and TMA rows),
// marching y / z sweeps (register prefetch and TMA ring), and the one-kernel hydrodynamics stage.  build.py compiles this
// file once per pair (-DIDFX_INST_SOLVER=s -DIDFX_INST_LIM=l), each into its own object: the register allocation of
// these kernels sits at the edge of 3 CTAs per SM (168 registers) and was found to change with the other kernels of the
// translation unit and with nvcc's -split-compile partitioning, i.e. with unrelated edits and with the core count of
// the build machine (z sweep at 512^3: 5.8 or 6.9 ms).  One pair per object, no split compile: the same code everywhere.
#include "host.cuh"

#ifndef IDFX_INST_SOLVER
#error "compile with -DIDFX_INST_SOLVER=<0..4> -DIDFX_INST_LIM=<0..3> (paper_2304_13746_b200/build.py)"
#endif

namespace idfx {

template <int SOLVER, int LIM, bool MHD>
void launch_x_tma(idfx_ctx* c, dim3 grid, const FluxXTArgs& ta) {
  if constexpr (MHD) k_flux_x_tma<SOLVER, LIM><<<grid, 128, 0, c->stream>>>(c->g, ta, c->mapV[0], c->mapB[0]);
}

template <int SOLVER, int LIM, bool MHD>
void launch_march_tma(idfx_ctx* c, int d, dim3 grid, const FluxTArgs& ta, bool want_dt, bool uct, bool apply) {
  if constexpr (MHD) {
    const Geom& g = c->g;
    if (d == 1) {
      if (want_dt) k_flux_march_tma<SOLVER, LIM, 1, true, true, false><<<grid, 128, 0, c->stream>>>(g, ta, c->mapV[1], c->mapB[1]);
      else if (uct) k_flux_march_tma<SOLVER, LIM, 1, false, true, false><<<grid, 128, 0, c->stream>>>(g, ta, c->mapV[1], c->mapB[1]);
      else k_flux_march_tma<SOLVER, LIM, 1, false, false, false><<<grid, 128, 0, c->stream>>>(g, ta, c->mapV[1], c->mapB[1]);
    } else if (apply) {
      if (uct) k_flux_march_tma<SOLVER, LIM, 2, false, true, true><<<grid, 128, 0, c->stream>>>(g, ta, c->mapV[2], c->mapB[2]);
      else k_flux_march_tma<SOLVER, LIM, 2, false, false, true><<<grid, 128, 0, c->stream>>>(g, ta, c->mapV[2], c->mapB[2]);
    } else {
      if (want_dt) k_flux_march_tma<SOLVER, LIM, 2, true, true, false><<<grid, 128, 0, c->stream>>>(g, ta, c->mapV[2], c->mapB[2]);
      else if (uct) k_flux_march_tma<SOLVER, LIM, 2, false, true, false><<<grid, 128, 0, c->stream>>>(g, ta, c->mapV[2], c->mapB[2]);
      else k_flux_march_tma<SOLVER, LIM, 2, false, false, false><<<grid, 128, 0, c->stream>>>(g, ta, c->mapV[2], c->mapB[2]);
    }
  }
}

template <int SOLVER, int LIM, bool MHD>
void launch_sweeps_t(idfx_ctx* c, const double* const Bf[3], bool want_dt, const ApplyInfo& ap) {
  const Geom& g = c->g;
  const bool uct = c->emf == EMF_UCT;
  {  // x: faces 0..nx of every row
    FluxXArgs a;
    a.q[0] = c->vfield(0);
    a.q[1] = c->vfield(1);
    a.q[2] = c->vfield(2);
    a.q[3] = c->vfield(3);
    a.q[4] = c->vfield(4);
    a.q[5] = c->vfield(6);
    a.q[6] = c->vfield(7);
    a.bn = MHD ? Bf[0] : nullptr;
    for (int n = 0; n < 5; ++n) a.FH[n] = c->field(F_FX + n);
    a.FB[0] = c->field(F_FB + 0);
    a.FB[1] = c->field(F_FB + 1);
    a.cf = want_dt ? c->field(F_CFX) : nullptr;
    a.sg = uct ? c->sgn(0) : nullptr;
    const int gx = (g.nx + 1 + 30) / 31;
    const long long nrows = (long long)g.ny * g.nz;
    long long rpw = gx * nrows / 9472;
    rpw = rpw < 1 ? 1 : (rpw > 32 ? 32 : rpw);
    a.rows_per_warp = (int)rpw;
    dim3 grid(gx, (unsigned)((nrows + 4 * rpw - 1) / (4 * rpw)));
    LaunchScope ls(c, K_FLUX_X);
    // Measured: the TMA rows win up to 256^3 (0.64 vs 0.69 ms), but at 512^3 their 36-column boxes for 31 faces cost
    // 23 GB instead of 18 GB of DRAM traffic per launch and lose (5.6 vs 4.9 ms under ncu): long rows use the shuffle kernel.
    if (MHD && c->use_tma && g.nx <= 384) {
      FluxXTArgs ta;
      ta.fV0 = c->vcur ? 11 : 0;
      ta.fB = (int)((Bf[0] - c->field(F_BA)) / g.np);
      for (int n = 0; n < 5; ++n) ta.FH[n] = a.FH[n];
      ta.FB[0] = a.FB[0];
      ta.FB[1] = a.FB[1];
      ta.cf = a.cf;
      ta.sg = a.sg;
      const long long per_chunk = (long long)gx * ((g.ny + 3) / 4);
      long long nch = (148 * 16 + per_chunk - 1) / per_chunk;
      const long long maxch = g.nz / 8 > 0 ? g.nz / 8 : 1;
      nch = nch < 1 ? 1 : (nch > maxch ? maxch : nch);
      ta.chunk = (int)((g.nz + nch - 1) / nch);
      dim3 tgrid(gx, (g.ny + 3) / 4, (unsigned)((g.nz + ta.chunk - 1) / ta.chunk));
      launch_x_tma<SOLVER, LIM, MHD>(c, tgrid, ta);
    } else {
      k_flux_x<SOLVER, LIM, MHD><<<grid, 128, 0, c->stream>>>(g, a);
    }
  }
  for (int d = 1; d < 3; ++d) {  // y then z: marching pencils
    const int ib = (d + 1) % 3, ie = (d + 2) % 3;
    FluxMArgs a;
    a.q[0] = c->vfield(0);
    a.q[1] = c->vfield(1 + d);
    a.q[2] = c->vfield(1 + ib);
    a.q[3] = c->vfield(1 + ie);
    a.q[4] = c->vfield(4);
    a.q[5] = c->vfield(5 + ib);
    a.q[6] = c->vfield(5 + ie);
    a.bn = MHD ? Bf[d] : nullptr;
    a.sd = d == 1 ? g.sy : g.sz;
    a.st = d == 1 ? g.sz : g.sy;
    a.ns = d == 1 ? g.ny : g.nz;
    a.nt = d == 1 ? g.nz : g.ny;
    for (int n = 0; n < 5; ++n) {
      a.FX[n] = c->field(F_FX + n);
      a.R[n] = c->field(F_R + n);
    }
    a.cfx = c->field(F_CFX);
    a.csum = c->field(F_CS);
    a.FB[0] = c->field(F_FB + 2 * d);
    a.FB[1] = c->field(F_FB + 2 * d + 1);
    a.SG = c->sgn(d);
    a.sc = c->sc;
    const long long per_chunk = (long long)((g.nx + 31) / 32) * ((a.nt + 3) / 4);
    long long nch = (148 * 16 + per_chunk - 1) / per_chunk;
    const long long maxch = a.ns / 8 > 0 ? a.ns / 8 : 1;
    nch = nch < 1 ? 1 : (nch > maxch ? maxch : nch);
    a.chunk = (int)((a.ns + nch - 1) / nch);
    dim3 grid((g.nx + 31) / 32, (a.nt + 3) / 4, (unsigned)((a.ns + a.chunk - 1) / a.chunk));
    LaunchScope ls(c, K_FLUX_X + d);
    if (MHD && c->use_tma) {
      FluxTArgs ta;
      ta.fV0 = c->vcur ? 11 : 0;
      ta.fB = (int)((Bf[d] - c->field(F_BA)) / g.np);
      ta.ns = a.ns; ta.nt = a.nt; ta.chunk = a.chunk; ta.sd = a.sd; ta.st = a.st;
      for (int n = 0; n < 5; ++n) { ta.FX[n] = a.FX[n]; ta.R[n] = a.R[n]; }
      ta.cfx = a.cfx; ta.csum = a.csum; ta.FB[0] = a.FB[0]; ta.FB[1] = a.FB[1]; ta.SG = a.SG; ta.sc = a.sc;
      for (int n = 0; n < 5; ++n) {
        ta.Uin[n] = c->field(ap.uin + n);
        ta.U0[n] = c->field(F_UA + n);
        ta.Uout[n] = c->field(ap.uout + n);
      }
      ta.w = ap.w;
      ta.w0 = ap.w0;
      launch_march_tma<SOLVER, LIM, MHD>(c, d, grid, ta, want_dt, uct, ap.on && d == 2);
      continue;
    }
    if (d == 1) {
      if (want_dt) k_flux_march<SOLVER, LIM, MHD, 1, true, true><<<grid, 128, 0, c->stream>>>(g, a);
      else if (uct) k_flux_march<SOLVER, LIM, MHD, 1, false, true><<<grid, 128, 0, c->stream>>>(g, a);
      else k_flux_march<SOLVER, LIM, MHD, 1, false, false><<<grid, 128, 0, c->stream>>>(g, a);
    } else {
      if (want_dt) k_flux_march<SOLVER, LIM, MHD, 2, true, true><<<grid, 128, 0, c->stream>>>(g, a);
      else if (uct) k_flux_march<SOLVER, LIM, MHD, 2, false, true><<<grid, 128, 0, c->stream>>>(g, a);
      else k_flux_march<SOLVER, LIM, MHD, 2, false, false><<<grid, 128, 0, c->stream>>>(g, a);
    }
  }
}

template <int SOLVER, int LIM>
HdKernel hd_kernel_sl(bool first) {
  return first ? (HdKernel)k_hd_stage<SOLVER, LIM, true> : (HdKernel)k_hd_stage<SOLVER, LIM, false>;
}

template <int SOLVER, int LIM>
MhdKernel mhd_kernel_sl(bool first, int emf_mode) {
  switch (emf_mode) {
    case EMF_UCT: return first ? (MhdKernel)k_mhd_stage<SOLVER, LIM, EMF_UCT, true> : (MhdKernel)k_mhd_stage<SOLVER, LIM, EMF_UCT, false>;
    case EMF_UCT0: return first ? (MhdKernel)k_mhd_stage<SOLVER, LIM, EMF_UCT0, true> : (MhdKernel)k_mhd_stage<SOLVER, LIM, EMF_UCT0, false>;
    default: return first ? (MhdKernel)k_mhd_stage<SOLVER, LIM, EMF_ARITH, true> : (MhdKernel)k_mhd_stage<SOLVER, LIM, EMF_ARITH, false>;
  }
}

// MHD: every solver but HLLC; hydrodynamics: every solver but HLLD (idfx_create refuses the other combinations)
#if IDFX_INST_SOLVER != 1
template void launch_sweeps_t<IDFX_INST_SOLVER, IDFX_INST_LIM, true>(idfx_ctx*, const double* const[3], bool, const ApplyInfo&);
template MhdKernel mhd_kernel_sl<IDFX_INST_SOLVER, IDFX_INST_LIM>(bool, int);
#endif
#if IDFX_INST_SOLVER != 2
template void launch_sweeps_t<IDFX_INST_SOLVER, IDFX_INST_LIM, false>(idfx_ctx*, const double* const[3], bool, const ApplyInfo&);
template HdKernel hd_kernel_sl<IDFX_INST_SOLVER, IDFX_INST_LIM>(bool);
#endif

}  // namespace idfx
