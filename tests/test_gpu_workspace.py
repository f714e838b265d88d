"""The workspace contract of include/idfx.h: every access of every kernel stays inside the idfx_workspace_bytes(ctx) bytes
handed to idfx_bind.  The number of fields depends on what the context needs (hydrodynamics keeps no face field, only PPM
keeps -(v x Bc), the face fluxes of B and the sign bytes in memory; the vector-potential form, the 2D EMFs and PPM add their
own groups), so each layout is run between two canary regions: the workspace is a window in the middle of a larger
allocation filled with a byte pattern, and after set_state, three cycles, compute_dt and get_state both sides must still
hold the pattern.  (Accesses that stray INSIDE the workspace, into another field, change results and are caught by the
parity tests.)"""
import os
import sys

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2304_13746_b200 import idfx as I  # noqa: E402
from paper_2304_13746_b200 import inputs  # noqa: E402

pytestmark = pytest.mark.gpu

GUARD = 8 << 20   # bytes on each side: 35 padded fields of the 24 x 22 x 20 box
PATTERN = 0xA5

LAYOUTS = [
    # tag, mhd, solver, limiter, emf, keywords, fields the workspace holds
    ("hd", False, I.SOLVER_HLLC, I.LIMITER_VANLEER, I.EMF_NONE, {}, 25),
    ("hd-rk3-outflow", False, I.SOLVER_HLL, I.LIMITER_LIMO3, I.EMF_NONE, dict(nstages=3, boundary=I.BOUNDARY_OUTFLOW), 25),
    ("hd-ppm", False, I.SOLVER_ROE, I.LIMITER_PPM, I.EMF_NONE, {}, 25 + 7 + 18),
    ("mhd", True, I.SOLVER_HLLD, I.LIMITER_VANLEER, I.EMF_UCT_CONTACT, {}, 43),
    ("mhd-rk3", True, I.SOLVER_ROE, I.LIMITER_MINMOD, I.EMF_ARITHMETIC, dict(nstages=3), 43),
    ("mhd-outflow", True, I.SOLVER_HLLD, I.LIMITER_VANLEER, I.EMF_UCT_CONTACT, dict(boundary=I.BOUNDARY_OUTFLOW), 43),
    ("mhd-floor", True, I.SOLVER_HLLD, I.LIMITER_VANLEER, I.EMF_UCT_0, dict(pressure_floor=1e-3), 43),
    ("mhd-potential", True, I.SOLVER_HLLD, I.LIMITER_VANLEER, I.EMF_UCT_CONTACT, dict(ct_form=I.CT_POTENTIAL), 43 + 12),
    ("mhd-hll2d", True, I.SOLVER_HLL, I.LIMITER_VANLEER, I.EMF_UCT_HLL, {}, 43 + 15),
    ("mhd-hlld2d", True, I.SOLVER_HLLD, I.LIMITER_LIMO3, I.EMF_UCT_HLLD, {}, 43 + 18),
    ("mhd-ppm", True, I.SOLVER_HLLD, I.LIMITER_PPM, I.EMF_UCT_CONTACT, {}, 53 + 18),
    ("mhd-ppm-rk3", True, I.SOLVER_HLL, I.LIMITER_PPM, I.EMF_UCT_0, dict(nstages=3), 53 + 18),
]


def state(shape, mhd):
    nx, ny, nz = shape
    n = max(shape)
    prim, b = inputs.turbulence_mhd(n, 3, 2, 0.3, 4.0) if mhd else inputs.turbulence_hd(n, 3, 2, 0.3)
    # a box with three different extents cut out of the periodic cube: not periodic itself, which only makes the flow
    # rougher; the face field stays divergence-free cell by cell
    prim = prim[:, :nz, :ny, :nx].contiguous()
    return prim, (b[:, :nz, :ny, :nx].contiguous() if mhd else None)


@pytest.mark.parametrize("tag,mhd,solver,lim,emf,kw,nfields", LAYOUTS, ids=[l[0] for l in LAYOUTS])
def test_no_access_outside_the_workspace(tag, mhd, solver, lim, emf, kw, nfields):
    shape = (24, 22, 20)
    nx, ny, nz = shape
    sim = I.Idfx(nx, ny, nz, 1.0 / nx, 5.0 / 3.0, solver, lim, emf, **kw)
    nbytes = sim.L.idfx_workspace_bytes(sim.h)
    pitch = (nx + 18 + 15) // 16 * 16                      # active cells start at column 16
    npad = (pitch * (ny + 4) * (nz + 4) + 31) // 32 * 32   # doubles per field, a multiple of 256 bytes
    assert nbytes == nfields * npad * 8 + 256, "the layout this test (and DESIGN.md section 6) states"
    big = torch.full((GUARD + nbytes + GUARD,), PATTERN, dtype=torch.uint8, device="cuda:0")
    assert big.data_ptr() % 256 == 0
    torch.cuda.synchronize()
    I._check(sim.L.idfx_bind(sim.h, big.data_ptr() + GUARD, nbytes, sim.stream.cuda_stream))
    sim.workspace = big          # keeps the allocation alive for the context
    prim, b = state(shape, mhd)
    sim.set_state(prim.cuda(), b.cuda() if mhd else None)
    sim.advance(3, 0.3)
    dt = sim.compute_dt(0.3)
    out = sim.get_state()
    sim.get_conserved()
    if kw.get("ct_form"):
        sim.get_potential()
    torch.cuda.synchronize()
    assert sim.status() == 0 and dt > 0.0 and bool(torch.isfinite(out[0]).all())
    assert bool((big[:GUARD] == PATTERN).all()), "a kernel wrote below the workspace"
    assert bool((big[GUARD + nbytes:] == PATTERN).all()), "a kernel wrote beyond the workspace"
    sim.close()
