"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bar (BASELINE.json north_star): per field max|a-b| / max|b| <= 1e-10 on the conserved variables and the face
field after each configuration's step count; dt within 1e-12 relative (reading G15 for fields that cross zero).
"""
import math

import numpy as np
import pytest
import torch

from paper_2304_13746_b200 import inputs

pytestmark = pytest.mark.gpu

HLL, HLLC, HLLD, ROE, RUSANOV = 0, 1, 2, 3, 4
FLAT, MINMOD, VANLEER = 0, 1, 2
EMF_NONE, EMF_ARITH, EMF_UCT, EMF_UCT0 = 0, 1, 2, 3
TOL = 1e-10
TOL_DT = 1e-12


@pytest.fixture(scope="module")
def idfx():
    from paper_2304_13746_b200 import idfx as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.lib()
    return m


def rel_err(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def assert_state_close(sim, ref, tol=TOL, what=""):
    cons, bf = sim.get_conserved()
    rc, rb = ref.get_conserved()
    cons = cons.cpu().numpy()
    names = ["rho", "mx", "my", "mz", "E"]
    for v in range(5):
        e = rel_err(cons[v], rc[v])
        assert e <= tol, "%s %s: rel err %.3e" % (what, names[v], e)
    if rb is not None:
        bf = bf.cpu().numpy()
        for d in range(3):
            scale = max(np.abs(rb).max(), 1e-300)          # a component may vanish identically
            e = float(np.abs(bf[d] - rb[d]).max() / scale)
            assert e <= tol, "%s B%s: rel err %.3e" % (what, "xyz"[d], e)


def smooth_ic(nx, ny, nz, seed, mhd=True):
    """Smooth periodic fields on a ragged box (test-local)."""
    rng = np.random.default_rng(seed)
    dx = 1.0 / max(nx, ny, nz)
    cx, cy, cz = (np.arange(nx) + 0.5) / nx, (np.arange(ny) + 0.5) / ny, (np.arange(nz) + 0.5) / nz
    ex, ey, ez = np.arange(nx) / nx, np.arange(ny) / ny, np.arange(nz) / nz

    def wave(z, y, x):
        Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
        k = rng.integers(1, 3, size=3)
        return np.sin(2 * np.pi * (k[0] * X + k[1] * Y + k[2] * Z) + rng.uniform(0, 2 * np.pi))
    prim = np.empty((5, nz, ny, nx))
    prim[0] = 1.0 + 0.3 * wave(cz, cy, cx)
    for d in range(3):
        prim[1 + d] = 0.6 * wave(cz, cy, cx) + 0.3 * wave(cz, cy, cx)
    prim[4] = 1.0 + 0.3 * wave(cz, cy, cx)
    if not mhd:
        return prim, None, dx
    ax, ay, az = 0.05 * wave(ez, ey, cx), 0.05 * wave(ez, cy, ex), 0.05 * wave(cz, ey, ex)
    up = lambda a, d: np.roll(a, -1, d)
    b = np.stack([((up(az, 1) - az) - (up(ay, 0) - ay)) / dx,
                  ((up(ax, 0) - ax) - (up(az, 2) - az)) / dx,
                  ((up(ay, 2) - ay) - (up(ax, 1) - ax)) / dx])
    b[0] += 0.4
    b[1] -= 0.3
    b[2] += 0.2
    return prim, b, dx


def make_pair(idfx, R, nx, ny, nz, dx, gamma, solver, limiter, emf, prim, b):
    sim = idfx.Idfx(nx, ny, nz, dx, gamma, solver, limiter, emf)
    sim.set_state(torch.from_numpy(prim).cuda(), None if b is None else torch.from_numpy(b).cuda())
    ref = R.Oracle(nx, ny, nz, dx, gamma, solver, limiter, emf)
    ref.set_state(prim, b)
    return sim, ref


COMBOS = [
    (HLL, FLAT, EMF_NONE), (HLL, VANLEER, EMF_NONE), (HLLC, MINMOD, EMF_NONE), (HLLC, VANLEER, EMF_NONE),
    (ROE, VANLEER, EMF_NONE), (ROE, MINMOD, EMF_NONE),
    (HLL, VANLEER, EMF_ARITH), (HLL, MINMOD, EMF_UCT), (HLLD, VANLEER, EMF_ARITH), (HLLD, VANLEER, EMF_UCT),
    (HLLD, MINMOD, EMF_UCT), (HLLD, FLAT, EMF_ARITH), (ROE, VANLEER, EMF_ARITH), (ROE, VANLEER, EMF_UCT),
    (ROE, MINMOD, EMF_ARITH), (RUSANOV, VANLEER, EMF_NONE), (RUSANOV, VANLEER, EMF_UCT), (RUSANOV, MINMOD, EMF_ARITH),
    (HLLD, VANLEER, EMF_UCT0), (ROE, MINMOD, EMF_UCT0),
]


@pytest.mark.parametrize("solver,limiter,emf", COMBOS)
def test_every_scheme_combination_ragged_box(idfx, R, solver, limiter, emf):
    """Element-by-element parity after every step on a ragged box (spans several thread blocks, every
    dimension different, none a multiple of the tile sizes)."""
    nx, ny, nz = 37, 21, 13
    prim, b, dx = smooth_ic(nx, ny, nz, 11, emf != EMF_NONE)
    sim, ref = make_pair(idfx, R, nx, ny, nz, dx, 5.0 / 3.0, solver, limiter, emf, prim, b)
    assert_state_close(sim, ref, 1e-14, "after set_state")
    for s in range(4):
        dt_g, dt_r = sim.compute_dt(0.4), ref.compute_dt(0.4)
        assert abs(dt_g - dt_r) <= TOL_DT * dt_r
        sim.advance(1, 0.4)
        ref.advance(1, 0.4)
        assert abs(sim.last_dt() - ref.last_dt()) <= TOL_DT * ref.last_dt()
        assert_state_close(sim, ref, TOL, "step %d" % s)
    assert sim.status() == 0 and ref.status() == 0
    assert ref.roe_fallbacks() == 0


# Thin boxes that are long in ONE direction: the whole oracle runs on them in a second, and the long direction crosses
# every kind of seam of the launch configuration used at 512^3 -- the 31-cell x tiles of the one-kernel stages (nx = 385 =
# 12 x 31 + 13 and nx = 400 end in a partial tile, nx = 512 is the headline row length), their 11-row (MHD) / 7-row (HD) y
# tiles, their z chunks (nz = 100: several chunks of >= 16 planes per CTA) and the 32 x 4 x 8 tiles of k_ct_update.
THIN_BOXES = [(400, 12, 10), (385, 12, 10), (512, 12, 10), (10, 130, 12), (12, 10, 100), (70, 30, 40)]
THIN_SCHEMES = [(HLLD, VANLEER, EMF_UCT), (ROE, VANLEER, EMF_UCT), (HLL, VANLEER, EMF_UCT), (HLLD, MINMOD, EMF_ARITH),
                (HLLC, VANLEER, EMF_NONE)]


@pytest.mark.parametrize("solver,limiter,emf", THIN_SCHEMES)
@pytest.mark.parametrize("shape", THIN_BOXES)
def test_tile_and_chunk_seams_on_thin_boxes(idfx, R, shape, solver, limiter, emf):
    nx, ny, nz = shape
    prim, b, dx = smooth_ic(nx, ny, nz, 23, emf != EMF_NONE)
    if b is not None:
        # smooth_ic differentiates its potential with dx = 1 / (longest side): across the short sides of a thin box the
        # field would be (longest / shortest) times stronger (beta << 1); scale the varying part back
        mean = np.array([0.4, -0.3, 0.2]).reshape(3, 1, 1, 1)
        b = mean + (b - mean) * (min(shape) / max(shape))
    sim, ref = make_pair(idfx, R, nx, ny, nz, dx, 5.0 / 3.0, solver, limiter, emf, prim, b)
    for s in range(4):
        sim.advance(1, 0.4)
        ref.advance(1, 0.4)
        assert abs(sim.last_dt() - ref.last_dt()) <= TOL_DT * ref.last_dt(), "dt of cycle %d" % s
        assert_state_close(sim, ref, TOL, "%dx%dx%d cycle %d" % (nx, ny, nz, s))
    assert sim.status() == 0 and ref.status() == 0
    assert float(sim.get_state()[0][4].min()) > 0.2   # a well-behaved flow: the comparison is not of two blow-ups


def run_config(idfx, R, name, n=None, steps=None):
    prim, b, cfg = inputs.make(name, n=n)
    N = cfg["n"]
    steps = steps or cfg["steps"]
    sim, ref = make_pair(idfx, R, N, N, N, cfg["dx"], cfg["gamma"], cfg["solver"], cfg["limiter"], cfg["emf"],
                         prim.numpy(), None if b is None else b.numpy())
    sim.advance(steps, cfg["cfl"])
    ref.advance(steps, cfg["cfl"])
    assert sim.status() == 0 and ref.status() == 0
    assert abs(sim.last_dt() - ref.last_dt()) <= TOL_DT * ref.last_dt()
    assert_state_close(sim, ref, TOL, name)
    cons, bf = sim.get_conserved()
    rc, rb = ref.get_conserved()
    worst = max(rel_err(cons[v].cpu().numpy(), rc[v]) for v in range(5))
    if rb is not None:
        worst = max(worst, float(np.abs(bf.cpu().numpy() - rb).max() / np.abs(rb).max()))
    print("%s n=%d steps=%d: worst relative error %.3e, dt rel diff %.1e" % (
        name, N, steps, worst, abs(sim.last_dt() - ref.last_dt()) / ref.last_dt()))
    return sim, ref


def test_config1_full(idfx, R):
    """BASELINE config 1 as specified: 32^3 MHD, van Leer + HLLD + arithmetic CT + RK2, CFL 0.3, 10 steps."""
    sim, ref = run_config(idfx, R, "config1")
    _, bf = sim.get_conserved()
    bf = bf.cpu().numpy()
    div = (np.roll(bf[0], -1, 2) - bf[0]) + (np.roll(bf[1], -1, 1) - bf[1]) + (np.roll(bf[2], -1, 0) - bf[2])
    assert np.abs(div).max() / np.abs(bf).max() <= 1e-13


@pytest.mark.parametrize("name,n,steps", [("config2", 48, 6), ("config3", 48, 6), ("config4", 40, 4), ("config5", 48, 4)])
def test_configs_reduced_size(idfx, R, name, n, steps):
    """The recipes of BASELINE configs 2-5 at a size the oracle finishes in seconds (same scheme, CFL, input
    recipe).  Full sizes: test_gpu_fullsize.py."""
    run_config(idfx, R, name, n=n, steps=steps)


def test_step_with_given_dt_equals_advance(idfx, R):
    nx, ny, nz = 24, 20, 16
    prim, b, dx = smooth_ic(nx, ny, nz, 3)
    sim, ref = make_pair(idfx, R, nx, ny, nz, dx, 5.0 / 3.0, HLLD, VANLEER, EMF_UCT, prim, b)
    dt = sim.compute_dt(0.3)
    sim.step(dt)
    assert sim.last_dt() == dt
    ref.step(dt)
    assert_state_close(sim, ref, TOL)
    sim2 = idfx.Idfx(nx, ny, nz, dx, 5.0 / 3.0, HLLD, VANLEER, EMF_UCT)
    sim2.set_state(torch.from_numpy(prim).cuda(), torch.from_numpy(b).cuda())
    sim2.advance(1, 0.3)
    assert abs(sim2.last_dt() - dt) <= 1e-14 * dt
    c1, b1 = sim.get_conserved()
    c2, b2 = sim2.get_conserved()
    assert float((c1 - c2).abs().max()) <= 1e-13 and float((b1 - b2).abs().max()) <= 1e-13


def test_state_roundtrip_and_host_variants(idfx):
    nx, ny, nz = 19, 8, 11
    prim, b, dx = smooth_ic(nx, ny, nz, 5)
    tp, tb = torch.from_numpy(prim), torch.from_numpy(b)
    sim = idfx.Idfx(nx, ny, nz, dx, 1.4, HLLD, VANLEER, EMF_ARITH)
    sim.set_state(tp.cuda(), tb.cuda())
    p1, b1 = sim.get_state()
    assert torch.equal(b1.cpu(), tb)                                  # face field bit-exact
    assert float((p1.cpu() - tp).abs().max()) <= 4e-15                # prims to a few ulp
    sim_h = idfx.Idfx(nx, ny, nz, dx, 1.4, HLLD, VANLEER, EMF_ARITH)
    sim_h.set_state(tp.pin_memory(), tb.pin_memory())                 # host buffers through the C ABI
    sim.advance(2, 0.4)
    sim_h.advance(2, 0.4)
    ph, bh = sim_h.get_state(host=True)
    pd, bd = sim.get_state()
    assert torch.equal(ph, pd.cpu()) and torch.equal(bh, bd.cpu())
    assert sim.launch_count() > 0


def test_uniform_state_and_conservation_on_device(idfx):
    n = 16
    prim = np.empty((5, n, n, n))
    for v, val in enumerate((1.3, 0.4, -0.7, 0.2, 0.8)):
        prim[v] = val
    b = np.empty((3, n, n, n))
    for d, val in enumerate((0.5, -0.3, 0.9)):
        b[d] = val
    sim = idfx.Idfx(n, n, n, 1.0 / n, 5.0 / 3.0, HLLD, VANLEER, EMF_UCT)
    sim.set_state(torch.from_numpy(prim).cuda(), torch.from_numpy(b).cuda())
    c0, _ = sim.get_conserved()
    sim.advance(3, 0.5)
    c1, b1 = sim.get_conserved()
    for v in range(5):
        assert bool((c1[v] == c1[v].flatten()[0]).all())
        assert abs(float(c1[v].flatten()[0] - c0[v].flatten()[0])) <= 1e-14 * max(1.0, abs(float(c0[v].flatten()[0])))
    assert torch.equal(b1.cpu(), torch.from_numpy(b))
    # conservation and div B on smooth data
    prim, b, dx = smooth_ic(24, 24, 24, 9)
    sim = idfx.Idfx(24, 24, 24, dx, 5.0 / 3.0, ROE, VANLEER, EMF_UCT)
    sim.set_state(torch.from_numpy(prim).cuda(), torch.from_numpy(b).cuda())
    c0, b0 = sim.get_conserved()
    sim.advance(8, 0.4)
    c1, b1 = sim.get_conserved()
    for v in range(5):
        assert abs(float(c1[v].sum() - c0[v].sum())) <= 1e-13 * max(float(c0[v].abs().sum()), 1.0)
    for d in range(3):
        assert abs(float(b1[d].sum() - b0[d].sum())) <= 1e-13 * float(b0[d].abs().sum()) + 1e-13
    div = (torch.roll(b1[0], -1, 2) - b1[0]) + (torch.roll(b1[1], -1, 1) - b1[1]) + (torch.roll(b1[2], -1, 0) - b1[2])
    assert float(div.abs().max() / b1.abs().max()) <= 1e-13


def test_error_codes_on_device(idfx):
    sim = idfx.Idfx(8, 8, 8, 0.125, 1.4, HLLC, MINMOD, EMF_NONE)
    with pytest.raises(idfx.IdfxError) as e:
        sim.compute_dt(1.2)
    assert e.value.code == idfx.ERR_INVALID_ARG
    with pytest.raises(idfx.IdfxError):
        sim.step(-1.0)
    with pytest.raises(idfx.IdfxError):
        sim.advance(-1, 0.3)
    prim = torch.ones((5, 8, 8, 8), dtype=torch.float64, device="cuda")
    prim[4, 2, 3, 4] = -1.0
    sim.set_state(prim)
    assert sim.status() == idfx.ERR_UNPHYSICAL                        # no floors (G13): sticky flag
    assert sim.status() == idfx.ERR_UNPHYSICAL


def test_minimum_size_box(idfx, R):
    """n = 4 per dimension is the smallest box the library accepts (ghost images overlap the whole box)."""
    prim, b, dx = smooth_ic(4, 5, 6, 21)
    sim, ref = make_pair(idfx, R, 4, 5, 6, dx, 5.0 / 3.0, HLLD, VANLEER, EMF_UCT, prim, b)
    sim.advance(3, 0.3)
    ref.advance(3, 0.3)
    assert_state_close(sim, ref, TOL)
    # hydrodynamics: the one-kernel stage with a box far smaller than its 31 x 7 tile and its 4-stage plane ring
    for shape in ((4, 4, 4), (6, 4, 5)):
        prim, _, dx = smooth_ic(*shape, 22, mhd=False)
        sim, ref = make_pair(idfx, R, *shape, dx, 5.0 / 3.0, HLLC, MINMOD, EMF_NONE, prim, None)
        sim.advance(3, 0.4)
        ref.advance(3, 0.4)
        assert abs(sim.last_dt() - ref.last_dt()) <= TOL_DT * ref.last_dt()
        assert_state_close(sim, ref, TOL, "HD %dx%dx%d" % shape)


def test_alternate_code_paths_in_a_subprocess(idfx):
    """IDFX_GRAPH=0 (no CUDA-graph replay: every cycle enqueued kernel by kernel) is read at idfx_bind; run one MHD and
    one HD parity case under it in a fresh process."""
    import os
    import subprocess
    import sys
    code = (
        "import sys, numpy as np, torch\n"
        "sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
        "from oracle import idfxref as R\n"
        "from paper_2304_13746_b200 import idfx\n"
        "import test_gpu_parity as T\n"
        "prim, b, dx = T.smooth_ic(37, 21, 13, 11)\n"
        "sim, ref = T.make_pair(idfx, R, 37, 21, 13, dx, 5.0 / 3.0, T.HLLD, T.VANLEER, T.EMF_UCT, prim, b)\n"
        "sim.advance(3, 0.4); ref.advance(3, 0.4)\n"
        "T.assert_state_close(sim, ref, T.TOL)\n"
        "assert abs(sim.last_dt() - ref.last_dt()) <= T.TOL_DT * ref.last_dt()\n"
        "print('ok')\n"
    ) % (os.path.dirname(os.path.dirname(os.path.abspath(__file__))), os.path.dirname(os.path.abspath(__file__)))
    for env_add in ({"IDFX_GRAPH": "0"},):
        p = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=300,
                           env=dict(os.environ, **env_add))
        assert p.returncode == 0 and "ok" in p.stdout, (env_add, p.stderr[-2000:])
    code_hd = code.replace("T.smooth_ic(37, 21, 13, 11)", "T.smooth_ic(37, 21, 13, 11, mhd=False)").replace(
        "T.HLLD, T.VANLEER, T.EMF_UCT", "T.HLLC, T.VANLEER, T.EMF_NONE")
    for env_add in ({"IDFX_GRAPH": "0"},):
        p = subprocess.run([sys.executable, "-c", code_hd], capture_output=True, text=True, timeout=300,
                           env=dict(os.environ, **env_add))
        assert p.returncode == 0 and "ok" in p.stdout, (env_add, p.stderr[-2000:])
