"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

* configs 2, 3, 4 (128^3 x 50, 128^3 x 50, 256^3 x 20): the whole run on the GPU against sampled outputs and the
  complete dt history of the CPU oracle, stored by tests/golden/make_config_goldens.py (calls only oracle/).
* config 5 (512^3): the oracle cannot run the box in a test, but the scheme is local, so it can compute sampled
  outputs one by one: a 32^3 window cut out of the GPU state before a cycle, advanced by the oracle as a small
  periodic box with the same dt, agrees with the full computation on every cell further than 10 cells from the
  window boundary (domain of dependence of one RK2 cycle: <= 8 cells).  dt at full size is checked through the
  per-cell signal-speed sums the oracle computes on windows around the fastest cells.  Checked cycles: the first two,
  the eleventh and the twenty-second (the last one bench.py times: 2-3 warm-up + 20); windows sit on the corners of the
  periodic box, on the seams of the 31 x 11 tiles and z chunks of k_mhd_stage and of the 32 x 4 x 8 tiles of k_ct_update,
  and at random places.
"""
import os

import numpy as np
import pytest
import torch

from paper_2304_13746_b200 import inputs

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(__file__), "golden")
TOL, TOL_DT = 1e-10, 1e-12


@pytest.fixture(scope="module")
def idfx():
    from paper_2304_13746_b200 import idfx as m
    assert torch.cuda.is_available()
    m.lib()
    return m


@pytest.mark.parametrize("name", ["config2", "config3", "config4"])
def test_full_config_against_oracle_samples(idfx, name):
    path = os.path.join(GOLD, "config_samples_%s.npz" % name)
    if not os.path.exists(path):
        pytest.skip("golden samples for %s not generated (tests/golden/make_config_goldens.py)" % name)
    gold = np.load(path)
    # the SAME arrays the goldens were computed from: synthesised on the CPU (as make_config_goldens.py does), then copied
    prim, b, cfg = inputs.make(name)
    prim, b = prim.cuda(), (None if b is None else b.cuda())
    n = cfg["n"]
    assert n == int(gold["n"]) and cfg["steps"] == int(gold["steps"])
    sim = idfx.Idfx(n, n, n, cfg["dx"], cfg["gamma"], cfg["solver"], cfg["limiter"], cfg["emf"])
    sim.set_state(prim, b)
    for s in range(cfg["steps"]):
        sim.advance(1, cfg["cfl"])
        dt = sim.last_dt()
        assert abs(dt - gold["dts"][s]) <= TOL_DT * gold["dts"][s], "dt of cycle %d" % s
    assert sim.status() == 0
    cons, bf = sim.get_conserved()
    idx = torch.from_numpy(gold["idx"]).cuda()
    got = cons.reshape(5, -1)[:, idx].cpu().numpy()
    worst = 0.0
    for v in range(5):
        err = np.abs(got[v] - gold["cons"][v]).max() / gold["cons_max"][v]
        worst = max(worst, err)
        assert err <= TOL, "%s cons[%d]: %.3e" % (name, v, err)
        ssum = float(cons[v].sum())
        assert abs(ssum - gold["cons_sum"][v]) <= 1e-11 * max(abs(gold["cons_sum"][v]), float(cons[v].abs().sum()))
    if bf is not None:
        gotb = bf.reshape(3, -1)[:, idx].cpu().numpy()
        err = np.abs(gotb - gold["bface"]).max() / float(gold["bface_max"])
        assert err <= TOL, "%s bface: %.3e" % (name, err)
        div = (torch.roll(bf[0], -1, 2) - bf[0]) + (torch.roll(bf[1], -1, 1) - bf[1]) + (torch.roll(bf[2], -1, 0) - bf[2])
        assert float(div.abs().max() / bf.abs().max()) <= 1e-13
        worst = max(worst, err)
    print("%s full size: worst relative error at %d oracle sample points %.3e" % (name, len(gold["idx"]), worst))


def cut(t, origin, w):
    """Periodic w^3 window of a [var][nz][ny][nx] device tensor with lower corner origin = (ox, oy, oz)."""
    n = t.shape[-1]
    ix = (origin[0] + torch.arange(w, device=t.device)) % n
    iy = (origin[1] + torch.arange(w, device=t.device)) % n
    iz = (origin[2] + torch.arange(w, device=t.device)) % n
    return t[:, iz[:, None, None], iy[None, :, None], ix[None, None, :]].contiguous()


def test_config5_512_windows_against_oracle(idfx, R):
    name, W, M = "config5", 32, 10
    prim, b, cfg = inputs.make(name, device="cuda")
    n, dx, cfl = cfg["n"], cfg["dx"], cfg["cfl"]
    assert n == 512
    sim = idfx.Idfx(n, n, n, dx, cfg["gamma"], cfg["solver"], cfg["limiter"], cfg["emf"])
    sim.set_state(prim, b)
    del prim, b
    c_start, b_start = sim.get_conserved()
    sums0 = [float(c_start[v].sum()) for v in range(5)] + [float(b_start[d].sum()) for d in range(3)]
    abs0 = [float(c_start[v].abs().sum()) for v in range(5)] + [float(b_start[d].abs().sum()) for d in range(3)]
    del c_start, b_start
    rng = np.random.default_rng(5)
    origins = [(0, 0, 0), (n - 16, n - 16, n - 16), (n - 20, 3, 250), (100, n - 12, n - 30)]
    # seams of the launch configuration at 512^3: x tiles start at 31 m (the last, partial one at 496), y tiles at 11 m
    # (last at 506), z chunks of 103 planes (5 chunks); k_ct_update tiles at multiples of (32, 4, 8)
    origins += [(31 * 5 - 16, 11 * 9 - 16, 103 - 16), (496 - 16, 506 - 16, 412 - 16), (31 * 11 - 16, 11 * 30 - 16, 309 - 16),
                (32 * 7 - 16, 4 * 50 - 16, 8 * 33 - 16)]
    origins += [tuple(int(x) for x in rng.integers(0, n, 3)) for _ in range(6)]
    worst = 0.0
    done = 0
    for cycle in (0, 1, 10, 21):
        sim.advance(cycle - done, cfl)
        done = cycle + 1
        p0, b0 = sim.get_state()
        # ---- dt at full size: windows around the cells with the largest cell-centred estimate ----
        rho, pr = p0[0], p0[4]
        bc = torch.stack([0.5 * (b0[d] + torch.roll(b0[d], -1, 2 - d)) for d in range(3)])
        a2, b2 = cfg["gamma"] * pr / rho, (bc * bc).sum(0) / rho
        est = torch.zeros_like(rho)
        for d in range(3):
            cf = torch.sqrt(0.5 * (a2 + b2 + torch.sqrt(torch.clamp((a2 + b2) ** 2 - 4 * a2 * bc[d] ** 2 / rho, min=0))))
            est += p0[1 + d].abs() + cf
        del bc, a2, b2, cf
        top = torch.topk(est.flatten(), 4096).indices.cpu().numpy()
        del est
        hot = []
        for f in top:
            kz, jy, ix = np.unravel_index(int(f), (n, n, n))
            o = (int(ix) - W // 2, int(jy) - W // 2, int(kz) - W // 2)
            if all(max(abs(o[0] - h[0]), abs(o[1] - h[1]), abs(o[2] - h[2])) > 6 for h in hot):
                hot.append(o)
            if len(hot) == 6:
                break
        dt_gpu = sim.compute_dt(cfl)
        smax = 0.0
        for o in hot:
            ref = R.Oracle(W, W, W, dx, cfg["gamma"], cfg["solver"], cfg["limiter"], cfg["emf"])
            ref.set_state(cut(p0, o, W).cpu().numpy(), cut(b0, o, W).cpu().numpy())
            ref.compute_dt(cfl)
            s = np.zeros((W, W, W))
            for d in range(3):
                cface = ref.get_flux(d)[1]
                s += np.maximum(cface, np.roll(cface, -1, 2 - d))       # G8: larger of the cell's two faces
            smax = max(smax, float(s[M:W - M, M:W - M, M:W - M].max()) / dx)
        assert abs(cfl / smax - dt_gpu) <= TOL_DT * dt_gpu, (cfl / smax, dt_gpu)
        # ---- one cycle on the GPU, the same cycle on every window by the oracle ----
        sim.advance(1, cfl)
        assert abs(sim.last_dt() - dt_gpu) <= 1e-14 * dt_gpu
        c1, b1 = sim.get_conserved()
        scale_c = [float(c1[v].abs().max()) for v in range(5)]
        scale_b = float(b1.abs().max())
        for o in origins:
            ref = R.Oracle(W, W, W, dx, cfg["gamma"], cfg["solver"], cfg["limiter"], cfg["emf"])
            ref.set_state(cut(p0, o, W).cpu().numpy(), cut(b0, o, W).cpu().numpy())
            ref.step(dt_gpu)
            rc, rb = ref.get_conserved()
            gc, gb = cut(c1, o, W).cpu().numpy(), cut(b1, o, W).cpu().numpy()
            sl = (slice(None), slice(M, W - M), slice(M, W - M), slice(M, W - M))
            for v in range(5):
                err = np.abs(gc[sl][v] - rc[sl][v]).max() / scale_c[v]
                worst = max(worst, err)
                assert err <= TOL, ("cycle", cycle, "window", o, "cons", v, err)
            err = np.abs(gb[sl] - rb[sl]).max() / scale_b
            worst = max(worst, err)
            assert err <= TOL, ("cycle", cycle, "window", o, "bface", err)
        del p0, b0, c1, b1
    assert sim.status() == 0
    # properties that hold at any size, on the whole box after the 22 cycles: conservation on the periodic box and div B
    c_end, b_end = sim.get_conserved()
    sums1 = [float(c_end[v].sum()) for v in range(5)] + [float(b_end[d].sum()) for d in range(3)]
    for s0, s1, a0 in zip(sums0, sums1, abs0):
        assert abs(s1 - s0) <= 1e-11 * a0, (s0, s1, a0)     # 1.3e8 cells summed in fp64: ~1e-13 of the absolute sum per pass
    div = (torch.roll(b_end[0], -1, 2) - b_end[0]) + (torch.roll(b_end[1], -1, 1) - b_end[1]) + (torch.roll(b_end[2], -1, 0) - b_end[2])
    divb = float(div.abs().max() / b_end.abs().max())
    assert divb <= 1e-13, divb
    print("config5 512^3: worst relative window error %.3e; after 22 cycles max|div B| dx / max|B| = %.2e, conserved sums within 1e-11" % (worst, divb))


def test_config2_recipe_512_hd_windows_against_oracle(idfx, R):
    """Hydrodynamics at 512^3 (config 2 recipe, the size bench.py --workload config2 --n 512 and the Sedov workload run
    at) through the one-kernel stage, in the launch configuration used there: dt against the oracle on windows around the
    fastest cells, then one cycle on 10 windows (corners of the periodic box, tile and chunk seams, random places)."""
    name, W, M = "config2", 32, 10
    prim, _, cfg = inputs.make(name, n=512, device="cuda")
    n, dx, cfl = cfg["n"], cfg["dx"], cfg["cfl"]
    sim = idfx.Idfx(n, n, n, dx, cfg["gamma"], cfg["solver"], cfg["limiter"], cfg["emf"])
    sim.set_state(prim, None)
    del prim
    rng = np.random.default_rng(6)
    origins = [(0, 0, 0), (n - 16, n - 16, n - 16), (31 * 7 - 16, 7 * 30 - 16, 128 - 16), (n - 20, 3, 250)]
    origins += [tuple(int(x) for x in rng.integers(0, n, 3)) for _ in range(6)]
    worst = 0.0
    for cycle in range(2):
        p0, _ = sim.get_state()
        est = torch.sqrt(cfg["gamma"] * p0[4] / p0[0]) * 3 + p0[1].abs() + p0[2].abs() + p0[3].abs()
        top = torch.topk(est.flatten(), 4096).indices.cpu().numpy()
        del est
        hot = []
        for f in top:
            kz, jy, ix = np.unravel_index(int(f), (n, n, n))
            o = (int(ix) - W // 2, int(jy) - W // 2, int(kz) - W // 2)
            if all(max(abs(o[0] - h[0]), abs(o[1] - h[1]), abs(o[2] - h[2])) > 6 for h in hot):
                hot.append(o)
            if len(hot) == 6:
                break
        dt_gpu = sim.compute_dt(cfl)
        smax = 0.0
        for o in hot:
            ref = R.Oracle(W, W, W, dx, cfg["gamma"], cfg["solver"], cfg["limiter"], cfg["emf"])
            ref.set_state(cut(p0, o, W).cpu().numpy())
            ref.compute_dt(cfl)
            s = np.zeros((W, W, W))
            for d in range(3):
                cface = ref.get_flux(d)[1]
                s += np.maximum(cface, np.roll(cface, -1, 2 - d))
            smax = max(smax, float(s[M:W - M, M:W - M, M:W - M].max()) / dx)
        assert abs(cfl / smax - dt_gpu) <= TOL_DT * dt_gpu, (cfl / smax, dt_gpu)
        sim.advance(1, cfl)
        assert abs(sim.last_dt() - dt_gpu) <= 1e-14 * dt_gpu
        c1, _ = sim.get_conserved()
        scale_c = [float(c1[v].abs().max()) for v in range(5)]
        for o in origins:
            ref = R.Oracle(W, W, W, dx, cfg["gamma"], cfg["solver"], cfg["limiter"], cfg["emf"])
            ref.set_state(cut(p0, o, W).cpu().numpy())
            ref.step(dt_gpu)
            rc, _ = ref.get_conserved()
            gc = cut(c1, o, W).cpu().numpy()
            sl = (slice(None), slice(M, W - M), slice(M, W - M), slice(M, W - M))
            for v in range(5):
                err = np.abs(gc[sl][v] - rc[sl][v]).max() / scale_c[v]
                worst = max(worst, err)
                assert err <= TOL, ("cycle", cycle, "window", o, "cons", v, err)
    assert sim.status() == 0
    print("config2 recipe at 512^3 (HD, fused stage kernel): worst relative error on %d windows x 2 cycles %.3e" % (len(origins), worst))
