"""Host-side checks that need no GPU: the C-ABI library builds for sm_100a, loads, exports every symbol that
include/idfx.h declares, validates arguments and refuses to run unbound; the input generators are seeded,
solenoidal and have the statistics the recipes state."""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

from paper_2304_13746_b200 import idfx, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2304_13746_b200 import build
    build.build()
    return idfx.lib()


def test_exports_every_declared_symbol(L):
    inc = os.path.join(ROOT, "include")
    header = "".join(open(os.path.join(inc, f)).read() for f in sorted(os.listdir(inc)) if f.endswith(".h"))
    declared = set(re.findall(r"\b(idfx_[a-z0-9_]+)\s*\(", header))
    assert declared == set(idfx.SYMBOLS)
    raw = ctypes.CDLL(idfx.LIB_PATH)
    for s in declared:
        assert getattr(raw, s) is not None


def test_create_validates_arguments(L):
    ok = L.idfx_create(8, 8, 8, 0.1, 5.0 / 3.0, idfx.SOLVER_HLLD, idfx.LIMITER_VANLEER, idfx.EMF_UCT_CONTACT)
    assert ok
    assert L.idfx_workspace_bytes(ok) > 8 * 8 * 8 * 8 * 16
    L.idfx_destroy(ok)
    bad = [
        (3, 8, 8, 0.1, 1.4, 0, 2, 0),      # n < 4
        (8, 8, 8, 0.0, 1.4, 0, 2, 0),      # dx
        (8, 8, 8, 0.1, 1.0, 0, 2, 0),      # gamma
        (8, 8, 8, 0.1, 1.4, 7, 2, 0),      # solver enum
        (8, 8, 8, 0.1, 1.4, 5, 2, 0),      # solver enum, one past Rusanov
        (8, 8, 8, 0.1, 1.4, 0, 5, 0),      # limiter enum
        (8, 8, 8, 0.1, 1.4, 0, 2, 9),      # emf enum
        (8, 8, 8, 0.1, 1.4, 0, 2, 5),      # emf enum, one past the 2D-HLL scheme
        (8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLLC, 2, idfx.EMF_ARITHMETIC),   # HLLC is HD-only
        (8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLLD, 2, idfx.EMF_NONE),         # HLLD is MHD-only
    ]
    for args in bad:
        assert not L.idfx_create(*args)
        assert len(L.idfx_last_error()) > 0


def test_unbound_context_refuses_to_run(L):
    h = L.idfx_create(8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLL, idfx.LIMITER_MINMOD, idfx.EMF_NONE)
    dt = ctypes.c_double()
    assert L.idfx_step(h, 0.1) == idfx.ERR_NOT_BOUND
    assert L.idfx_advance(h, 1, 0.3) == idfx.ERR_NOT_BOUND
    assert L.idfx_compute_dt(h, 0.3, ctypes.byref(dt)) == idfx.ERR_NOT_BOUND
    assert L.idfx_status(h) == idfx.ERR_NOT_BOUND
    assert L.idfx_bind(h, None, 0, None) == idfx.ERR_INVALID_ARG
    assert L.idfx_launch_count(h) == 0
    L.idfx_destroy(h)
    assert L.idfx_step(None, 0.1) == idfx.ERR_INVALID_ARG


def test_options_are_validated_on_the_host(L):
    """idfx_set_option / idfx_set_option_real touch no device memory: every rule of include/idfx.h can be checked here."""
    hd = L.idfx_create(8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLL, idfx.LIMITER_LIMO3, idfx.EMF_NONE)
    mhd = L.idfx_create(8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLLD, idfx.LIMITER_VANLEER, idfx.EMF_UCT_HLL)
    assert hd and mhd
    for h in (hd, mhd):
        for stages in (1, 2, 3):
            assert L.idfx_set_option(h, idfx.OPT_INTEGRATOR, stages) == idfx.OK
        for bad in (0, 4, -1):
            assert L.idfx_set_option(h, idfx.OPT_INTEGRATOR, bad) == idfx.ERR_INVALID_ARG
        assert L.idfx_set_option(h, 99, 0) == idfx.ERR_INVALID_ARG
        assert L.idfx_set_option_real(h, idfx.OPT_PRESSURE_FLOOR, 1e-6) == idfx.OK
        assert L.idfx_set_option_real(h, idfx.OPT_PRESSURE_FLOOR, -1.0) == idfx.ERR_INVALID_ARG
        assert L.idfx_set_option_real(h, idfx.OPT_INTEGRATOR, 2.0) == idfx.ERR_INVALID_ARG
    # the vector potential needs a magnetic field, outflow boundaries must not have one
    assert L.idfx_set_option(hd, idfx.OPT_CT_FORM, idfx.CT_POTENTIAL) == idfx.ERR_UNSUPPORTED
    assert L.idfx_set_option(mhd, idfx.OPT_BOUNDARY, idfx.BOUNDARY_OUTFLOW) == idfx.ERR_UNSUPPORTED
    assert L.idfx_set_option(hd, idfx.OPT_BOUNDARY, idfx.BOUNDARY_OUTFLOW) == idfx.OK
    # the workspace grows by 12 fields with the potential (and holds 15 more for the 2D-HLL EMF)
    w_face = L.idfx_workspace_bytes(mhd)
    assert L.idfx_set_option(mhd, idfx.OPT_CT_FORM, idfx.CT_POTENTIAL) == idfx.OK
    w_pot = L.idfx_workspace_bytes(mhd)
    plain = L.idfx_create(8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLLD, idfx.LIMITER_VANLEER, idfx.EMF_UCT_CONTACT)
    w_plain = L.idfx_workspace_bytes(plain)
    field = (w_pot - w_face) // 12
    assert field * 12 == w_pot - w_face and w_face - w_plain == 15 * field and field >= 12 ** 3 * 8
    for h in (hd, mhd, plain):
        L.idfx_destroy(h)
    assert L.idfx_set_option(None, idfx.OPT_INTEGRATOR, 2) == idfx.ERR_INVALID_ARG


def test_ppm_rules_on_the_host(L):
    """PPM (limiter 4): refused with the 2D-HLL EMF and with outflow boundaries, 18 more workspace fields (include/idfx.h)."""
    assert not L.idfx_create(8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLL, idfx.LIMITER_PPM, idfx.EMF_UCT_HLL)
    assert b"PPM" in L.idfx_last_error()
    assert not L.idfx_create(8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLL, 5, idfx.EMF_NONE)
    ppm = L.idfx_create(8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLLD, idfx.LIMITER_PPM, idfx.EMF_UCT_CONTACT)
    plm = L.idfx_create(8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLLD, idfx.LIMITER_VANLEER, idfx.EMF_UCT_CONTACT)
    hd = L.idfx_create(8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLLC, idfx.LIMITER_PPM, idfx.EMF_NONE)
    assert ppm and plm and hd
    extra = L.idfx_workspace_bytes(ppm) - L.idfx_workspace_bytes(plm)
    assert extra % 18 == 0 and extra // 18 >= 12 ** 3 * 8
    assert L.idfx_set_option(hd, idfx.OPT_BOUNDARY, idfx.BOUNDARY_OUTFLOW) == idfx.ERR_UNSUPPORTED
    assert L.idfx_set_option(hd, idfx.OPT_INTEGRATOR, 3) == idfx.OK
    for h in (ppm, plm, hd):
        L.idfx_destroy(h)


def test_binding_fails_loudly_without_gpu():
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError):
        idfx.Idfx(8, 8, 8, 0.1, 1.4, idfx.SOLVER_HLL, idfx.LIMITER_MINMOD, idfx.EMF_NONE)


# ---- input generators -------------------------------------------------------------------------
def divb(b):
    return (torch.roll(b[0], -1, 2) - b[0]) + (torch.roll(b[1], -1, 1) - b[1]) + (torch.roll(b[2], -1, 0) - b[2])


def test_mode_counts_match_recipe():
    assert len(inputs.half_space_modes(4)) == 128
    assert len(inputs.half_space_modes(8)) == 1054


def test_random_phase_field_is_the_stated_sum():
    n, modes = 12, inputs.half_space_modes(2)
    rng = np.random.default_rng(0)
    ph = rng.uniform(0, 2 * np.pi, len(modes))
    f = inputs.random_phase_field(n, modes, ph, (0.5, 0.0, 0.5)).numpy()
    x, y, z = (np.arange(n) + 0.5) / n, np.arange(n) / n, (np.arange(n) + 0.5) / n
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    ref = sum(np.cos(2 * np.pi * (k[0] * X + k[1] * Y + k[2] * Z) + p) for k, p in zip(modes, ph))
    np.testing.assert_allclose(f, ref, atol=1e-11)


@pytest.mark.parametrize("name,n", [("config1", 16), ("config3", 16), ("config4", 24), ("config5", 24)])
def test_configs_are_seeded_solenoidal_and_scaled(name, n):
    p1, b1, cfg = inputs.make(name, n=n)
    p2, b2, _ = inputs.make(name, n=n)
    assert torch.equal(p1, p2) and torch.equal(b1, b2)
    assert float(divb(b1).abs().max() * cfg["dx"] / b1.abs().max()) < 1e-12
    assert p1.dtype == torch.float64 and tuple(p1.shape) == (5, n, n, n)
    if name in ("config3", "config5"):
        assert float((b1 * b1).sum(0).mean()) == pytest.approx(0.2, rel=1e-12)          # beta = 10
        assert float((p1[1:4] ** 2).sum(0).mean()) == pytest.approx(5.0 / 3.0, rel=1e-12)  # rms Mach 1
    if name == "config4":
        assert float((b1 * b1).sum(0).mean()) == pytest.approx(2.0, rel=1e-12)          # beta = 1
        assert float(b1[2].mean()) == pytest.approx(0.1, abs=1e-12)
        assert float((p1[1:4] ** 2).sum(0).mean()) == pytest.approx(4 * 5.0 / 3.0, rel=1e-12)
        assert float(p1[0].log().std()) == pytest.approx(0.1, rel=0.05)
    if name == "config1":
        assert float(p1[0].mean()) == pytest.approx(25 / (36 * np.pi), abs=1e-4)
        assert float(b1[2].abs().max()) == 0.0


def test_config2_is_hydro():
    p, b, cfg = inputs.make("config2", n=16)
    assert b is None and cfg["emf"] == inputs.EMF_NONE and cfg["solver"] == inputs.SOLVER_HLLC
    assert float((p[1:4] ** 2).sum(0).mean()) == pytest.approx(0.25 * 5.0 / 3.0, rel=1e-12)
