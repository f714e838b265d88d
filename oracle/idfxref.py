"""ctypes loader for the CPU oracle (oracle/idfxref.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It holds argument marshalling only; every formula of the
method lives in idfxref.cpp.  Nothing here imports the CUDA package.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "idfxref.cpp")
_LIB = os.path.join(_HERE, "libidfxref.so")

SOLVER_HLL, SOLVER_HLLC, SOLVER_HLLD, SOLVER_ROE, SOLVER_RUSANOV = 0, 1, 2, 3, 4
LIMITER_FLAT, LIMITER_MINMOD, LIMITER_VANLEER, LIMITER_LIMO3 = 0, 1, 2, 3
OPT_INTEGRATOR, OPT_CT_FORM, OPT_PRESSURE_FLOOR, OPT_BOUNDARY = 0, 1, 2, 3
BOUNDARY_PERIODIC, BOUNDARY_OUTFLOW = 0, 1
CT_FACE, CT_POTENTIAL = 0, 1
EMF_NONE, EMF_ARITHMETIC, EMF_UCT_CONTACT, EMF_UCT_0, EMF_UCT_HLL, EMF_UCT_HLLD = 0, 1, 2, 3, 4, 5
OK, ERR_UNPHYSICAL = 0, -5

_lib = None


def build(force=False):
    """Compile the oracle (g++ -O2, FMA contraction off so the arithmetic is exactly as written)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", _SRC, "-o", tmp]
        )
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        L.idfxref_create.restype = vp
        L.idfxref_create.argtypes = [ci, ci, ci, cd, cd, ci, ci, ci]
        L.idfxref_destroy.argtypes = [vp]
        L.idfxref_destroy.restype = None
        for name in ("set_state", "get_state", "get_conserved"):
            f = getattr(L, "idfxref_" + name)
            f.argtypes = [vp, dp, dp]
            f.restype = ci
        L.idfxref_compute_dt.argtypes = [vp, cd, dp]
        L.idfxref_step.argtypes = [vp, cd]
        L.idfxref_advance.argtypes = [vp, ci, cd]
        L.idfxref_last_dt.argtypes = [vp, dp]
        L.idfxref_status.argtypes = [vp]
        L.idfxref_roe_fallbacks.argtypes = [vp]
        L.idfxref_roe_fallbacks.restype = ctypes.c_longlong
        L.idfxref_get_emf.argtypes = [vp, dp]
        L.idfxref_get_flux.argtypes = [vp, ci, dp, dp]
        L.idfxref_cons_from_prim.argtypes = [cd, dp, cd, dp]
        L.idfxref_cons_from_prim.restype = None
        L.idfxref_phys_flux.argtypes = [cd, dp, cd, dp]
        L.idfxref_phys_flux.restype = None
        L.idfxref_flux_from_cons.argtypes = [cd, dp, cd, dp]
        L.idfxref_flux_from_cons.restype = None
        L.idfxref_riemann.argtypes = [ci, cd, dp, dp, cd, dp, dp]
        L.idfxref_wave_speeds.argtypes = [cd, dp, dp, cd, dp, dp]
        L.idfxref_wave_speeds.restype = None
        L.idfxref_hlld_uct_coeffs.argtypes = [cd, dp, dp, cd, dp]
        L.idfxref_hlld_uct_coeffs.restype = None
        L.idfxref_slope.argtypes = [ci, cd, cd]
        L.idfxref_slope.restype = cd
        L.idfxref_hllc_fan.argtypes = [cd, dp, dp, dp, dp]
        L.idfxref_hllc_fan.restype = None
        L.idfxref_hlld_fan.argtypes = [cd, dp, dp, cd, dp, dp]
        L.idfxref_hlld_fan.restype = None
        L.idfxref_roe_system.argtypes = [cd, dp, dp, cd, dp, dp, dp]
        L.idfxref_set_option.argtypes = [vp, ci, ci]
        L.idfxref_set_option_real.argtypes = [vp, ci, cd]
        L.idfxref_floor_count.argtypes = [vp]
        L.idfxref_floor_count.restype = ctypes.c_longlong
        L.idfxref_advance_to.argtypes = [vp, cd, cd, ci, ctypes.POINTER(ci)]
        L.idfxref_time.argtypes = [vp, dp]
        L.idfxref_get_potential.argtypes = [vp, dp]
        L.idfxref_reconstruct.argtypes = [ci, cd, cd, cd, cd, dp, dp]
        L.idfxref_reconstruct.restype = None
        L.idfxref_ppm_faces.argtypes = [dp, dp, dp]
        L.idfxref_ppm_faces.restype = None
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if a is not None else None


def _c(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


class Oracle:
    """One oracle context: a periodic nx*ny*nz box (arrays are [var][nz][ny][nx])."""

    def __init__(self, nx, ny, nz, dx, gamma, solver, limiter, emf_mode, nstages=2, ct_form=CT_FACE, pressure_floor=0.0,
                 boundary=BOUNDARY_PERIODIC):
        self.L = lib()
        self.shape = (nz, ny, nx)
        self.mhd = emf_mode != EMF_NONE
        self.h = self.L.idfxref_create(nx, ny, nz, dx, gamma, solver, limiter, emf_mode)
        if not self.h:
            raise ValueError("idfxref_create rejected the arguments")
        if nstages != 2 and self.L.idfxref_set_option(self.h, OPT_INTEGRATOR, nstages) != OK:
            raise ValueError("bad number of stages")
        if ct_form != CT_FACE and self.L.idfxref_set_option(self.h, OPT_CT_FORM, ct_form) != OK:
            raise ValueError("bad CT form")
        if pressure_floor and self.L.idfxref_set_option_real(self.h, OPT_PRESSURE_FLOOR, pressure_floor) != OK:
            raise ValueError("bad pressure floor")
        if boundary != BOUNDARY_PERIODIC and self.L.idfxref_set_option(self.h, OPT_BOUNDARY, boundary) != OK:
            raise ValueError("bad boundary (with a magnetic field: outflow needs face CT, no PPM, no 2D-HLL EMF)")

    def close(self):
        if self.h:
            self.L.idfxref_destroy(self.h)
            self.h = None

    def __del__(self):
        self.close()

    def set_state(self, prim, bface=None):
        prim, bface = _c(prim), _c(bface)
        assert prim.shape == (5,) + self.shape
        assert bface is None or bface.shape == (3,) + self.shape
        return self.L.idfxref_set_state(self.h, _p(prim), _p(bface))

    def get_state(self):
        prim = np.empty((5,) + self.shape)
        bface = np.empty((3,) + self.shape) if self.mhd else None
        self.L.idfxref_get_state(self.h, _p(prim), _p(bface))
        return prim, bface

    def get_conserved(self):
        cons = np.empty((5,) + self.shape)
        bface = np.empty((3,) + self.shape) if self.mhd else None
        self.L.idfxref_get_conserved(self.h, _p(cons), _p(bface))
        return cons, bface

    def compute_dt(self, cfl):
        dt = ctypes.c_double()
        rc = self.L.idfxref_compute_dt(self.h, cfl, ctypes.byref(dt))
        if rc == -1:
            raise ValueError("bad cfl")
        return dt.value

    def step(self, dt):
        return self.L.idfxref_step(self.h, dt)

    def advance(self, nsteps, cfl):
        return self.L.idfxref_advance(self.h, nsteps, cfl)

    def advance_to(self, t_end, cfl, max_steps=1 << 30):
        """Returns (status, number of cycles taken)."""
        n = ctypes.c_int()
        rc = self.L.idfxref_advance_to(self.h, t_end, cfl, max_steps, ctypes.byref(n))
        return rc, n.value

    def floor_count(self):
        return self.L.idfxref_floor_count(self.h)

    def time(self):
        t = ctypes.c_double()
        self.L.idfxref_time(self.h, ctypes.byref(t))
        return t.value

    def get_potential(self):
        pot = np.empty((3,) + self.shape)
        if self.L.idfxref_get_potential(self.h, _p(pot)) != OK:
            raise ValueError("no vector potential in this context")
        return pot

    def last_dt(self):
        dt = ctypes.c_double()
        self.L.idfxref_last_dt(self.h, ctypes.byref(dt))
        return dt.value

    def status(self):
        return self.L.idfxref_status(self.h)

    def roe_fallbacks(self):
        return self.L.idfxref_roe_fallbacks(self.h)

    def get_emf(self):
        emf = np.empty((3,) + self.shape)
        self.L.idfxref_get_emf(self.h, _p(emf))
        return emf

    def get_flux(self, d):
        flux = np.empty((7,) + self.shape)
        cface = np.empty(self.shape)
        self.L.idfxref_get_flux(self.h, d, _p(flux), _p(cface))
        return flux, cface


# ---- point-wise helpers for the pins -----------------------------------------------------------
def _v7(w):
    a = np.zeros(7)
    w = np.asarray(w, dtype=np.float64)
    a[: w.size] = w
    return a


def cons_from_prim(gamma, W, Bn=0.0):
    U = np.empty(7)
    lib().idfxref_cons_from_prim(gamma, _p(_v7(W)), Bn, _p(U))
    return U


def phys_flux(gamma, W, Bn=0.0):
    F = np.empty(7)
    lib().idfxref_phys_flux(gamma, _p(_v7(W)), Bn, _p(F))
    return F


def flux_from_cons(gamma, U, Bn=0.0):
    F = np.empty(7)
    lib().idfxref_flux_from_cons(gamma, _p(_v7(U)), Bn, _p(F))
    return F


def riemann(solver, gamma, WL, WR, Bn=0.0):
    """Returns (F[7], c_face, fell_back_to_hll)."""
    F = np.empty(7)
    c = ctypes.c_double()
    fb = lib().idfxref_riemann(solver, gamma, _p(_v7(WL)), _p(_v7(WR)), Bn, _p(F), ctypes.byref(c))
    return F, c.value, fb


def wave_speeds(gamma, WL, WR, Bn=0.0):
    sl, sr = ctypes.c_double(), ctypes.c_double()
    lib().idfxref_wave_speeds(gamma, _p(_v7(WL)), _p(_v7(WR)), Bn, ctypes.byref(sl), ctypes.byref(sr))
    return sl.value, sr.value


def hlld_uct_coeffs(gamma, WL, WR, Bn):
    """(a_L, d_L, d_R, vbar_t1, vbar_t2) of the 2D-HLLD EMF at one face (reading G24)."""
    out = np.empty(5)
    lib().idfxref_hlld_uct_coeffs(gamma, _p(_v7(WL)), _p(_v7(WR)), Bn, _p(out))
    return out


def slope(limiter, dm, dp):
    return lib().idfxref_slope(limiter, dm, dp)


def reconstruct(limiter, qm, q0, qp, dx):
    """(value at the lower face, value at the upper face) of cell i's reconstruction."""
    lo, hi = ctypes.c_double(), ctypes.c_double()
    lib().idfxref_reconstruct(limiter, qm, q0, qp, dx, ctypes.byref(lo), ctypes.byref(hi))
    return lo.value, hi.value


def ppm_faces(a5):
    """(value at the lower face, value at the upper face) of cell j's PPM parabola from (a_{j-2}, ..., a_{j+2})."""
    a = np.ascontiguousarray(a5, dtype=np.float64)
    assert a.shape == (5,)
    lo, hi = ctypes.c_double(), ctypes.c_double()
    lib().idfxref_ppm_faces(_p(a), ctypes.byref(lo), ctypes.byref(hi))
    return lo.value, hi.value


def hllc_fan(gamma, WL, WR):
    S = np.empty(3)
    st = np.empty((2, 5))
    lib().idfxref_hllc_fan(gamma, _p(_v7(WL)), _p(_v7(WR)), _p(S), _p(st))
    return S, st


def hlld_fan(gamma, WL, WR, Bn):
    S = np.empty(5)
    st = np.empty((4, 7))
    lib().idfxref_hlld_fan(gamma, _p(_v7(WL)), _p(_v7(WR)), Bn, _p(S), _p(st))
    return S, st


def roe_system(gamma, WL, WR, Bn):
    lam = np.empty(7)
    R = np.empty((7, 7))
    Lm = np.empty((7, 7))
    ok = lib().idfxref_roe_system(gamma, _p(_v7(WL)), _p(_v7(WR)), Bn, _p(lam), _p(R), _p(Lm))
    return ok, lam, R, Lm
