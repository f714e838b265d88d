"""Thin ctypes binding over the C-ABI library (include/idfx.h) — argument marshalling only.

Every step of the method runs in the CUDA kernels of libidfx.so; torch is used for device memory (the
workspace and the state tensors) and for the stream.  There is no CPU fallback: if the library is
missing or no CUDA device is present, calls raise.
"""
import ctypes
import os

import torch

SOLVER_HLL, SOLVER_HLLC, SOLVER_HLLD, SOLVER_ROE, SOLVER_RUSANOV = 0, 1, 2, 3, 4
LIMITER_FLAT, LIMITER_MINMOD, LIMITER_VANLEER, LIMITER_LIMO3, LIMITER_PPM = 0, 1, 2, 3, 4
OPT_INTEGRATOR, OPT_CT_FORM, OPT_PRESSURE_FLOOR, OPT_BOUNDARY, OPT_EXCHANGE_DIRS, OPT_OUTFLOW_SIDES = 0, 1, 2, 3, 4, 5
BOUNDARY_PERIODIC, BOUNDARY_OUTFLOW = 0, 1
CT_FACE, CT_POTENTIAL = 0, 1
EMF_NONE, EMF_ARITHMETIC, EMF_UCT_CONTACT, EMF_UCT_0, EMF_UCT_HLL, EMF_UCT_HLLD = 0, 1, 2, 3, 4, 5
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_NOT_BOUND, ERR_CUDA, ERR_UNPHYSICAL = 0, -1, -2, -3, -4, -5

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libidfx.so")

# every symbol include/idfx.h declares
SYMBOLS = (
    "idfx_create", "idfx_workspace_bytes", "idfx_bind", "idfx_set_state", "idfx_set_state_host",
    "idfx_get_state", "idfx_get_state_host", "idfx_get_conserved", "idfx_compute_dt", "idfx_step",
    "idfx_advance", "idfx_last_dt", "idfx_status", "idfx_launch_count", "idfx_last_error", "idfx_destroy",
    "idfx_profile_enable", "idfx_profile_read", "idfx_profile_kernel_name",
    "idfx_set_option", "idfx_advance_to", "idfx_time", "idfx_get_potential", "idfx_set_option_real", "idfx_floor_count",
    "idfx_probe_fp64",
    "idfx_noalloc_compute_dt", "idfx_noalloc_last_error",
    "idfx_cycle_begin", "idfx_stage_flux", "idfx_stage_update", "idfx_cycle_end", "idfx_dt_reduce_offset",
    "idfx_set_state_finish", "idfx_halo_count", "idfx_halo_pack", "idfx_halo_unpack", "idfx_halo_fill", "idfx_halo_push",
)

_lib = None


class IdfxError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("idfx error %d: %s" % (code, msg))
        self.code = code


def lib():
    """Loads libidfx.so (built by paper_2304_13746_b200/build.py or __graft_entry__.build())."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("%s is missing: run `python -m paper_2304_13746_b200.build` (nvcc, sm_100a)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cd, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
        dp = ctypes.POINTER(ctypes.c_double)
        L.idfx_create.restype = vp
        L.idfx_create.argtypes = [ci, ci, ci, cd, cd, ci, ci, ci]
        L.idfx_workspace_bytes.restype = sz
        L.idfx_workspace_bytes.argtypes = [vp]
        L.idfx_bind.argtypes = [vp, vp, sz, vp]
        for n in ("idfx_set_state", "idfx_set_state_host", "idfx_get_state", "idfx_get_state_host", "idfx_get_conserved"):
            getattr(L, n).argtypes = [vp, vp, vp]
        L.idfx_compute_dt.argtypes = [vp, cd, dp]
        L.idfx_step.argtypes = [vp, cd]
        L.idfx_advance.argtypes = [vp, ci, cd]
        L.idfx_last_dt.argtypes = [vp, dp]
        L.idfx_set_option.argtypes = [vp, ci, ci]
        L.idfx_advance_to.argtypes = [vp, cd, cd, ci, ctypes.POINTER(ci), dp]
        L.idfx_time.argtypes = [vp, dp]
        L.idfx_get_potential.argtypes = [vp, vp]
        L.idfx_set_option_real.argtypes = [vp, ci, cd]
        L.idfx_floor_count.argtypes = [vp, ctypes.POINTER(ctypes.c_longlong)]
        L.idfx_status.argtypes = [vp]
        L.idfx_launch_count.argtypes = [vp]
        L.idfx_launch_count.restype = ctypes.c_longlong
        L.idfx_profile_enable.argtypes = [vp, ci]
        L.idfx_profile_read.argtypes = [vp, ci, dp, ctypes.POINTER(ctypes.c_longlong)]
        L.idfx_profile_kernel_name.argtypes = [ci]
        L.idfx_profile_kernel_name.restype = ctypes.c_char_p
        L.idfx_probe_fp64.argtypes = [vp, ci, dp, dp]
        L.idfx_cycle_begin.argtypes = [vp, cd, cd]
        L.idfx_stage_flux.argtypes = [vp, ci]
        L.idfx_stage_update.argtypes = [vp, ci]
        L.idfx_cycle_end.argtypes = [vp]
        L.idfx_dt_reduce_offset.argtypes = [vp]
        L.idfx_dt_reduce_offset.restype = sz
        L.idfx_set_state_finish.argtypes = [vp]
        L.idfx_halo_count.argtypes = [vp, ci]
        L.idfx_halo_count.restype = ctypes.c_longlong
        L.idfx_halo_pack.argtypes = [vp, ci, ci, vp]
        L.idfx_halo_unpack.argtypes = [vp, ci, ci, vp]
        L.idfx_halo_fill.argtypes = [vp, ci, ci, ci]
        L.idfx_halo_push.argtypes = [vp, ci, ci, vp]
        L.idfx_noalloc_compute_dt.argtypes = [ci, ci, ci, cd, cd, ci, vp, vp, cd, vp, vp]
        L.idfx_noalloc_last_error.restype = ctypes.c_char_p
        L.idfx_last_error.restype = ctypes.c_char_p
        L.idfx_destroy.argtypes = [vp]
        L.idfx_destroy.restype = None
        _lib = L
    return _lib


def _check(rc):
    if rc != OK:
        raise IdfxError(rc, lib().idfx_last_error().decode())


def probe_fp64(repeats=5):
    """(TFLOP/s, 1e12 fp64 instructions/s) of chains of independent DFMAs on the current device."""
    tf, ti = ctypes.c_double(), ctypes.c_double()
    rc = lib().idfx_probe_fp64(torch.cuda.current_stream().cuda_stream, repeats, ctypes.byref(tf), ctypes.byref(ti))
    if rc != OK:
        raise IdfxError(rc, "fp64 probe failed")
    return tf.value, ti.value


NOALLOC_MAX_CELLS = 262144   # include/idfx_noalloc.h


def noalloc_compute_dt(prim, bface, dx, gamma, limiter, cfl, out=None):
    """The CFL step of a periodic box given as contiguous device tensors, through the entry point that allocates nothing
    (include/idfx_noalloc.h; at most NOALLOC_MAX_CELLS cells; calls that overlap on the GPU race on its static scratch).
    `out`: a one-element float64 device tensor for the result (made here when None: that allocation is torch's, the
    library call itself allocates nothing).  Enqueued on torch's current stream; returns `out` without synchronising."""
    assert prim.is_cuda and prim.dtype == torch.float64 and prim.is_contiguous() and prim.shape[0] == 5
    nz, ny, nx = prim.shape[1:]
    if bface is not None:
        assert bface.is_cuda and bface.dtype == torch.float64 and bface.is_contiguous() and tuple(bface.shape) == (3, nz, ny, nx)
    if out is None:
        out = torch.empty(1, dtype=torch.float64, device=prim.device)
    with torch.cuda.device(prim.device):
        rc = lib().idfx_noalloc_compute_dt(nx, ny, nz, dx, gamma, limiter, prim.data_ptr(),
                                           bface.data_ptr() if bface is not None else None, cfl,
                                           torch.cuda.current_stream(prim.device).cuda_stream, out.data_ptr())
    if rc != OK:
        raise IdfxError(rc, lib().idfx_noalloc_last_error().decode())
    return out


class Idfx:
    """One periodic nx*ny*nz box on one GPU.  Tensors are float64, [var][nz][ny][nx]."""

    def __init__(self, nx, ny, nz, dx, gamma, solver, limiter, emf_mode, device="cuda:0", stream=None, nstages=2,
                 ct_form=CT_FACE, pressure_floor=0.0, boundary=BOUNDARY_PERIODIC, exchange_dirs=0, outflow_sides=0):
        self.L = lib()
        self.h = self.L.idfx_create(nx, ny, nz, dx, gamma, solver, limiter, emf_mode)
        if not self.h:
            raise IdfxError(ERR_INVALID_ARG, self.L.idfx_last_error().decode())
        if nstages != 2:
            _check(self.L.idfx_set_option(self.h, OPT_INTEGRATOR, nstages))
        if ct_form != CT_FACE:
            _check(self.L.idfx_set_option(self.h, OPT_CT_FORM, ct_form))
        if pressure_floor:
            _check(self.L.idfx_set_option_real(self.h, OPT_PRESSURE_FLOOR, pressure_floor))
        if boundary != BOUNDARY_PERIODIC:
            _check(self.L.idfx_set_option(self.h, OPT_BOUNDARY, boundary))
        if exchange_dirs:
            _check(self.L.idfx_set_option(self.h, OPT_EXCHANGE_DIRS, exchange_dirs))
        if outflow_sides:
            _check(self.L.idfx_set_option(self.h, OPT_OUTFLOW_SIDES, outflow_sides))
        self.nstages = nstages
        if not torch.cuda.is_available():
            raise RuntimeError("idfx needs a CUDA device; there is no CPU fallback")
        self.device = torch.device(device)
        self.shape = (nz, ny, nx)
        self.mhd = emf_mode != EMF_NONE
        nbytes = self.L.idfx_workspace_bytes(self.h)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        # The library enqueues on its own stream (a non-default stream can be captured into CUDA graphs); every call
        # below orders that stream after the caller's current stream and the caller's stream after it.
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
        _check(self.L.idfx_bind(self.h, self.workspace.data_ptr(), nbytes, self.stream.cuda_stream))

    class _Ordered:
        def __init__(self, sim):
            self.sim = sim

        def __enter__(self):
            self.cur = torch.cuda.current_stream(self.sim.device)
            if self.cur != self.sim.stream:
                self.sim.stream.wait_stream(self.cur)

        def __exit__(self, *exc):
            if self.cur != self.sim.stream:
                self.cur.wait_stream(self.sim.stream)
            return False

    def _ordered(self):
        return Idfx._Ordered(self)

    def close(self):
        if getattr(self, "h", None):
            self.L.idfx_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        self.close()

    def _dev(self, t, nvar):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == (nvar,) + self.shape
        return t.data_ptr()

    def _host(self, t, nvar):
        assert (not t.is_cuda) and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == (nvar,) + self.shape
        return t.data_ptr()

    def set_state(self, prim, bface=None):
        host = not prim.is_cuda
        f = self.L.idfx_set_state_host if host else self.L.idfx_set_state
        p = self._host if host else self._dev
        with self._ordered():
            _check(f(self.h, p(prim, 5), p(bface, 3) if bface is not None else None))

    def get_state(self, out_prim=None, out_bface=None, host=False):
        dev = "cpu" if host else self.device
        if out_prim is None:
            out_prim = torch.empty((5,) + self.shape, dtype=torch.float64, device=dev, pin_memory=host)
        if out_bface is None and self.mhd:
            out_bface = torch.empty((3,) + self.shape, dtype=torch.float64, device=dev, pin_memory=host)
        f = self.L.idfx_get_state_host if host else self.L.idfx_get_state
        p = self._host if host else self._dev
        with self._ordered():
            _check(f(self.h, p(out_prim, 5), p(out_bface, 3) if out_bface is not None else None))
        return out_prim, out_bface

    def get_conserved(self):
        cons = torch.empty((5,) + self.shape, dtype=torch.float64, device=self.device)
        bface = torch.empty((3,) + self.shape, dtype=torch.float64, device=self.device) if self.mhd else None
        with self._ordered():
            _check(self.L.idfx_get_conserved(self.h, cons.data_ptr(), bface.data_ptr() if self.mhd else None))
        return cons, bface

    def compute_dt(self, cfl):
        dt = ctypes.c_double()
        with self._ordered():
            _check(self.L.idfx_compute_dt(self.h, cfl, ctypes.byref(dt)))
        return dt.value

    def step(self, dt):
        with self._ordered():
            _check(self.L.idfx_step(self.h, dt))

    def advance(self, nsteps, cfl):
        with self._ordered():
            _check(self.L.idfx_advance(self.h, nsteps, cfl))

    def set_integrator(self, nstages):
        _check(self.L.idfx_set_option(self.h, OPT_INTEGRATOR, nstages))
        self.nstages = nstages

    # ---- the cycle in pieces and the halo slabs (include/idfx.h, "The cycle in pieces"; driven by decomp.py) ----
    def cycle_begin(self, dt, cfl):
        with self._ordered():
            _check(self.L.idfx_cycle_begin(self.h, dt, cfl))

    def stage_flux(self, stage):
        with self._ordered():
            _check(self.L.idfx_stage_flux(self.h, stage))

    def stage_update(self, stage):
        with self._ordered():
            _check(self.L.idfx_stage_update(self.h, stage))

    def cycle_end(self):
        _check(self.L.idfx_cycle_end(self.h))

    def set_state_finish(self):
        with self._ordered():
            _check(self.L.idfx_set_state_finish(self.h))

    def dt_word(self):
        """The 8 bytes of the workspace that hold max_cells sum_d c_d/dx of the running cycle, as a float64 view."""
        off = self.L.idfx_dt_reduce_offset(self.h)
        return self.workspace[off:off + 8].view(torch.float64)

    def halo_count(self, d):
        return self.L.idfx_halo_count(self.h, d)

    def new_buffer(self, count):
        return torch.empty(count, dtype=torch.float64, device=self.device)

    def adopt(self, buf):
        """A neighbour's packed slab, on this context's device (a peer copy when the neighbour lives on another GPU)."""
        return buf if buf.device == self.device else buf.to(self.device)

    def halo_pack(self, d, side, buf):
        assert buf.is_cuda and buf.dtype == torch.float64 and buf.is_contiguous() and buf.numel() >= self.halo_count(d)
        with self._ordered():
            _check(self.L.idfx_halo_pack(self.h, d, side, buf.data_ptr()))

    def halo_unpack(self, d, side, buf):
        assert buf.is_cuda and buf.dtype == torch.float64 and buf.is_contiguous() and buf.numel() >= self.halo_count(d)
        with self._ordered():
            _check(self.L.idfx_halo_unpack(self.h, d, side, buf.data_ptr()))

    def halo_push(self, d, side, neighbour):
        """My two layers next to `side` straight into `neighbour`'s ghost layers of the opposite side (same process)."""
        nb_cur = torch.cuda.current_stream(neighbour.device)
        if nb_cur != neighbour.stream:
            nb_cur.wait_stream(neighbour.stream)      # the neighbour is done with its ghost layers
        with self._ordered():
            if neighbour.device != self.device:
                self.stream.wait_stream(nb_cur)
            _check(self.L.idfx_halo_push(self.h, d, side, neighbour.h))
        if neighbour.device != self.device:
            nb_cur.wait_stream(self.stream)

    def halo_fill(self, d, side, zero_gradient):
        with self._ordered():
            _check(self.L.idfx_halo_fill(self.h, d, side, 1 if zero_gradient else 0))

    def advance_to(self, t_end, cfl, max_steps=(1 << 31) - 1):
        """Returns (number of cycles taken, time reached)."""
        n, t = ctypes.c_int(), ctypes.c_double()
        with self._ordered():
            _check(self.L.idfx_advance_to(self.h, t_end, cfl, max_steps, ctypes.byref(n), ctypes.byref(t)))
        return n.value, t.value

    def floor_count(self):
        n = ctypes.c_longlong()
        _check(self.L.idfx_floor_count(self.h, ctypes.byref(n)))
        return n.value

    def time(self):
        t = ctypes.c_double()
        _check(self.L.idfx_time(self.h, ctypes.byref(t)))
        return t.value

    def get_potential(self):
        pot = torch.empty((3,) + self.shape, dtype=torch.float64, device=self.device)
        with self._ordered():
            _check(self.L.idfx_get_potential(self.h, pot.data_ptr()))
        return pot

    def last_dt(self):
        dt = ctypes.c_double()
        _check(self.L.idfx_last_dt(self.h, ctypes.byref(dt)))
        return dt.value

    def status(self):
        return self.L.idfx_status(self.h)

    def launch_count(self):
        return self.L.idfx_launch_count(self.h)

    def profile(self, on):
        _check(self.L.idfx_profile_enable(self.h, 1 if on else 0))

    def profile_read(self):
        """{kernel class: (total ms, launches)} accumulated since profile(True)."""
        out = {}
        k = 0
        while True:
            name = self.L.idfx_profile_kernel_name(k)
            if name is None:
                return out
            ms, n = ctypes.c_double(), ctypes.c_longlong()
            _check(self.L.idfx_profile_read(self.h, k, ctypes.byref(ms), ctypes.byref(n)))
            out[name.decode()] = (ms.value, n.value)
            k += 1
