"""Thin ctypes binding of the C ABI in include/phx.h (libphx.so, hand-written sm_100a CUDA).

Argument marshalling only: every step of the GRMHD update runs in the CUDA kernels behind the
C ABI.  There is no CPU fallback: importing works without a GPU (so that the symbol table can be
checked), but every call needs CUDA tensors and the library fails loudly if it is missing.
Function names mirror the C entry points without the `phx_` prefix.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libphx.so")

OK, EINVAL, ECUDA, ENOMEM, EUNSUPPORTED = 0, 1, 2, 3, 4
M_RHO_FLOOR, M_EPS_FLOOR, M_EPS_CLIPPED, M_W_CEIL, M_NOCONV, M_BAD_INPUT, M_EXCISED, M_SCALAR_CLIPPED = 1, 2, 4, 8, 16, 32, 64, 128
FLOOR_CONST, FLOOR_EXP_X1, FLOOR_POW_X1, FLOOR_POW_R = 0, 1, 2, 3

KERNEL_CLASSES = ("sweep_x", "sweep_y", "sweep_z", "update", "fill_ghosts", "cfl", "prim_to_cons", "c2p", "copy")

EXPORTS = (
    "phx_init_mesh", "phx_free_mesh", "phx_field_elems", "phx_mask_elems", "phx_prim_to_cons",
    "phx_cons_to_prim", "phx_fill_ghosts", "phx_rk_stage", "phx_cfl_dt", "phx_rk2_step",
    "phx_evolve_host", "phx_debug_flux", "phx_launch_count", "phx_last_error",
    "phx_profile_enable", "phx_profile_read", "phx_rk2_step_cfl", "phx_evolve_device", "phx_debug_enable_flux",
    "phx_debug_fp64_peak", "phx_count_masked",
)


class Params(C.Structure):
    """Mirror of phx_params (include/phx.h)."""
    _fields_ = [
        ("metric", C.c_int), ("bh_mass", C.c_double), ("bh_spin", C.c_double), ("r_excise", C.c_double),
        ("nbx", C.c_int), ("nby", C.c_int), ("nbz", C.c_int),
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ng", C.c_int),
        ("xmin", C.c_double * 3), ("xmax", C.c_double * 3), ("bc", (C.c_int * 2) * 3),
        ("gamma_ad", C.c_double), ("recon", C.c_int), ("riemann", C.c_int), ("use_ct", C.c_int),
        ("rho_floor", C.c_double), ("eps_floor", C.c_double), ("w_max", C.c_double),
        ("c2p_tol", C.c_double), ("c2p_maxit", C.c_int), ("shift", C.c_double * 3),
        ("nscalar", C.c_int), ("scalar_min", C.c_double), ("scalar_max", C.c_double),
        ("floor_form", C.c_int), ("floor_alpha_rho", C.c_double), ("floor_alpha_eps", C.c_double),
    ]

# parameters added after the first version of the ABI: optional in the dictionaries, with the values that switch them off
_OPTIONAL = dict(shift=(0.0, 0.0, 0.0), nscalar=0, scalar_min=0.0, scalar_max=1.0, floor_form=0,
                 floor_alpha_rho=2.0, floor_alpha_eps=1.0)


def make_params(p: dict) -> Params:
    q = Params()
    for name, _ in Params._fields_:
        v = p.get(name, _OPTIONAL[name]) if name in _OPTIONAL else p[name]
        if name in ("xmin", "xmax", "shift"):
            setattr(q, name, (C.c_double * 3)(*[float(t) for t in v]))
        elif name == "bc":
            arr = ((C.c_int * 2) * 3)()
            for d in range(3):
                arr[d][0], arr[d][1] = int(v[d][0]), int(v[d][1])
            q.bc = arr
        else:
            setattr(q, name, v)
    return q


class PhxError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"phx error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libphx.so (built by paper_2410_09146_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: run `python -m paper_2410_09146_b200.build` (no CPU fallback exists)")
        L = C.CDLL(LIB_PATH)
        vp, dp, ucp, pp = C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(Params)
        L.phx_init_mesh.argtypes = [pp, vp, C.POINTER(vp)]
        L.phx_free_mesh.argtypes = [vp]
        L.phx_field_elems.argtypes = [vp]; L.phx_field_elems.restype = C.c_size_t
        L.phx_mask_elems.argtypes = [vp]; L.phx_mask_elems.restype = C.c_size_t
        L.phx_prim_to_cons.argtypes = [vp, dp, dp, vp]
        L.phx_cons_to_prim.argtypes = [vp, dp, dp, ucp, vp]
        L.phx_fill_ghosts.argtypes = [vp, dp, vp]
        L.phx_rk_stage.argtypes = [vp, C.c_double, C.c_double, C.c_double, dp, dp, dp, ucp, vp]
        L.phx_cfl_dt.argtypes = [vp, dp, C.c_double, dp, C.POINTER(C.c_double), vp]
        L.phx_rk2_step.argtypes = [vp, dp, dp, dp, dp, ucp, vp]
        L.phx_rk2_step_cfl.argtypes = [vp, C.c_double, dp, dp, dp, dp, ucp, vp]
        L.phx_evolve_device.argtypes = [vp, C.c_int, C.c_double, dp, dp, dp, dp, dp, ucp, vp]
        L.phx_evolve_host.argtypes = [vp, vp, C.c_int, C.c_double, vp, vp, vp, C.POINTER(C.c_double), vp]
        L.phx_debug_flux.argtypes = [vp, C.c_int, dp, vp]
        L.phx_debug_enable_flux.argtypes = [vp, C.c_int]
        L.phx_launch_count.argtypes = [vp]; L.phx_launch_count.restype = C.c_ulonglong
        L.phx_profile_enable.argtypes = [vp, C.c_int]
        L.phx_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_ulonglong)]
        L.phx_debug_fp64_peak.argtypes = [C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int), vp]
        L.phx_count_masked.argtypes = [vp, ucp, C.c_uint, vp, C.POINTER(C.c_ulonglong), vp]
        L.phx_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(rc):
    if rc != OK:
        raise PhxError(rc, lib().phx_last_error().decode())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _dev(t, dtype, numel, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous() and t.numel() == numel):
        raise PhxError(EINVAL, f"{name}: need a contiguous CUDA tensor of {dtype} with {numel} elements")
    return C.c_void_p(t.data_ptr())


class Mesh:
    """Owner of a phx_mesh handle."""

    def __init__(self, params: dict, stream=None):
        self.params = dict(params)
        self._h = C.c_void_p()
        _check(lib().phx_init_mesh(C.byref(make_params(params)), _stream(stream), C.byref(self._h)))
        self.field_elems = lib().phx_field_elems(self._h)
        self.mask_elems = lib().phx_mask_elems(self._h)

    @property
    def handle(self):
        if not self._h:
            raise PhxError(EINVAL, "mesh already freed")
        return self._h

    def launch_count(self) -> int:
        return int(lib().phx_launch_count(self.handle))

    def debug_enable_flux(self, on=True):
        """Make the sweeps store every component of the raw Riemann fluxes (needed before debug_flux)."""
        _check(lib().phx_debug_enable_flux(self.handle, 1 if on else 0))

    def debug_flux(self, d, shape, stream=None):
        """Copy of the mesh-owned raw Riemann flux of direction d as a CUDA tensor of `shape`."""
        out = torch.empty(shape, dtype=torch.float64, device="cuda")
        _check(lib().phx_debug_flux(self.handle, int(d), _dev(out, torch.float64, self.field_elems, "out"), _stream(stream)))
        return out

    def profile_enable(self, max_records):
        _check(lib().phx_profile_enable(self.handle, int(max_records)))

    def profile_read(self):
        """{kernel class: (summed ms, records)} of the launches recorded since the last read."""
        ms = (C.c_double * len(KERNEL_CLASSES))(); n = (C.c_ulonglong * len(KERNEL_CLASSES))()
        _check(lib().phx_profile_read(self.handle, ms, n))
        return {k: (ms[i], int(n[i])) for i, k in enumerate(KERNEL_CLASSES)}

    def free(self):
        if self._h:
            lib().phx_free_mesh(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def init_mesh(params: dict, stream=None) -> Mesh:
    return Mesh(params, stream)


def free_mesh(mesh: Mesh):
    mesh.free()


def prim_to_cons(mesh, prim, cons, stream=None):
    n = mesh.field_elems
    _check(lib().phx_prim_to_cons(mesh.handle, _dev(prim, torch.float64, n, "prim"), _dev(cons, torch.float64, n, "cons"), _stream(stream)))
    return cons


def cons_to_prim(mesh, cons, prim, mask, stream=None):
    n = mesh.field_elems
    _check(lib().phx_cons_to_prim(mesh.handle, _dev(cons, torch.float64, n, "cons"), _dev(prim, torch.float64, n, "prim"),
                                  _dev(mask, torch.uint8, mesh.mask_elems, "mask"), _stream(stream)))
    return prim, mask


def fill_ghosts(mesh, prim, stream=None):
    _check(lib().phx_fill_ghosts(mesh.handle, _dev(prim, torch.float64, mesh.field_elems, "prim"), _stream(stream)))
    return prim


def rk_stage(mesh, g0, g1, beta_dt, cons0, cons, prim, mask, stream=None):
    n = mesh.field_elems
    _check(lib().phx_rk_stage(mesh.handle, float(g0), float(g1), float(beta_dt), _dev(cons0, torch.float64, n, "cons0"),
                              _dev(cons, torch.float64, n, "cons"), _dev(prim, torch.float64, n, "prim"),
                              _dev(mask, torch.uint8, mesh.mask_elems, "mask"), _stream(stream)))


def cfl_dt(mesh, prim, cfl, d_dt, host=False, stream=None):
    """d_dt: 1-element CUDA fp64 tensor.  host=True also returns the value (synchronises the stream)."""
    h = C.c_double(0.0)
    _check(lib().phx_cfl_dt(mesh.handle, _dev(prim, torch.float64, mesh.field_elems, "prim"), float(cfl),
                            _dev(d_dt, torch.float64, 1, "d_dt"), C.byref(h) if host else None, _stream(stream)))
    return h.value if host else None


def rk2_step(mesh, d_dt, cons0, cons, prim, mask, stream=None):
    n = mesh.field_elems
    _check(lib().phx_rk2_step(mesh.handle, _dev(d_dt, torch.float64, 1, "d_dt"), _dev(cons0, torch.float64, n, "cons0"),
                              _dev(cons, torch.float64, n, "cons"), _dev(prim, torch.float64, n, "prim"),
                              _dev(mask, torch.uint8, mesh.mask_elems, "mask"), _stream(stream)))


def rk2_step_cfl(mesh, cfl, d_dt, cons0, cons, prim, mask, stream=None):
    """RK2 step with dt = d_dt[0], then d_dt[0] <- the CFL time step of the new state (reduction fused into stage 2)."""
    n = mesh.field_elems
    _check(lib().phx_rk2_step_cfl(mesh.handle, float(cfl), _dev(d_dt, torch.float64, 1, "d_dt"), _dev(cons0, torch.float64, n, "cons0"),
                                  _dev(cons, torch.float64, n, "cons"), _dev(prim, torch.float64, n, "prim"),
                                  _dev(mask, torch.uint8, mesh.mask_elems, "mask"), _stream(stream)))


def evolve_device(mesh, nsteps, cfl, d_dt, cons0, cons, prim, mask, d_t=None, stream=None):
    """`nsteps` RK2 steps with dt kept on the device (= nsteps x rk2_step_cfl, replayed from a CUDA graph for nsteps >= 2).
    d_t: optional 1-element CUDA fp64 tensor accumulating the elapsed time."""
    n = mesh.field_elems
    _check(lib().phx_evolve_device(mesh.handle, int(nsteps), float(cfl), _dev(d_dt, torch.float64, 1, "d_dt"),
                                   _dev(d_t, torch.float64, 1, "d_t") if d_t is not None else None,
                                   _dev(cons0, torch.float64, n, "cons0"), _dev(cons, torch.float64, n, "cons"),
                                   _dev(prim, torch.float64, n, "prim"), _dev(mask, torch.uint8, mesh.mask_elems, "mask"), _stream(stream)))


def _host(t, dtype, numel, name, nullable=False):
    if t is None and nullable:
        return None
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == dtype and t.is_contiguous() and t.numel() == numel):
        raise PhxError(EINVAL, f"{name}: need a contiguous host tensor of {dtype} with {numel} elements")
    return C.c_void_p(t.data_ptr())


def evolve_host(mesh, h_prim_in, nsteps, cfl, h_prim_out, h_cons_out=None, h_mask_out=None, stream=None):
    """HOST-buffer path: H2D of the primitives, prim->cons, `nsteps` RK2 steps with the CFL time step kept
    on the device, D2H of the results.  Returns the elapsed simulation time."""
    n = mesh.field_elems
    t = C.c_double(0.0)
    _check(lib().phx_evolve_host(mesh.handle, _host(h_prim_in, torch.float64, n, "h_prim_in"), int(nsteps), float(cfl),
                                 _host(h_prim_out, torch.float64, n, "h_prim_out"),
                                 _host(h_cons_out, torch.float64, n, "h_cons_out", True),
                                 _host(h_mask_out, torch.uint8, mesh.mask_elems, "h_mask_out", True), C.byref(t), _stream(stream)))
    return t.value


def debug_fp64_peak(min_seconds=0.5, stream=None):
    """Measured peak of the fp64 pipe: (DFMA thread-instructions per second sustained over min_seconds, the same for the short
    calibration launch before it, milliseconds of the timed launch, SM count)."""
    r, rb, ms, nsm = C.c_double(), C.c_double(), C.c_double(), C.c_int()
    _check(lib().phx_debug_fp64_peak(float(min_seconds), C.byref(r), C.byref(rb), C.byref(ms), C.byref(nsm), _stream(stream)))
    return r.value, rb.value, ms.value, nsm.value


def count_masked(mesh, mask, bits, d_count=None, stream=None):
    """Number of interior cells whose mask carries any of `bits` (synchronises the stream)."""
    if d_count is None:
        d_count = torch.zeros(1, dtype=torch.int64, device="cuda")
    h = C.c_ulonglong(0)
    _check(lib().phx_count_masked(mesh.handle, _dev(mask, torch.uint8, mesh.mask_elems, "mask"), int(bits),
                                  _dev(d_count, torch.int64, 1, "d_count"), C.byref(h), _stream(stream)))
    return h.value
