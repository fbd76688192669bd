"""Thin ctypes binding of the C-ABI in include/gx.h -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libgx.so; this module never computes.
PyTorch is used by callers for device memory and streams; tensors are passed as raw pointers.
The functions carry the names of the C entry points.  If libgx.so is missing, loading fails loudly
(there is no CPU fallback).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("GX_LIBRARY_PATH") or os.path.join(_HERE, "libgx.so")

GX_OK, GX_ERR_ARG, GX_ERR_STATE, GX_ERR_UNSUPPORTED, GX_ERR_CUDA, GX_ERR_ALLOC = 0, -1, -2, -3, -4, -5
(GX_Q_NAKX, GX_Q_NAKY, GX_Q_NJ, GX_Q_G_ELEMS, GX_Q_PHI_ELEMS, GX_Q_WORKSPACE_BYTES,
 GX_Q_LAUNCHES_PER_NL, GX_Q_LAUNCHES_PER_RHS, GX_Q_NL_FLOPS, GX_Q_NL_BYTES, GX_Q_KERNEL_FAMILY) = range(11)
FAMILY_NAMES = {0: "scalar", 3: "row", 5: "rx", 6: "rxp", 7: "rxw"}

EXPORTED = ["gx_grid_create", "gx_grid_destroy", "gx_box_set", "gx_species_set", "gx_adiabatic_set",
            "gx_dissipation_set", "gx_boundary_set", "gx_damping_set", "gx_geometry_set", "gx_nonlinear_rhs", "gx_nonlinear_rhs_em", "gx_field_solve_em", "gx_nonlinear_rhs_host",
            "gx_field_solve", "gx_rhs", "gx_linear_rhs", "gx_linear_rhs_static", "gx_ssprk3_step", "gx_query", "gx_export_maps",
            "gx_export_tables", "gx_profile_set", "gx_profile_get", "gx_last_error", "gx_ubench_fp32", "gx_ubench_dft16"]

_lib = None


class GxError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"gx error {code}: {msg}")
        self.code = code


def load():
    """dlopen libgx.so (built in-tree by build.py) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(f"{LIB_PATH} not built: run `python -m paper_2209_06731_b200.build` "
                                "(the CUDA extension is required; there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, dp, i, d = C.c_void_p, C.POINTER(C.c_double), C.c_int, C.c_double
    lib.gx_grid_create.argtypes = [i, i, i, i, i, i, C.POINTER(vp)]
    lib.gx_grid_destroy.argtypes = [vp]
    lib.gx_box_set.argtypes = [vp, d, d, d]
    lib.gx_species_set.argtypes = [vp, i, d, d, d, d, d, d, d]
    lib.gx_adiabatic_set.argtypes = [vp, i, d]
    lib.gx_dissipation_set.argtypes = [vp, d, i, d]
    lib.gx_boundary_set.argtypes = [vp, i]
    lib.gx_damping_set.argtypes = [vp, d, d]
    lib.gx_geometry_set.argtypes = [vp] + [dp] * 10 + [d]
    lib.gx_nonlinear_rhs.argtypes = [vp, vp, vp, vp, vp]
    lib.gx_nonlinear_rhs_host.argtypes = [vp, vp, vp, vp, vp]
    lib.gx_nonlinear_rhs_em.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.gx_field_solve_em.argtypes = [vp, vp, d, vp, vp, vp, vp]
    lib.gx_field_solve.argtypes = [vp, vp, vp, vp]
    lib.gx_rhs.argtypes = [vp, vp, vp, vp]
    lib.gx_linear_rhs.argtypes = [vp, vp, vp, vp, vp]
    lib.gx_linear_rhs_static.argtypes = [vp, vp, vp, vp, vp]
    lib.gx_ssprk3_step.argtypes = [vp, vp, d, vp]
    lib.gx_query.argtypes = [vp, i, C.POINTER(C.c_longlong)]
    lib.gx_export_maps.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.gx_export_tables.argtypes = [vp, vp, vp, vp]
    lib.gx_profile_set.argtypes = [vp, i]
    lib.gx_profile_get.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
    lib.gx_last_error.argtypes = [vp]
    lib.gx_last_error.restype = C.c_char_p
    lib.gx_ubench_fp32.argtypes = [i, i, i, i, dp, dp]
    lib.gx_ubench_dft16.argtypes = [i, i, i, i, dp, dp]
    for name in EXPORTED:
        if name != "gx_last_error":
            getattr(lib, name).restype = i
    _lib = lib
    return lib


def _check(h, rc):
    if rc != GX_OK:
        msg = load().gx_last_error(h).decode() if h else ""
        raise GxError(rc, msg)


def _dptr(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64).ctypes.data_as(C.POINTER(C.c_double))


# ---- C entry points, same names -------------------------------------------------------------
def gx_grid_create(Nx, Ny, Nz, Nl, Nm, Ns):
    h = C.c_void_p()
    rc = load().gx_grid_create(Nx, Ny, Nz, Nl, Nm, Ns, C.byref(h))
    if rc != GX_OK:
        msg = load().gx_last_error(h).decode() if h else "gx_grid_create failed"
        if h:
            load().gx_grid_destroy(h)
        raise GxError(rc, msg)
    return h


def gx_grid_destroy(h):
    _check(None, load().gx_grid_destroy(h))


def gx_box_set(h, dky, dkx, shat):
    _check(h, load().gx_box_set(h, dky, dkx, shat))


def gx_species_set(h, s, Z, mass, temp, dens, tprim=0.0, fprim=0.0, nu_ss=0.0):
    _check(h, load().gx_species_set(h, s, Z, mass, temp, dens, tprim, fprim, nu_ss))


def gx_adiabatic_set(h, enabled, tau_fac=1.0):
    _check(h, load().gx_adiabatic_set(h, int(enabled), tau_fac))


def gx_boundary_set(h, linked):
    _check(h, load().gx_boundary_set(h, int(linked)))


def gx_damping_set(h, A, width_fraction=0.125):
    _check(h, load().gx_damping_set(h, A, width_fraction))


def gx_dissipation_set(h, D_hyper, n_hyper, f_hyp):
    _check(h, load().gx_dissipation_set(h, D_hyper, n_hyper, f_hyp))


def gx_geometry_set(h, bmag, gds2, gds21, gds22, gbdrift=None, gbdrift0=None, cvdrift=None, cvdrift0=None,
                    bgrad=None, jacobian=None, gradpar=1.0):
    arrs = [_dptr(a) for a in (bmag, gds2, gds21, gds22, gbdrift, gbdrift0, cvdrift, cvdrift0, bgrad, jacobian)]
    _check(h, load().gx_geometry_set(h, *arrs, gradpar))


def gx_nonlinear_rhs(h, g_ptr, phi_ptr, out_ptr, stream=0):
    _check(h, load().gx_nonlinear_rhs(h, g_ptr, phi_ptr, out_ptr, stream))


def gx_nonlinear_rhs_em(h, g_ptr, phi_ptr, apar_ptr, bpar_ptr, out_ptr, stream=0):
    _check(h, load().gx_nonlinear_rhs_em(h, g_ptr, phi_ptr, apar_ptr, bpar_ptr, out_ptr, stream))


def gx_field_solve_em(h, g_ptr, beta, phi_ptr, apar_ptr, bpar_ptr, stream=0):
    _check(h, load().gx_field_solve_em(h, g_ptr, float(beta), phi_ptr, apar_ptr, bpar_ptr, stream))


def gx_nonlinear_rhs_host(h, g_ptr, phi_ptr, out_ptr, stream=0):
    _check(h, load().gx_nonlinear_rhs_host(h, g_ptr, phi_ptr, out_ptr, stream))


def gx_field_solve(h, g_ptr, phi_ptr, stream=0):
    _check(h, load().gx_field_solve(h, g_ptr, phi_ptr, stream))


def gx_rhs(h, g_ptr, out_ptr, stream=0):
    _check(h, load().gx_rhs(h, g_ptr, out_ptr, stream))


def gx_linear_rhs(h, g_ptr, phi_ptr, out_ptr, stream=0):
    _check(h, load().gx_linear_rhs(h, g_ptr, phi_ptr, out_ptr, stream))


def gx_linear_rhs_static(h, g_ptr, phi_ptr, out_ptr, stream=0):
    _check(h, load().gx_linear_rhs_static(h, g_ptr, phi_ptr, out_ptr, stream))


def gx_ssprk3_step(h, g_ptr, dt, stream=0):
    _check(h, load().gx_ssprk3_step(h, g_ptr, float(dt), stream))


def gx_query(h, what):
    v = C.c_longlong()
    _check(h, load().gx_query(h, what, C.byref(v)))
    return v.value


def gx_export_maps(h):
    nakx, naky, nj = gx_query(h, GX_Q_NAKX), gx_query(h, GX_Q_NAKY), gx_query(h, GX_Q_NJ)
    return _export_maps(h, nakx, naky, nj)


def _export_maps(h, nakx, naky, nj, Nx=None, Ny=None):
    kx, ky, pr = np.zeros(nakx, np.int32), np.zeros(naky, np.int32), np.zeros(nakx, np.int32)
    xj, wj = np.zeros(nj), np.zeros(nj)
    mask = None
    if Nx is not None:
        mask = np.zeros((Nx, Ny // 2 + 1), np.uint8)
    _check(h, load().gx_export_maps(h, kx.ctypes.data, ky.ctypes.data, pr.ctypes.data,
                                    None if mask is None else mask.ctypes.data, xj.ctypes.data, wj.ctypes.data))
    return dict(kx_index=kx, ky_index=ky, pad_row=pr, mask=mask, lag_nodes=xj, lag_weights=wj)


def gx_export_tables(h, Nl, want_M_elems=0):
    nj = gx_query(h, GX_Q_NJ)
    T, Tinv = np.zeros((nj, Nl), np.float32), np.zeros((Nl, nj), np.float32)
    M = np.zeros(want_M_elems, np.float32) if want_M_elems else None
    _check(h, load().gx_export_tables(h, T.ctypes.data, Tinv.ctypes.data, None if M is None else M.ctypes.data))
    return T, Tinv, M


def gx_profile_set(h, enabled):
    _check(h, load().gx_profile_set(h, int(enabled)))


def gx_profile_get(h):
    """-> (ms[3] summed over the profiled calls: chi, bracket, laguerre-inverse; number of calls)"""
    ms = (C.c_double * 3)(0.0, 0.0, 0.0)
    n = C.c_longlong()
    _check(h, load().gx_profile_get(h, ms, C.byref(n)))
    return [ms[0], ms[1], ms[2]], n.value


UBENCH_KINDS = ["add.f32", "mul.f32", "fma.rn.f32", "add.f32x2", "mul.f32x2", "fma.rn.f32x2"]


def gx_ubench_fp32(kind, threads_per_block=512, blocks_per_sm=2, iters=4096):
    """-> (milliseconds, lane operations) of the FP32 pipe micro-benchmark (include/gx.h)."""
    ms, ops = C.c_double(), C.c_double()
    _check(None, load().gx_ubench_fp32(kind, threads_per_block, blocks_per_sm, iters, C.byref(ms), C.byref(ops)))
    return ms.value, ops.value


def gx_ubench_dft16(packed, threads_per_block=192, blocks_per_sm=2, iters=512):
    """-> (milliseconds, 16-point transforms done) of the register radix-16 micro-benchmark (include/gx.h)."""
    ms, n = C.c_double(), C.c_double()
    _check(None, load().gx_ubench_dft16(int(packed), threads_per_block, blocks_per_sm, iters, C.byref(ms), C.byref(n)))
    return ms.value, n.value


# ---- convenience wrapper (marshalling only) -------------------------------------------------------
class Grid:
    """Owns a gx_grid handle configured from an ``inputs.Config``; methods take torch CUDA tensors
    (complex64, contiguous) and pass their data pointers and the current stream to the C-ABI."""

    def __init__(self, cfg, geo=None, linked=False, damping=None):
        from . import inputs as I
        self.cfg = cfg
        self.geo = geo or I.geometry_arrays(cfg)
        self.h = gx_grid_create(cfg.Nx, cfg.Ny, cfg.Nz, cfg.Nl, cfg.Nm, cfg.Ns)
        gx_box_set(self.h, cfg.dky, cfg.dkx, cfg.shat)
        for s, sp in enumerate(cfg.species):
            gx_species_set(self.h, s, sp.Z, sp.mass, sp.temp, sp.dens, sp.tprim, sp.fprim, sp.nu_ss)
        gx_adiabatic_set(self.h, cfg.Ns == 1, cfg.tau_fac)
        gx_boundary_set(self.h, linked)
        if damping:
            gx_damping_set(self.h, damping["A"], damping.get("width_frac", 0.125))
        g = self.geo
        gx_geometry_set(self.h, g["bmag"], g["gds2"], g["gds21"], g["gds22"], g["gbdrift"], g["gbdrift0"],
                        g["cvdrift"], g["cvdrift0"], g["bgrad"], g["jacobian"], g["gradpar"])

    def close(self):
        if self.h is not None:
            gx_grid_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @staticmethod
    def _stream():
        import torch
        return torch.cuda.current_stream().cuda_stream

    def _chk(self, t, what, host=False):
        """Marshalling checks: dtype, contiguity, device and element count (GX_Q_G_ELEMS / GX_Q_PHI_ELEMS)."""
        import torch
        n = gx_query(self.h, GX_Q_G_ELEMS if what == "g" else GX_Q_PHI_ELEMS)
        if t.dtype != torch.complex64 or not t.is_contiguous() or t.numel() != n or (t.is_cuda == host):
            raise ValueError(f"{what}: expected a contiguous complex64 {'host' if host else 'CUDA'} tensor of {n} elements, "
                             f"got {t.dtype} {tuple(t.shape)} on {t.device}")
        return t.data_ptr()

    def nonlinear_rhs(self, g, phi, out):
        gx_nonlinear_rhs(self.h, self._chk(g, "g"), self._chk(phi, "phi"), self._chk(out, "g"), self._stream())
        return out

    def nonlinear_rhs_em(self, g, phi, apar, bpar, out):
        gx_nonlinear_rhs_em(self.h, self._chk(g, "g"), self._chk(phi, "phi"), self._chk(apar, "phi"), self._chk(bpar, "phi"),
                            self._chk(out, "g"), self._stream())
        return out

    def field_solve_em(self, g, beta, phi, apar, bpar):
        gx_field_solve_em(self.h, self._chk(g, "g"), beta, self._chk(phi, "phi"), self._chk(apar, "phi"), self._chk(bpar, "phi"),
                          self._stream())
        return phi, apar, bpar

    def nonlinear_rhs_host(self, g_host, phi_host, out_host):
        gx_nonlinear_rhs_host(self.h, self._chk(g_host, "g", True), self._chk(phi_host, "phi", True),
                              self._chk(out_host, "g", True), self._stream())
        return out_host

    def field_solve(self, g, phi):
        gx_field_solve(self.h, self._chk(g, "g"), self._chk(phi, "phi"), self._stream())
        return phi

    def rhs(self, g, out):
        gx_rhs(self.h, self._chk(g, "g"), self._chk(out, "g"), self._stream())
        return out

    def linear_rhs(self, g, phi, out):
        gx_linear_rhs(self.h, self._chk(g, "g"), self._chk(phi, "phi"), self._chk(out, "g"), self._stream())
        return out

    def linear_rhs_static(self, g, phi, out):
        """gx_linear_rhs with its workspace in the library's static device array (no allocation in the call)."""
        gx_linear_rhs_static(self.h, self._chk(g, "g"), self._chk(phi, "phi"), self._chk(out, "g"), self._stream())
        return out

    def ssprk3_step(self, g, dt):
        gx_ssprk3_step(self.h, self._chk(g, "g"), dt, self._stream())
        return g

    def export_maps(self):
        c = self.cfg
        return _export_maps(self.h, c.nakx, c.naky, c.nj, c.Nx, c.Ny)

    def query(self, what):
        return gx_query(self.h, what)
