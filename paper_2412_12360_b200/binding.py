"""Thin ctypes binding of include/fdtd.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; this module converts Python /
PyTorch objects to the plain pointers and structs the ABI takes.  PyTorch is used only for
device allocation and the current stream.  There is NO CPU fallback: if the shared library is
missing or cannot be loaded, importing this module raises.

The functions fdtd_create_grid / fdtd_forward / fdtd_backward / fdtd_destroy / fdtd_last_error /
fdtd_get_info / fdtd_version / fdtd_forward_host / fdtd_backward_host mirror the C entry points
one to one; `Grid` is a small convenience wrapper used by the tests and bench.py.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional, Sequence

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libfdtd_b200.so"

FDTD_OK, FDTD_EINVAL, FDTD_ENOMEM, FDTD_ECUDA, FDTD_ESTATE = 0, -1, -2, -3, -4
FDTD_PATH_AUTO, FDTD_PATH_GENERIC, FDTD_PATH_FUSED = 0, 1, 2
FDTD_FLAG_HOST_STAGING, FDTD_FLAG_RECORDER_FP16, FDTD_FLAG_ANISO_EPS = 1, 2, 4
PARTITION_NAMES = {0: "none (generic kernels)", 1: "contiguous runs", 2: "lock-step runs", 3: "waves of whole columns + levelled pool"}


class fdtd_grid_desc(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("courant", C.c_float),
                ("periodic", C.c_int32), ("pml_cells", C.c_int32),
                ("pml_m", C.c_float), ("pml_sigma_scale", C.c_float), ("pml_kappa_max", C.c_float),
                ("pml_alpha_max", C.c_float), ("pml_alpha_m", C.c_float), ("pml_eps_bg", C.c_float),
                ("max_steps", C.c_int32), ("record", C.c_int32),
                ("grad_lo", C.c_int32 * 3), ("grad_hi", C.c_int32 * 3),
                ("path", C.c_int32), ("flags", C.c_int32),
                ("z_global", C.c_int32), ("z_offset", C.c_int32), ("z_ghost_lo", C.c_int32), ("z_ghost_hi", C.c_int32),
                ("checkpoint_every", C.c_int32), ("reserved", C.c_int32 * 1)]


class fdtd_source(C.Structure):
    _fields_ = [("component", C.c_int32), ("lo", C.c_int32 * 3), ("hi", C.c_int32 * 3),
                ("profile", C.c_void_p), ("waveform", C.c_void_p)]


class fdtd_detector(C.Structure):
    _fields_ = [("component_mask", C.c_int32), ("lo", C.c_int32 * 3), ("hi", C.c_int32 * 3),
                ("n_freq", C.c_int32), ("omega", C.POINTER(C.c_float)), ("phasor", C.c_void_p)]


class fdtd_time_detector(C.Structure):
    _fields_ = [("kind", C.c_int32), ("component_mask", C.c_int32), ("lo", C.c_int32 * 3), ("hi", C.c_int32 * 3),
                ("stride", C.c_int32), ("out", C.c_void_p)]


FDTD_TD_SNAPSHOT, FDTD_TD_ENERGY = 0, 1


class fdtd_grid_info(C.Structure):
    _fields_ = [("path", C.c_int32), ("tile_x", C.c_int32), ("tile_y", C.c_int32), ("tile_z", C.c_int32),
                ("kernel_launches", C.c_int64), ("recorder_bytes", C.c_int64), ("scratch_bytes", C.c_int64),
                ("record_floats_per_step", C.c_int64), ("pipelined_inverse_ctas", C.c_int64),
                ("fused_step_launches", C.c_int64), ("fused_inverse_launches", C.c_int64), ("partition", C.c_int64)]


FDTD_PROF_CLASSES = 16


class fdtd_profile(C.Structure):
    _fields_ = [("n_classes", C.c_int32), ("reserved", C.c_int32),
                ("name", (C.c_char * 32) * FDTD_PROF_CLASSES),
                ("launches", C.c_int64 * FDTD_PROF_CLASSES), ("total_ms", C.c_double * FDTD_PROF_CLASSES)]


EXPORTS = ("fdtd_grad_rho", "fdtd_set_profiling", "fdtd_get_profile", "fdtd_create_grid", "fdtd_forward", "fdtd_backward", "fdtd_destroy", "fdtd_last_error",
           "fdtd_get_info", "fdtd_version", "fdtd_forward_host", "fdtd_backward_host", "fdtd_debug_partition",
           "fdtd_forward_td", "fdtd_backward_td", "fdtd_flux", "fdtd_flux_vjp", "fdtd_tfsf_plane",
           "fdtd_forward_range", "fdtd_backward_range", "fdtd_halo_export", "fdtd_halo_import",
           "fdtd_halo_volumes", "fdtd_halo_attach", "fdtd_halo_flags", "fdtd_halo_attach_flags", "fdtd_halo_sync_error", "fdtd_ipc_export", "fdtd_ipc_open", "fdtd_ipc_close", "fdtd_backward_mu", "fdtd_set_conductivity", "fdtd_probe_bandwidth", "fdtd_flux_static")


def _load():
    if not LIB_PATH.exists():
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2412_12360_b200.build` "
            "(there is no CPU fallback)")
    L = C.CDLL(str(LIB_PATH))
    vp, i32 = C.c_void_p, C.c_int32
    L.fdtd_create_grid.restype = C.c_int
    L.fdtd_create_grid.argtypes = [C.POINTER(fdtd_grid_desc), C.POINTER(vp)]
    L.fdtd_forward.restype = C.c_int
    L.fdtd_forward.argtypes = [vp, vp, vp, vp, C.POINTER(fdtd_source), i32, C.POINTER(fdtd_detector), i32, i32, vp]
    L.fdtd_forward_td.restype = C.c_int
    L.fdtd_forward_td.argtypes = [vp, vp, vp, vp, C.POINTER(fdtd_source), i32, C.POINTER(fdtd_detector), i32,
                                  C.POINTER(fdtd_time_detector), i32, i32, vp]
    L.fdtd_backward_td.restype = C.c_int
    L.fdtd_backward_td.argtypes = [vp, vp, vp, vp, C.POINTER(fdtd_source), i32, C.POINTER(fdtd_detector), i32,
                                   C.POINTER(vp), C.POINTER(fdtd_time_detector), i32, C.POINTER(vp), vp, i32, vp, vp, vp]
    L.fdtd_forward_range.restype = C.c_int
    L.fdtd_forward_range.argtypes = [vp, vp, vp, vp, C.POINTER(fdtd_source), i32, C.POINTER(fdtd_detector), i32, i32, i32, i32, vp]
    L.fdtd_backward_range.restype = C.c_int
    L.fdtd_backward_range.argtypes = [vp, vp, vp, vp, C.POINTER(fdtd_source), i32, C.POINTER(fdtd_detector), i32,
                                      C.POINTER(vp), vp, i32, i32, i32, vp, vp, vp]
    L.fdtd_backward_mu.restype = C.c_int
    L.fdtd_backward_mu.argtypes = [vp, vp, vp, vp, C.POINTER(fdtd_source), i32, C.POINTER(fdtd_detector), i32,
                                   C.POINTER(vp), vp, i32, vp, vp, vp, vp]
    L.fdtd_set_conductivity.restype = C.c_int
    L.fdtd_set_conductivity.argtypes = [vp, vp]
    L.fdtd_halo_export.restype = C.c_int
    L.fdtd_halo_export.argtypes = [vp, vp, i32, i32, i32, vp, vp]
    L.fdtd_halo_import.restype = C.c_int
    L.fdtd_halo_import.argtypes = [vp, vp, i32, i32, i32, vp, vp]
    L.fdtd_halo_volumes.restype = C.c_int
    L.fdtd_halo_volumes.argtypes = [vp, vp, i32, C.POINTER(vp), C.POINTER(vp)]
    L.fdtd_halo_attach.restype = C.c_int
    L.fdtd_halo_attach.argtypes = [vp, i32, i32, vp, vp, i32]
    L.fdtd_halo_flags.restype = C.c_int
    L.fdtd_halo_flags.argtypes = [vp, i32, C.POINTER(vp)]
    L.fdtd_halo_attach_flags.restype = C.c_int
    L.fdtd_halo_attach_flags.argtypes = [vp, i32, i32, vp]
    L.fdtd_halo_sync_error.restype = C.c_int
    L.fdtd_halo_sync_error.argtypes = [vp, C.POINTER(i32)]
    L.fdtd_ipc_export.restype = C.c_int
    L.fdtd_ipc_export.argtypes = [vp, C.c_char_p, C.POINTER(C.c_int64)]
    L.fdtd_ipc_open.restype = C.c_int
    L.fdtd_ipc_open.argtypes = [C.c_char_p, C.c_int64, C.POINTER(vp)]
    L.fdtd_ipc_close.restype = C.c_int
    L.fdtd_ipc_close.argtypes = [vp, C.c_int64]
    L.fdtd_flux.restype = C.c_int
    L.fdtd_flux.argtypes = [vp, C.POINTER(fdtd_detector), vp, i32, i32, vp, vp]
    L.fdtd_flux_vjp.restype = C.c_int
    L.fdtd_flux_vjp.argtypes = [vp, C.POINTER(fdtd_detector), vp, i32, i32, vp, vp, vp]
    L.fdtd_tfsf_plane.restype = C.c_int
    L.fdtd_tfsf_plane.argtypes = [C.c_float, C.c_float, C.c_float, i32, i32, i32, i32, vp, vp, vp,
                                  C.POINTER(i32), C.POINTER(i32), vp]
    L.fdtd_backward.restype = C.c_int
    L.fdtd_backward.argtypes = [vp, vp, vp, vp, C.POINTER(fdtd_source), i32, C.POINTER(fdtd_detector), i32,
                                C.POINTER(vp), vp, i32, vp, vp, vp]
    L.fdtd_destroy.restype = C.c_int
    L.fdtd_destroy.argtypes = [vp]
    L.fdtd_last_error.restype = C.c_char_p
    L.fdtd_last_error.argtypes = []
    L.fdtd_get_info.restype = C.c_int
    L.fdtd_get_info.argtypes = [vp, C.POINTER(fdtd_grid_info)]
    L.fdtd_version.restype = C.c_char_p
    L.fdtd_grad_rho.restype = C.c_int
    L.fdtd_grad_rho.argtypes = [vp, vp, vp, C.c_float, C.POINTER(i32), C.POINTER(i32), vp, vp]
    L.fdtd_set_profiling.restype = C.c_int
    L.fdtd_set_profiling.argtypes = [vp, i32]
    L.fdtd_get_profile.restype = C.c_int
    L.fdtd_get_profile.argtypes = [vp, C.POINTER(fdtd_profile)]
    L.fdtd_forward_host.restype = C.c_int
    L.fdtd_forward_host.argtypes = L.fdtd_forward.argtypes
    L.fdtd_backward_host.restype = C.c_int
    L.fdtd_backward_host.argtypes = L.fdtd_backward.argtypes
    return L


_L = _load()


class FdtdError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"fdtd error {code}: {msg}")
        self.code = code


def fdtd_last_error() -> str:
    return _L.fdtd_last_error().decode()


def fdtd_version() -> str:
    return _L.fdtd_version().decode()


def fdtd_debug_partition(nx, ny, nz, d, tile_x, tile_y, n_cta, wy=1.0, wz=0.8, lockstep=True):
    """Host-only: the step kernels' work partition as a list of (cta, i0, j0, k0, k1) (include/fdtd.h)."""
    _L.fdtd_debug_partition.restype = C.c_int
    _L.fdtd_debug_partition.argtypes = [C.c_int32] * 7 + [C.c_double, C.c_double, C.c_int32, C.POINTER(C.c_int32), C.c_int32]
    n = _L.fdtd_debug_partition(nx, ny, nz, d, tile_x, tile_y, n_cta, wy, wz, int(bool(lockstep)), None, 0)
    if n < 0:
        raise FdtdError(n, fdtd_last_error())
    buf = (C.c_int32 * (5 * n))()
    _L.fdtd_debug_partition(nx, ny, nz, d, tile_x, tile_y, n_cta, wy, wz, int(bool(lockstep)), buf, n)
    return [tuple(buf[5 * q:5 * q + 5]) for q in range(n)]


def _check(rc: int):
    if rc != 0:
        raise FdtdError(rc, fdtd_last_error())


def fdtd_create_grid(desc: fdtd_grid_desc) -> C.c_void_p:
    h = C.c_void_p()
    _check(_L.fdtd_create_grid(C.byref(desc), C.byref(h)))
    return h


def fdtd_destroy(grid) -> None:
    _check(_L.fdtd_destroy(grid))


def fdtd_get_info(grid) -> fdtd_grid_info:
    info = fdtd_grid_info()
    _check(_L.fdtd_get_info(grid, C.byref(info)))
    return info


def fdtd_grad_rho(grid, dL_dinv_eps, inv_eps, delta_eps, lo, hi, dL_drho, stream) -> None:
    lo_a, hi_a = (C.c_int32 * 3)(*lo), (C.c_int32 * 3)(*hi)
    _check(_L.fdtd_grad_rho(grid, _ptr(dL_dinv_eps), _ptr(inv_eps), float(delta_eps), lo_a, hi_a, _ptr(dL_drho), stream))


def fdtd_set_profiling(grid, enable: bool) -> None:
    _check(_L.fdtd_set_profiling(grid, int(bool(enable))))


def fdtd_get_profile(grid) -> dict:
    """{kernel class: (launches, total_ms)} since profiling was enabled / last read."""
    p = fdtd_profile()
    _check(_L.fdtd_get_profile(grid, C.byref(p)))
    return {bytes(p.name[c]).split(b"\0")[0].decode(): (int(p.launches[c]), float(p.total_ms[c]))
            for c in range(p.n_classes) if p.launches[c]}


def _ptr(t) -> Optional[int]:
    """Device/host pointer of a torch tensor or numpy array (None passes through)."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        assert t.is_contiguous()
        return t.data_ptr()
    assert t.flags.c_contiguous
    return t.ctypes.data


def fdtd_forward(grid, fields, inv_eps, inv_mu, src, n_src, det, n_det, n_steps, stream) -> None:
    _check(_L.fdtd_forward(grid, _ptr(fields), _ptr(inv_eps), _ptr(inv_mu), src, n_src, det, n_det, n_steps, stream))


def fdtd_backward(grid, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, dL_dfields, n_steps,
                  dL_dinv_eps, dL_dfields0, stream) -> None:
    _check(_L.fdtd_backward(grid, _ptr(fields), _ptr(inv_eps), _ptr(inv_mu), src, n_src, det, n_det,
                            dL_dphasor, _ptr(dL_dfields), n_steps, _ptr(dL_dinv_eps), _ptr(dL_dfields0), stream))


def fdtd_forward_td(grid, fields, inv_eps, inv_mu, src, n_src, det, n_det, td, n_td, n_steps, stream) -> None:
    _check(_L.fdtd_forward_td(grid, _ptr(fields), _ptr(inv_eps), _ptr(inv_mu), src, n_src, det, n_det, td, n_td, n_steps, stream))


def fdtd_backward_td(grid, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, td, n_td, dL_dtd, dL_dfields,
                     n_steps, dL_dinv_eps, dL_dfields0, stream) -> None:
    _check(_L.fdtd_backward_td(grid, _ptr(fields), _ptr(inv_eps), _ptr(inv_mu), src, n_src, det, n_det, dL_dphasor,
                               td, n_td, dL_dtd, _ptr(dL_dfields), n_steps, _ptr(dL_dinv_eps), _ptr(dL_dfields0), stream))


def fdtd_forward_range(grid, fields, inv_eps, inv_mu, src, n_src, det, n_det, n_begin, n_end, n_total, stream) -> None:
    _check(_L.fdtd_forward_range(grid, _ptr(fields), _ptr(inv_eps), _ptr(inv_mu), src, n_src, det, n_det,
                                 int(n_begin), int(n_end), int(n_total), stream))


def fdtd_backward_range(grid, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, dL_dfields, n_hi, n_lo, n_total,
                        dL_dinv_eps, dL_dfields0, stream) -> None:
    _check(_L.fdtd_backward_range(grid, _ptr(fields), _ptr(inv_eps), _ptr(inv_mu), src, n_src, det, n_det, dL_dphasor,
                                  _ptr(dL_dfields), int(n_hi), int(n_lo), int(n_total), _ptr(dL_dinv_eps), _ptr(dL_dfields0), stream))


def fdtd_backward_mu(grid, fields, inv_eps, inv_mu, src, n_src, det, n_det, dL_dphasor, dL_dfields, n_steps,
                     dL_dinv_eps, dL_dinv_mu, dL_dfields0, stream) -> None:
    _check(_L.fdtd_backward_mu(grid, _ptr(fields), _ptr(inv_eps), _ptr(inv_mu), src, n_src, det, n_det, dL_dphasor,
                               _ptr(dL_dfields), n_steps, _ptr(dL_dinv_eps), _ptr(dL_dinv_mu), _ptr(dL_dfields0), stream))


def fdtd_probe_bandwidth(pattern, nx, ny, nz, tile_y, runs, unroll, blocks, threads, reps, vin, vout, stream) -> float:
    """GB/s of the 7-read / 6-write probe (include/fdtd.h); vin: 7 volumes, vout: 6 volumes (cuda tensors)."""
    _L.fdtd_probe_bandwidth.restype = C.c_int
    _L.fdtd_probe_bandwidth.argtypes = [C.c_int32] * 10 + [C.c_void_p, C.c_void_p, C.POINTER(C.c_double), C.c_void_p]
    out = C.c_double(0.0)
    _check(_L.fdtd_probe_bandwidth(pattern, nx, ny, nz, tile_y, runs, unroll, blocks, threads, reps, _ptr(vin), _ptr(vout),
                                   C.byref(out), stream))
    return out.value


def fdtd_halo_export(grid, fields, which, n, side, out, stream) -> None:
    _check(_L.fdtd_halo_export(grid, _ptr(fields), int(which), int(n), int(side), _ptr(out), stream))


def fdtd_halo_import(grid, fields, which, n, side, buf, stream) -> None:
    _check(_L.fdtd_halo_import(grid, _ptr(fields), int(which), int(n), int(side), _ptr(buf), stream))


def fdtd_halo_volumes(grid, fields, which):
    """(vol0, vol1): device addresses (int) of the two ping-pong volumes of the primal fields (which = 0) / cotangents (1)."""
    a, b = C.c_void_p(), C.c_void_p()
    _check(_L.fdtd_halo_volumes(grid, _ptr(fields), int(which), C.byref(a), C.byref(b)))
    return int(a.value), int(b.value)


def fdtd_halo_attach(grid, which, side, peer_vol0, peer_vol1, peer_nz) -> None:
    """peer_vol0 / peer_vol1: device addresses (int) of the neighbour's fdtd_halo_volumes, or None / None to detach."""
    _check(_L.fdtd_halo_attach(grid, int(which), int(side), C.c_void_p(peer_vol0), C.c_void_p(peer_vol1), int(peer_nz)))


def fdtd_halo_flags(grid, which) -> int:
    """Device address (int) of this grid's two ordering flags of `which`."""
    p = C.c_void_p()
    _check(_L.fdtd_halo_flags(grid, int(which), C.byref(p)))
    return int(p.value)


def fdtd_halo_attach_flags(grid, which, side, peer_flags) -> None:
    _check(_L.fdtd_halo_attach_flags(grid, int(which), int(side), C.c_void_p(peer_flags)))


def fdtd_halo_sync_error(grid) -> int:
    v = C.c_int32(0)
    _check(_L.fdtd_halo_sync_error(grid, C.byref(v)))
    return int(v.value)


def fdtd_ipc_export(dev_ptr: int):
    """(64-byte handle, offset) of a device address, to be opened by another process with fdtd_ipc_open."""
    h = C.create_string_buffer(64)
    off = C.c_int64(0)
    _check(_L.fdtd_ipc_export(C.c_void_p(dev_ptr), h, C.byref(off)))
    return h.raw, int(off.value)


def fdtd_ipc_open(handle: bytes, offset: int) -> int:
    p = C.c_void_p()
    _check(_L.fdtd_ipc_open(C.create_string_buffer(handle, 64), int(offset), C.byref(p)))
    return int(p.value)


def fdtd_ipc_close(dev_ptr: int, offset: int) -> None:
    _check(_L.fdtd_ipc_close(C.c_void_p(dev_ptr), int(offset)))


def fdtd_flux(grid, det, phasor, axis, interpolate, flux, stream) -> None:
    _check(_L.fdtd_flux(grid, det, _ptr(phasor), int(axis), int(bool(interpolate)), _ptr(flux), stream))


FDTD_FLUX_STATIC_MAX_CELLS = 4194304


def fdtd_flux_static(det, phasor, axis, interpolate, flux, stream) -> None:
    """fdtd_flux without a grid and without any device allocation (include/fdtd.h): scratch in a static __device__ array;
    planes of at most FDTD_FLUX_STATIC_MAX_CELLS cells.  det: a fdtd_detector struct (HOST); phasor, flux: cuda tensors."""
    _L.fdtd_flux_static.restype = C.c_int
    _L.fdtd_flux_static.argtypes = [C.POINTER(fdtd_detector), C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
    _check(_L.fdtd_flux_static(det, _ptr(phasor), int(axis), int(bool(interpolate)), _ptr(flux), stream))


def fdtd_flux_vjp(grid, det, phasor, axis, interpolate, dL_dflux, dL_dphasor, stream) -> None:
    _check(_L.fdtd_flux_vjp(grid, det, _ptr(phasor), int(axis), int(bool(interpolate)), _ptr(dL_dflux), _ptr(dL_dphasor), stream))


def fdtd_tfsf_plane(courant, eps_r, mu_r, axis, pol, direction, n_steps, base, wE, wH, stream):
    """Returns (h_component, h_plane_offset); wE / wH (device, n_steps floats) are written."""
    hc, off = C.c_int32(0), C.c_int32(0)
    _check(_L.fdtd_tfsf_plane(float(courant), float(eps_r), float(mu_r), int(axis), int(pol), int(direction), int(n_steps),
                              _ptr(base), _ptr(wE), _ptr(wH), C.byref(hc), C.byref(off), stream))
    return hc.value, off.value


def fdtd_forward_host(grid, h_fields, h_inv_eps, h_inv_mu, src, n_src, det, n_det, n_steps, stream) -> None:
    _check(_L.fdtd_forward_host(grid, _ptr(h_fields), _ptr(h_inv_eps), _ptr(h_inv_mu), src, n_src, det, n_det,
                                n_steps, stream))


def fdtd_backward_host(grid, h_fields, h_inv_eps, h_inv_mu, src, n_src, det, n_det, h_dL_dphasor, h_dL_dfields,
                       n_steps, h_dL_dinv_eps, h_dL_dfields0, stream) -> None:
    _check(_L.fdtd_backward_host(grid, _ptr(h_fields), _ptr(h_inv_eps), _ptr(h_inv_mu), src, n_src, det, n_det,
                                 h_dL_dphasor, _ptr(h_dL_dfields), n_steps, _ptr(h_dL_dinv_eps),
                                 _ptr(h_dL_dfields0), stream))


# --------------------------------------------------------------------------------------------
# convenience wrapper (marshalling only)
# --------------------------------------------------------------------------------------------
def make_desc(nx, ny, nz, courant, periodic=False, pml_cells=0, pml_m=0.0, pml_sigma_scale=0.0,
              pml_kappa_max=0.0, pml_alpha_max=0.0, pml_alpha_m=0.0, pml_eps_bg=0.0, max_steps=0,
              record=False, grad_lo=None, grad_hi=None, path=FDTD_PATH_AUTO, flags=0,
              z_global=0, z_offset=0, z_ghost_lo=0, z_ghost_hi=0, checkpoint_every=0) -> fdtd_grid_desc:
    d = fdtd_grid_desc()
    d.nx, d.ny, d.nz, d.courant = nx, ny, nz, courant
    d.periodic, d.pml_cells = int(bool(periodic)), pml_cells
    d.pml_m, d.pml_sigma_scale, d.pml_kappa_max = pml_m, pml_sigma_scale, pml_kappa_max
    d.pml_alpha_max, d.pml_alpha_m, d.pml_eps_bg = pml_alpha_max, pml_alpha_m, pml_eps_bg
    d.max_steps, d.record, d.path, d.flags = max_steps, int(record), path, int(flags)
    d.z_global, d.z_offset, d.z_ghost_lo, d.z_ghost_hi = int(z_global), int(z_offset), int(z_ghost_lo), int(z_ghost_hi)
    d.checkpoint_every = int(checkpoint_every)
    if grad_lo is not None:
        d.grad_lo[:] = list(grad_lo)
        d.grad_hi[:] = list(grad_hi)
    return d


class Grid:
    """Owns one fdtd_grid handle; marshals workloads.Source / workloads.Detector style objects."""

    def __init__(self, **kw):
        import torch  # device memory + streams only
        self.torch = torch
        self.desc = make_desc(**kw)
        self.shape = (self.desc.nz, self.desc.ny, self.desc.nx)
        self.h = fdtd_create_grid(self.desc)
        self._keep = []

    def close(self):
        if getattr(self, "h", None):
            fdtd_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self) -> fdtd_grid_info:
        return fdtd_get_info(self.h)

    # -- marshalling -----------------------------------------------------------------------------
    def _dev(self, a):
        torch = self.torch
        if a is None:
            return None
        if isinstance(a, torch.Tensor):
            return a.to(device="cuda", dtype=torch.float32).contiguous()
        return torch.as_tensor(a, dtype=torch.float32).contiguous().cuda()

    def marshal_sources(self, sources, host=False):
        n = len(sources)
        arr = (fdtd_source * max(n, 1))()
        keep = []
        for s, q in zip(arr, sources):
            s.component = int(q.component)
            s.lo[:] = list(q.lo)
            s.hi[:] = list(q.hi)
            if host:
                import numpy as np
                prof = None if q.profile is None else np.ascontiguousarray(q.profile, dtype=np.float32)
                wav = np.ascontiguousarray(q.waveform, dtype=np.float32)
            else:
                prof, wav = self._dev(q.profile), self._dev(q.waveform)
            keep += [prof, wav]
            s.profile = _ptr(prof)
            s.waveform = _ptr(wav)
        return arr, n, keep

    def marshal_detectors(self, detectors, phasors):
        n = len(detectors)
        arr = (fdtd_detector * max(n, 1))()
        keep = []
        for idx, (s, q) in enumerate(zip(arr, detectors)):
            s.component_mask = int(q.component_mask)
            s.lo[:] = list(q.lo)
            s.hi[:] = list(q.hi)
            om = (C.c_float * len(q.omega))(*[float(o) for o in q.omega])
            keep.append(om)
            s.n_freq = len(q.omega)
            s.omega = C.cast(om, C.POINTER(C.c_float))
            s.phasor = None if phasors is None else _ptr(phasors[idx])
        return arr, n, keep

    def marshal_time_detectors(self, tdets, outs):
        n = len(tdets)
        arr = (fdtd_time_detector * max(n, 1))()
        for idx, (s, q) in enumerate(zip(arr, tdets)):
            s.kind = FDTD_TD_ENERGY if q.kind == "energy" else FDTD_TD_SNAPSHOT
            s.component_mask = int(q.component_mask)
            s.lo[:] = list(q.lo)
            s.hi[:] = list(q.hi)
            s.stride = int(q.stride)
            s.out = None if outs is None else _ptr(outs[idx])
        return arr, n

    def stream(self):
        return C.c_void_p(self.torch.cuda.current_stream().cuda_stream)

    def set_conductivity(self, sigma):
        """N4: normalised electric conductivity per voxel (cuda tensor / array) or None; kept alive by this object."""
        self._sigma = self._dev(sigma)
        _check(_L.fdtd_set_conductivity(self.h, _ptr(self._sigma)))

    # -- N2: flux from phasors, TFSF plane source ------------------------------------------------
    def flux(self, det, phasor, axis, interpolate=False):
        darr, nd, k = self.marshal_detectors([det], None)
        out = self.torch.empty(len(det.omega), dtype=self.torch.float32, device="cuda")
        fdtd_flux(self.h, darr, phasor, axis, interpolate, out, self.stream())
        return out

    def flux_vjp(self, det, phasor, axis, interpolate, dL_dflux):
        darr, nd, k = self.marshal_detectors([det], None)
        out = self.torch.empty_like(phasor)
        fdtd_flux_vjp(self.h, darr, phasor, axis, interpolate, self._dev(dL_dflux), out, self.stream())
        return out

    def tfsf_plane(self, eps_r, mu_r, axis, pol, direction, base):
        """(wE, wH, h_component, h_plane_offset) of a one-directional plane source; wE / wH are cuda tensors."""
        b = self._dev(base)
        wE, wH = self.torch.empty_like(b), self.torch.empty_like(b)
        hc, off = fdtd_tfsf_plane(self.desc.courant, eps_r, mu_r, axis, pol, direction, b.numel(), b, wE, wH, self.stream())
        return wE, wH, hc, off

    # -- device entry points ---------------------------------------------------------------------
    def forward(self, fields, inv_eps, inv_mu=None, sources=(), detectors=(), n_steps=0, phasors=None, time_detectors=()):
        """fields: cuda float32 [6,nz,ny,nx], updated in place.  Returns the phasor tensors; the outputs of the
        time-domain detectors are left in self.time_outputs."""
        torch = self.torch
        if phasors is None:
            phasors = [torch.zeros(d.phasor_shape, dtype=torch.float32, device="cuda") for d in detectors]
        sarr, ns, k1 = self.marshal_sources(sources)
        darr, nd, k2 = self.marshal_detectors(detectors, phasors)
        if time_detectors:
            self.time_outputs = [torch.zeros(t.out_shape(int(n_steps)), dtype=torch.float32, device="cuda") for t in time_detectors]
            tarr, nt = self.marshal_time_detectors(time_detectors, self.time_outputs)
            fdtd_forward_td(self.h, fields, inv_eps, inv_mu, sarr, ns, darr, nd, tarr, nt, int(n_steps), self.stream())
        else:
            self.time_outputs = []
            fdtd_forward(self.h, fields, inv_eps, inv_mu, sarr, ns, darr, nd, int(n_steps), self.stream())
        self._keep = [k1, k2, sarr, darr]
        return phasors

    def backward(self, fields, inv_eps, inv_mu=None, sources=(), detectors=(), dL_dphasor=None,
                 dL_dfields=None, n_steps=0, want_dL_dfields0=False, out=None, want_grad=True, time_detectors=(), dL_dtime=None, grad_mu=None):
        """want_grad=False: adjoint sweep only (dL_dinv_eps = NULL): returns (None, cotangent of state 0)."""
        torch = self.torch
        sarr, ns, k1 = self.marshal_sources(sources)
        darr, nd, k2 = self.marshal_detectors(detectors, None)
        cot = None
        if dL_dphasor is not None:
            cot = (C.c_void_p * max(nd, 1))()
            for i, G in enumerate(dL_dphasor):
                cot[i] = _ptr(G)
        gshape = ((3,) + self.shape) if (self.desc.flags & FDTD_FLAG_ANISO_EPS) else self.shape
        g = None if not want_grad else (out if out is not None else torch.empty(gshape, dtype=torch.float32, device="cuda"))
        lam0 = torch.empty((6,) + self.shape, dtype=torch.float32, device="cuda") if (want_dL_dfields0 or not want_grad) else None
        if grad_mu is not None:          # N4: dL/d inv_mu into the caller's volume
            fdtd_backward_mu(self.h, fields, inv_eps, inv_mu, sarr, ns, darr, nd, cot, dL_dfields, int(n_steps),
                             g, grad_mu, lam0, self.stream())
        elif time_detectors:
            tarr, nt = self.marshal_time_detectors(time_detectors, None)
            tcot = (C.c_void_p * max(nt, 1))()
            for i, G in enumerate(dL_dtime or []):
                tcot[i] = _ptr(G)
            fdtd_backward_td(self.h, fields, inv_eps, inv_mu, sarr, ns, darr, nd, cot, tarr, nt, tcot, dL_dfields,
                             int(n_steps), g, lam0, self.stream())
        else:
            fdtd_backward(self.h, fields, inv_eps, inv_mu, sarr, ns, darr, nd, cot, dL_dfields, int(n_steps),
                          g, lam0, self.stream())
        self._keep = [k1, k2, sarr, darr, cot, dL_dphasor, dL_dtime]
        return g, lam0
