"""ctypes wrapper around oracle/fdtd_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
leg may import this module.  It imports nothing from paper_2412_12360_b200 and shares
no code with the CUDA path.  Sources / detectors are duck-typed: any object with the
attributes (component, lo, hi, profile, waveform) / (component_mask, lo, hi, omega).

Passages followed: PAPER.md Eq. 1-2 (L64-66), L68-72, L80-84; readings R1..R22 in
DESIGN.md section 3.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_BUILD = _HERE / "build"
_SRC = _HERE / "fdtd_oracle.c"


def build(force: bool = False) -> dict:
    """Compile the oracle twice (fp64 parity reference, fp32 timed baseline)."""
    _BUILD.mkdir(exist_ok=True)
    out = {}
    for tag, real in (("f64", "double"), ("f32", "float")):
        so = _BUILD / f"liborc_{tag}.so"
        if force or not so.exists() or so.stat().st_mtime < _SRC.stat().st_mtime:
            tmp = so.with_suffix(f".tmp{os.getpid()}.so")
            cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp",
                   f"-DREAL={real}", str(_SRC), "-o", str(tmp), "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, so)
        out[tag] = so
    return out


class _Desc(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("periodic", C.c_int), ("d", C.c_int),
                ("S", C.c_double), ("m", C.c_double), ("sigma_max", C.c_double),
                ("kappa_max", C.c_double), ("alpha_max", C.c_double), ("alpha_m", C.c_double)]


class _Source(C.Structure):
    _fields_ = [("comp", C.c_int), ("lo", C.c_int * 3), ("hi", C.c_int * 3),
                ("profile", C.c_void_p), ("waveform", C.c_void_p)]


class _TDetector(C.Structure):
    _fields_ = [("kind", C.c_int), ("mask", C.c_int), ("lo", C.c_int * 3), ("hi", C.c_int * 3),
                ("stride", C.c_int), ("out", C.c_void_p)]


class _Detector(C.Structure):
    _fields_ = [("mask", C.c_int), ("lo", C.c_int * 3), ("hi", C.c_int * 3),
                ("n_freq", C.c_int), ("omega", C.c_void_p), ("phasor", C.c_void_p)]


_LIBS: dict = {}


def _lib(tag: str):
    if tag not in _LIBS:
        so = build()[tag]
        L = C.CDLL(str(so))
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Desc)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_psi.restype = C.c_void_p
        L.orc_psi.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.orc_lpsi.restype = C.c_void_p
        L.orc_lpsi.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.orc_zero_psi.argtypes = [C.c_void_p]
        L.orc_zero_lpsi.argtypes = [C.c_void_p]
        L.orc_record_stride.restype = C.c_size_t
        L.orc_record_stride.argtypes = [C.POINTER(_Desc)]
        L.orc_cpml_table.argtypes = [C.POINTER(_Desc), C.c_int, C.c_int] + [C.c_void_p] * 3
        L.orc_step_E.argtypes = [C.c_void_p] * 4
        L.orc_step_H.argtypes = [C.c_void_p] * 3
        L.orc_adj_H.argtypes = [C.c_void_p] * 3
        L.orc_adj_E.argtypes = [C.c_void_p] * 3
        L.orc_inv_H.argtypes = [C.c_void_p] * 4
        L.orc_inv_E_grad.argtypes = [C.c_void_p] * 6
        L.orc_forward.restype = C.c_int
        L.orc_forward.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                  C.c_void_p, C.c_int, C.c_void_p, C.c_int,
                                  C.c_int, C.c_void_p, C.c_void_p]
        L.orc_backward.restype = C.c_int
        L.orc_backward.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                   C.c_void_p, C.c_int, C.c_void_p, C.c_int,
                                   C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                   C.c_void_p, C.c_void_p]
        L.orc_forward_td.restype = C.c_int
        L.orc_forward_td.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_int,
                                     C.c_int, C.c_void_p, C.c_void_p]
        L.orc_backward_mu.restype = C.c_int
        L.orc_backward_mu.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                      C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p,
                                      C.c_void_p, C.c_int, C.c_void_p,
                                      C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_backward_td.restype = C.c_int
        L.orc_backward_td.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                      C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p,
                                      C.c_void_p, C.c_int, C.c_void_p,
                                      C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_flux.restype = C.c_int
        L.orc_flux.argtypes = [C.POINTER(_Detector), C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.orc_flux_vjp.restype = C.c_int
        L.orc_flux_vjp.argtypes = [C.POINTER(_Detector), C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_tfsf_plane.restype = C.c_int
        L.orc_tfsf_plane.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int,
                                     C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_int)]
        L.orc_backward_tape.restype = C.c_int
        L.orc_backward_tape.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p,
                                        C.c_void_p, C.c_int, C.c_void_p, C.c_void_p,
                                        C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_grad_rho.argtypes = [C.POINTER(_Desc), C.c_void_p, C.c_void_p, C.c_double,
                                   C.POINTER(C.c_int), C.POINTER(C.c_int), C.c_void_p]
        L.orc_set_ftz.argtypes = [C.c_int]
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        _LIBS[tag] = L
    return _LIBS[tag]


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Oracle:
    """One grid of the CPU oracle.  dtype float64 = parity reference, float32 = timed baseline.

    CPML constants: 0 selects the default of reading R8 (m=3, sigma_scale=0.8(m+1),
    kappa_max=1, alpha_max=0, alpha_m=1, eps_bg=1); sigma_max = sigma_scale/sqrt(eps_bg).
    """

    def __init__(self, nx, ny, nz, courant, periodic=False, pml_cells=0,
                 pml_m=0.0, pml_sigma_scale=0.0, pml_kappa_max=0.0, pml_alpha_max=0.0,
                 pml_alpha_m=0.0, pml_eps_bg=0.0, dtype=np.float64):
        self.dtype = np.dtype(dtype)
        self.tag = "f64" if self.dtype == np.float64 else "f32"
        self.L = _lib(self.tag)
        m = pml_m if pml_m > 0 else 3.0
        ss = pml_sigma_scale if pml_sigma_scale > 0 else 0.8 * (m + 1.0)
        km = pml_kappa_max if pml_kappa_max > 0 else 1.0
        am = pml_alpha_m if pml_alpha_m > 0 else 1.0
        eb = pml_eps_bg if pml_eps_bg > 0 else 1.0
        self.desc = _Desc(nx, ny, nz, int(bool(periodic)), int(pml_cells), float(courant),
                          m, ss / math.sqrt(eb), km, float(pml_alpha_max), am)
        self.shape = (nz, ny, nx)
        self.nc = nx * ny * nz
        self.d = int(pml_cells)
        self.h = self.L.orc_create(C.byref(self.desc))
        if not self.h:
            raise ValueError("orc_create rejected the descriptor")
        self._keep = []

    def __del__(self):
        try:
            if getattr(self, "h", None):
                self.L.orc_destroy(self.h)
                self.h = None
        except Exception:
            pass

    # ---- helpers ---------------------------------------------------------
    def arr(self, a, shape=None):
        if a is None:
            return None
        a = np.ascontiguousarray(a, dtype=self.dtype)
        if shape is not None:
            assert a.size == int(np.prod(shape)), (a.shape, shape)
        return a

    def zeros_fields(self):
        return np.zeros((6,) + self.shape, dtype=self.dtype)

    def record_stride(self):
        return int(self.L.orc_record_stride(C.byref(self.desc)))

    def cpml_table(self, axis, half):
        n = (self.desc.nx, self.desc.ny, self.desc.nz)[axis]
        b, a, ik = (np.zeros(n, dtype=np.float64) for _ in range(3))
        self.L.orc_cpml_table(C.byref(self.desc), axis, half, _ptr(b), _ptr(a), _ptr(ik))
        return b, a, ik

    def _view(self, p):
        buf = (C.c_char * (self.nc * self.dtype.itemsize)).from_address(p)
        return np.frombuffer(buf, dtype=self.dtype).reshape(self.shape)

    def psi(self, is_H, c, s):
        return self._view(self.L.orc_psi(self.h, int(is_H), c, s))

    def lpsi(self, is_H, c, s):
        return self._view(self.L.orc_lpsi(self.h, int(is_H), c, s))

    def zero_psi(self):
        self.L.orc_zero_psi(self.h)

    def zero_lpsi(self):
        self.L.orc_zero_lpsi(self.h)

    def set_aniso(self, on=True):
        """N4 (reading R30): inv_eps and its gradient become [3, nz, ny, nx], one volume per E component."""
        self.aniso = bool(on)
        self.L.orc_set_aniso.argtypes = [C.c_void_p, C.c_int]
        self.L.orc_set_aniso(self.h, int(self.aniso))

    def _ie(self, inv_eps):
        return self.arr(inv_eps, ((3,) + self.shape) if getattr(self, "aniso", False) else self.shape)

    def _gshape(self):
        return ((3,) + self.shape) if getattr(self, "aniso", False) else self.shape

    def set_sigma(self, sigma):
        """N4 (reading R29): normalised electric conductivity per voxel for the lossy E update, or None (lossless)."""
        self._sigma = self.arr(sigma, self.shape)
        self.L.orc_set_sigma.argtypes = [C.c_void_p, C.c_void_p]
        self.L.orc_set_sigma(self.h, _ptr(self._sigma))

    def _sources(self, sources):
        n = len(sources)
        arr = (_Source * max(n, 1))()
        keep = []
        for s, q in zip(arr, sources):
            s.comp = int(q.component)
            s.lo[:] = list(q.lo)
            s.hi[:] = list(q.hi)
            prof = self.arr(q.profile)
            wav = self.arr(q.waveform)
            keep += [prof, wav]
            s.profile = None if prof is None else prof.ctypes.data
            s.waveform = wav.ctypes.data
        return arr, n, keep

    def _detectors(self, detectors, phasors):
        n = len(detectors)
        arr = (_Detector * max(n, 1))()
        keep = []
        for idx, (s, q) in enumerate(zip(arr, detectors)):
            s.mask = int(q.component_mask)
            s.lo[:] = list(q.lo)
            s.hi[:] = list(q.hi)
            om = np.ascontiguousarray(q.omega, dtype=np.float64)
            s.n_freq = om.size
            s.omega = om.ctypes.data
            keep.append(om)
            s.phasor = None if phasors is None else phasors[idx].ctypes.data
        return arr, n, keep

    @staticmethod
    def tdet_shape(td, n_steps):
        """Output shape of a time-domain detector (kind 'snapshot' | 'energy', component_mask, lo, hi, stride)."""
        n_rec = n_steps // td.stride
        if td.kind == "energy":
            return (n_rec,)
        ncomp = bin(int(td.component_mask) & 63).count("1")
        return (n_rec, ncomp, td.hi[2] - td.lo[2], td.hi[1] - td.lo[1], td.hi[0] - td.lo[0])

    def _tdetectors(self, tdets, outs):
        n = len(tdets)
        arr = (_TDetector * max(n, 1))()
        for idx, (s, q) in enumerate(zip(arr, tdets)):
            s.kind = 1 if q.kind == "energy" else 0
            s.mask = int(q.component_mask)
            s.lo[:] = list(q.lo)
            s.hi[:] = list(q.hi)
            s.stride = int(q.stride)
            s.out = None if outs is None else outs[idx].ctypes.data
        return arr, n

    @staticmethod
    def phasor_shape(det):
        ncomp = bin(int(det.component_mask) & 63).count("1")
        bz, by, bx = (det.hi[2] - det.lo[2], det.hi[1] - det.lo[1], det.hi[0] - det.lo[0])
        return (len(det.omega), ncomp, bz, by, bx, 2)

    # ---- single steps (for the pins) --------------------------------------
    def step_E(self, fields, ie, bracket=None):
        self.L.orc_step_E(self.h, _ptr(fields), _ptr(ie), _ptr(bracket))

    def step_H(self, fields, im=None):
        self.L.orc_step_H(self.h, _ptr(fields), _ptr(im))

    def adj_H(self, lam, im=None):
        self.L.orc_adj_H(self.h, _ptr(lam), _ptr(im))

    def adj_E(self, lam, ie):
        self.L.orc_adj_E(self.h, _ptr(lam), _ptr(ie))

    def inv_H(self, fields, im=None, rec_n=None):
        self.L.orc_inv_H(self.h, _ptr(fields), _ptr(im), _ptr(rec_n))

    def inv_E_grad(self, fields, ie, lam=None, g=None, rec_n=None):
        self.L.orc_inv_E_grad(self.h, _ptr(fields), _ptr(ie), _ptr(lam), _ptr(g), _ptr(rec_n))

    # ---- drivers ------------------------------------------------------------
    def forward(self, fields, inv_eps, inv_mu=None, sources=(), detectors=(), n_steps=0,
                record=False, tape=False, phasors=None, reset_psi=True, time_detectors=()):
        """Runs n_steps in place on `fields` (dtype self.dtype, shape [6,nz,ny,nx]).

        Returns dict(phasors=[...], rec=array|None, tape=array|None)."""
        assert fields.dtype == self.dtype and fields.flags.c_contiguous
        ie = self._ie(inv_eps)
        im = self.arr(inv_mu, self.shape)
        if reset_psi:
            self.zero_psi()
        if phasors is None:
            phasors = [np.zeros(self.phasor_shape(d), dtype=self.dtype) for d in detectors]
        sarr, ns, k1 = self._sources(sources)
        darr, nd, k2 = self._detectors(detectors, phasors)
        rec = np.zeros((n_steps, self.record_stride()), dtype=self.dtype) if record else None
        tp = np.zeros((n_steps, 3) + self.shape, dtype=self.dtype) if tape else None
        touts = [np.zeros(self.tdet_shape(t, n_steps), dtype=self.dtype) for t in time_detectors]
        tarr, nt = self._tdetectors(time_detectors, touts)
        rc = self.L.orc_forward_td(self.h, _ptr(fields), _ptr(ie), _ptr(im), sarr, ns, darr, nd, tarr, nt,
                                   int(n_steps), _ptr(rec), _ptr(tp))
        assert rc == 0, rc
        return {"phasors": phasors, "rec": rec, "tape": tp, "time_outputs": touts}

    def backward(self, fields, inv_eps, inv_mu=None, sources=(), detectors=(),
                 dL_dphasor=None, dL_dfields=None, n_steps=0, rec=None, time_detectors=(), dL_dtime=None,
                 want_grad_mu=False):
        """Time-reversed gradient.  `fields` (state n_steps) is overwritten by the
        reconstructed state 0 on I.  Returns (g, dL_dfields0), or (g, dL_dfields0, dL/d inv_mu) with want_grad_mu (N4)."""
        assert fields.dtype == self.dtype and fields.flags.c_contiguous
        ie = self._ie(inv_eps)
        im = self.arr(inv_mu, self.shape)
        sarr, ns, k1 = self._sources(sources)
        darr, nd, k2 = self._detectors(detectors, None)
        gp = None
        keep = []
        if dL_dphasor is not None:
            gp = (C.c_void_p * max(nd, 1))()
            for i, G in enumerate(dL_dphasor):
                Ga = self.arr(G)
                keep.append(Ga)
                gp[i] = None if Ga is None else Ga.ctypes.data
        dLf = self.arr(dL_dfields)
        g = np.zeros(self._gshape(), dtype=self.dtype)
        lam0 = np.zeros((6,) + self.shape, dtype=self.dtype)
        tarr, nt = self._tdetectors(time_detectors, None)
        tp = None
        if dL_dtime is not None:
            tp = (C.c_void_p * max(nt, 1))()
            for i, G in enumerate(dL_dtime):
                Ga = self.arr(G)
                keep.append(Ga)
                tp[i] = None if Ga is None else Ga.ctypes.data
        g_mu = np.zeros(self.shape, dtype=self.dtype) if want_grad_mu else None
        rc = self.L.orc_backward_mu(self.h, _ptr(fields), _ptr(ie), _ptr(im), sarr, ns, darr, nd, gp,
                                    tarr, nt, tp, _ptr(dLf), int(n_steps), _ptr(rec), _ptr(g), _ptr(lam0), _ptr(g_mu))
        assert rc == 0, rc
        return (g, lam0, g_mu) if want_grad_mu else (g, lam0)

    # ---- N2: flux from phasors, TFSF plane source ----------------------------
    def flux(self, det, phasor, axis, interpolate=False):
        """Poynting flux through the detector's plane along +axis for every frequency (reading R24)."""
        P = self.arr(phasor)
        darr, nd, k2 = self._detectors([det], [P])
        out = np.zeros(len(det.omega), dtype=self.dtype)
        rc = self.L.orc_flux(darr, _ptr(P), int(axis), int(bool(interpolate)), _ptr(out))
        assert rc == 0, rc
        return out

    def flux_vjp(self, det, phasor, axis, interpolate, dL_dflux):
        P = self.arr(phasor)
        darr, nd, k2 = self._detectors([det], [P])
        G = self.arr(dL_dflux)
        out = np.zeros_like(P)
        rc = self.L.orc_flux_vjp(darr, _ptr(P), int(axis), int(bool(interpolate)), _ptr(G), _ptr(out))
        assert rc == 0, rc
        return out

    def tfsf_plane(self, courant, eps_r, mu_r, axis, pol, direction, base):
        """Waveforms of the E patch and the H patch of a one-directional plane source (reading R25).
        Returns (wE, wH, h_component, h_plane_offset); all fp64."""
        base = np.ascontiguousarray(base, dtype=np.float64)
        wE, wH = np.zeros_like(base), np.zeros_like(base)
        off = C.c_int(0)
        hc = self.L.orc_tfsf_plane(float(courant), float(eps_r), float(mu_r), int(axis), int(pol), int(direction),
                                   base.size, _ptr(base), _ptr(wE), _ptr(wH), C.byref(off))
        assert hc >= 3, hc
        return wE, wH, hc, off.value

    def backward_tape(self, inv_eps, inv_mu=None, detectors=(), dL_dphasor=None,
                      dL_dfields=None, n_steps=0, tape=None):
        ie = self._ie(inv_eps)
        im = self.arr(inv_mu, self.shape)
        darr, nd, k2 = self._detectors(detectors, None)
        gp = None
        keep = []
        if dL_dphasor is not None:
            gp = (C.c_void_p * max(nd, 1))()
            for i, G in enumerate(dL_dphasor):
                Ga = self.arr(G)
                keep.append(Ga)
                gp[i] = None if Ga is None else Ga.ctypes.data
        dLf = self.arr(dL_dfields)
        g = np.zeros(self._gshape(), dtype=self.dtype)
        lam0 = np.zeros((6,) + self.shape, dtype=self.dtype)
        rc = self.L.orc_backward_tape(self.h, _ptr(ie), _ptr(im), darr, nd, gp, _ptr(dLf),
                                      int(n_steps), _ptr(tape), _ptr(g), _ptr(lam0))
        assert rc == 0, rc
        return g, lam0

    def grad_rho(self, g, inv_eps, delta_eps, lo, hi):
        """B6 (reading R20): dL/drho on the design box [lo, hi) from g = dL/d(inv_eps); box-shaped [k][j][i]."""
        g = self.arr(g, self.shape)
        ie = self.arr(inv_eps, self.shape)
        out = np.zeros((hi[2] - lo[2], hi[1] - lo[1], hi[0] - lo[0]), dtype=self.dtype)
        self.L.orc_grad_rho(C.byref(self.desc), _ptr(g), _ptr(ie), float(delta_eps),
                            (C.c_int * 3)(*lo), (C.c_int * 3)(*hi), _ptr(out))
        return out

    def set_ftz(self, on=True):
        self.L.orc_set_ftz(int(on))

    def set_num_threads(self, n):
        self.L.orc_set_num_threads(int(n))

    def num_threads(self):
        return int(self.L.orc_num_threads())
