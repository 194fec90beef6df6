"""Seeded synthetic input generators (the ONLY module shared by the CUDA path's tests /
bench and the oracle's tests).  It holds none of the method's arithmetic: it only
builds input arrays (inverse permittivity, source profiles, source waveforms, detector
boxes and frequencies) and names the loss.  numpy only; importing it loads no native code.

The paper's workloads are inverse-design volumes: a high-contrast design block inside a
uniform cladding, PML on every face, one source plane, detector planes (PAPER.md L106,
L130, L162).  Its actual geometries (ref. 14 coupler, bend, stitching device) are not
available; the recipes below take their shapes and value ranges and stand in for them
(BASELINE.json `configs`).

RNG recipe: numpy.random.default_rng(seed).random(shape, dtype=float32), memory order
[k][j][i]; eps computed in fp32; inv_eps = float32(1)/eps.  The identical fp32 arrays
feed the oracle and the GPU.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np

COURANT = 0.99 / math.sqrt(3.0)   # PAPER.md L106 "courant factor of 0.99"; reading R2


@dataclass
class Source:
    """Additive patch F_c[box] += profile[cell] * waveform[n]."""
    component: int                       # 0..5 = Ex,Ey,Ez,Hx,Hy,Hz
    lo: Tuple[int, int, int]             # (i,j,k) inclusive
    hi: Tuple[int, int, int]             # (i,j,k) exclusive
    waveform: np.ndarray                 # float32 [n_steps]
    profile: Optional[np.ndarray] = None  # float32 box-shaped [k][j][i]; None => 1


@dataclass
class Detector:
    """Running DFT on a box."""
    component_mask: int
    lo: Tuple[int, int, int]
    hi: Tuple[int, int, int]
    omega: Sequence[float]               # rad / step (rounded to fp32 so both sides see the same value)

    def __post_init__(self):
        self.omega = [float(np.float32(o)) for o in self.omega]

    @property
    def n_comp(self) -> int:
        return bin(self.component_mask & 63).count("1")

    @property
    def phasor_shape(self):
        return (len(self.omega), self.n_comp, self.hi[2] - self.lo[2],
                self.hi[1] - self.lo[1], self.hi[0] - self.lo[0], 2)


@dataclass
class TimeDetector:
    """Time-domain detector: fires after every `stride`-th step.
    kind 'snapshot': the components of component_mask on the box; 'energy': the electromagnetic energy in the box."""
    kind: str
    lo: Tuple[int, int, int]
    hi: Tuple[int, int, int]
    stride: int = 1
    component_mask: int = 0

    def out_shape(self, n_steps: int):
        n_rec = n_steps // self.stride
        if self.kind == "energy":
            return (n_rec,)
        return (n_rec, bin(self.component_mask & 63).count("1"), self.hi[2] - self.lo[2], self.hi[1] - self.lo[1], self.hi[0] - self.lo[0])


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    n_steps: int
    inv_eps: np.ndarray                  # float32 [nz][ny][nx]
    sources: List[Source]
    detectors: List[Detector]
    courant: float = COURANT
    periodic: bool = False
    pml_cells: int = 0
    pml_eps_bg: float = 0.0
    pml_kappa_max: float = 0.0
    pml_alpha_max: float = 0.0
    loss: str = "none"                   # "final_E2" | "final_E2_interior" | "phasor_power" | "none"
    loss_detectors: Tuple[int, ...] = ()  # detectors carrying the phasor-power loss
    design_lo: Optional[Tuple[int, int, int]] = None
    design_hi: Optional[Tuple[int, int, int]] = None
    eps: Optional[np.ndarray] = None     # float32, kept for the rho chain rule
    meta: dict = field(default_factory=dict)

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz

    def grid_kwargs(self) -> dict:
        return dict(nx=self.nx, ny=self.ny, nz=self.nz, courant=self.courant,
                    periodic=self.periodic, pml_cells=self.pml_cells,
                    pml_eps_bg=self.pml_eps_bg, pml_kappa_max=self.pml_kappa_max,
                    pml_alpha_max=self.pml_alpha_max)


def omega_ppw(ppw: float, courant: float = COURANT) -> float:
    """Angular frequency in rad/step of a wave with `ppw` vacuum cells per wavelength."""
    return 2.0 * math.pi * courant / ppw


def gaussian_sine(n_steps: int, n0: float, w: float, ppw: float, courant: float = COURANT) -> np.ndarray:
    """Reading R12: s_n = exp(-(n-n0)^2/(2 w^2)) sin(omega (n-n0)), computed in fp64, stored fp32."""
    n = np.arange(n_steps, dtype=np.float64)
    s = np.exp(-((n - n0) ** 2) / (2.0 * w * w)) * np.sin(omega_ppw(ppw, courant) * (n - n0))
    return s.astype(np.float32)


def gaussian_profile(lo, hi, centre, sigma) -> np.ndarray:
    """exp(-((i-ci)^2+(j-cj)^2)/(2 sigma^2)) on an xy box (one k plane), float32 [1][by][bx]."""
    i = np.arange(lo[0], hi[0], dtype=np.float64)[None, :]
    j = np.arange(lo[1], hi[1], dtype=np.float64)[:, None]
    p = np.exp(-((i - centre[0]) ** 2 + (j - centre[1]) ** 2) / (2.0 * sigma * sigma))
    return p.astype(np.float32)[None, :, :]


def _inv(eps: np.ndarray) -> np.ndarray:
    return (np.float32(1.0) / eps.astype(np.float32)).astype(np.float32)


def extrude_into_pml(vol: np.ndarray, d: int) -> np.ndarray:
    """Reading R9: make `vol` invariant along each PML normal inside the slab by copying the
    interface value outward (axis order z, y, x)."""
    v = vol.copy()
    nz, ny, nx = v.shape
    if d <= 0:
        return v
    v[:d, :, :] = v[d:d + 1, :, :]
    v[nz - d:, :, :] = v[nz - d - 1:nz - d, :, :]
    v[:, :d, :] = v[:, d:d + 1, :]
    v[:, ny - d:, :] = v[:, ny - d - 1:ny - d, :]
    v[:, :, :d] = v[:, :, d:d + 1]
    v[:, :, nx - d:] = v[:, :, nx - d - 1:nx - d]
    return v


# --------------------------------------------------------------------------- configs
def c1(n: int = 16, n_steps: int = 100, seed: int = 1) -> Workload:
    """configs[0]: periodic box, random eps in [1,4], Ez dipole, loss = sum E^2 at the end."""
    u = np.random.default_rng(seed).random((n, n, n), dtype=np.float32)
    eps = (np.float32(1.0) + np.float32(3.0) * u).astype(np.float32)
    c = n // 2
    src = Source(2, (c, c, c), (c + 1, c + 1, c + 1), gaussian_sine(n_steps, 20, 6, 8))
    return Workload("C1", n, n, n, n_steps, _inv(eps), [src], [], periodic=True,
                    loss="final_E2", eps=eps)


def c2(n: int = 64, d: int = 10, n_steps: int = 1000) -> Workload:
    """configs[1]: CPML box, centred eps=2.25 block, Ey plane source, Ey DFT plane; forward only."""
    s = n / 64.0
    eps = np.ones((n, n, n), dtype=np.float32)
    b0, b1 = int(round(20 * s)), int(round(44 * s))
    eps[b0:b1, b0:b1, b0:b1] = np.float32(2.25)
    ks, kd = int(round(15 * s)), int(round(50 * s))
    src = Source(1, (0, 0, ks), (n, n, ks + 1), gaussian_sine(n_steps, 90, 30, 16))
    det = Detector(1 << 1, (d, d, kd), (n - d, n - d, kd + 1), [omega_ppw(16)])
    return Workload("C2", n, n, n, n_steps, _inv(eps), [src], [det], pml_cells=d, eps=eps)


def c3(n: int = 200, d: int = 12, n_steps: int = 2000, seed: int = 3, source_k: int | None = None) -> Workload:
    """configs[2] (the graded config): silica-like cladding, random design block, Gaussian-profile
    Ey source plane, Ey DFT plane; loss = phasor power; gradient wrt rho via inv_eps."""
    s = n / 200.0
    eps_bg = np.float32(2.085)
    eps = np.full((n, n, n), eps_bg, dtype=np.float32)
    x0, x1 = int(round(40 * s)), int(round(160 * s))
    z0, z1 = int(round(70 * s)), int(round(130 * s))
    rho = np.random.default_rng(seed).random((z1 - z0, x1 - x0, x1 - x0), dtype=np.float32)
    eps[z0:z1, x0:x1, x0:x1] = eps_bg + np.float32(12.25 - 2.085) * rho
    ks, kd = max(d + 1, int(round(20 * s))), min(n - d - 2, int(round(170 * s)))
    if source_k is not None:          # truncated full-size parity runs: the source plane next to the design box
        ks = source_k
    lo, hi = (d, d, ks), (n - d, n - d, ks + 1)
    ctr = (n - 1) / 2.0
    prof = gaussian_profile(lo, hi, (ctr, ctr), 20.0 * s)
    ppw = 31.0 * max(s, 0.3)
    wav = gaussian_sine(n_steps, 240 * max(s, 0.15), 80 * max(s, 0.15), ppw)
    src = Source(1, lo, hi, wav, prof)
    det = Detector(1 << 1, (d, d, kd), (n - d, n - d, kd + 1), [omega_ppw(ppw)])
    return Workload("C3", n, n, n, n_steps, _inv(eps), [src], [det], pml_cells=d,
                    pml_eps_bg=2.085, loss="phasor_power", loss_detectors=(0,),
                    design_lo=(x0, x0, z0), design_hi=(x1, x1, z1), eps=eps,
                    meta={"rho": rho, "delta_eps": 12.25 - 2.085})


def c3_mini(nx: int = 88, ny: int = 52, nz: int = 44, d: int = 8, n_steps: int = 200, seed: int = 33,
            kappa_max: float = 0.0, alpha_max: float = 0.0) -> Workload:
    """Non-cubic miniature of C3 (ragged tile tails on every axis) that the oracle finishes in seconds:
    cladding eps=2.085, random design block, Gaussian-profile Ey source plane, Ey+Hx DFT plane.  The default
    200 steps let the pulse (centre step 30) cross the design block and the detector plane, so the phasor-power
    gradient is well conditioned (fp32 build of the oracle vs its fp64 build: 4e-7 of max|g|; at 60 steps, before
    the pulse reaches the detector, it is 3e-4)."""
    eps_bg = np.float32(2.085)
    eps = np.full((nz, ny, nx), eps_bg, dtype=np.float32)
    x0, x1 = d + (nx - 2 * d) // 4, nx - d - (nx - 2 * d) // 4
    y0, y1 = d + (ny - 2 * d) // 4, ny - d - (ny - 2 * d) // 4
    z0, z1 = d + (nz - 2 * d) // 3, nz - d - (nz - 2 * d) // 3
    rho = np.random.default_rng(seed).random((z1 - z0, y1 - y0, x1 - x0), dtype=np.float32)
    eps[z0:z1, y0:y1, x0:x1] = eps_bg + np.float32(12.25 - 2.085) * rho
    ks, kd = d + 2, nz - d - 3
    lo, hi = (d, d, ks), (nx - d, ny - d, ks + 1)
    prof = gaussian_profile(lo, hi, ((nx - 1) / 2.0, (ny - 1) / 2.0), 0.15 * nx)
    wav = gaussian_sine(n_steps, 30, 10, 12)
    src = Source(1, lo, hi, wav, prof)
    det = Detector((1 << 1) | (1 << 3), (d, d, kd), (nx - d, ny - d, kd + 1), [omega_ppw(12), omega_ppw(14)])
    return Workload("C3-mini", nx, ny, nz, n_steps, _inv(eps), [src], [det], pml_cells=d,
                    pml_eps_bg=2.085, pml_kappa_max=kappa_max, pml_alpha_max=alpha_max,
                    loss="phasor_power", loss_detectors=(0,),
                    design_lo=(x0, y0, z0), design_hi=(x1, y1, z1), eps=eps,
                    meta={"rho": rho, "delta_eps": 12.25 - 2.085})


def c4(nx: int = 800, ny: int = 800, nz: int = 600, d: int = 16, n_steps: int = 5000,
       seed: int = 4) -> Workload:
    """configs[3]: memory-scale run; binary 4x4x4 blocks in the design region, 2 detector planes,
    3 frequencies; loss on the far plane only."""
    sx, sz = nx / 800.0, nz / 600.0
    eps_bg = np.float32(2.085)
    eps = np.full((nz, ny, nx), eps_bg, dtype=np.float32)
    x0, x1 = int(round(100 * sx)) // 4 * 4, int(round(700 * sx)) // 4 * 4
    y0, y1 = int(round(100 * ny / 800.0)) // 4 * 4, int(round(700 * ny / 800.0)) // 4 * 4
    z0, z1 = int(round(200 * sz)) // 4 * 4, int(round(400 * sz)) // 4 * 4
    bz, by, bx = (z1 - z0) // 4, (y1 - y0) // 4, (x1 - x0) // 4
    u = np.random.default_rng(seed).random((bz, by, bx), dtype=np.float32)
    blk = np.where(u < np.float32(0.5), np.float32(12.25), eps_bg).astype(np.float32)
    eps[z0:z0 + 4 * bz, y0:y0 + 4 * by, x0:x0 + 4 * bx] = np.repeat(np.repeat(np.repeat(blk, 4, 0), 4, 1), 4, 2)
    ks = max(d + 1, int(round(40 * sz)))
    k_near, k_far = max(d + 2, int(round(60 * sz))), min(nz - d - 2, int(round(540 * sz)))
    lo, hi = (d, d, ks), (nx - d, ny - d, ks + 1)
    prof = gaussian_profile(lo, hi, ((nx - 1) / 2.0, (ny - 1) / 2.0), 100.0 * sx)
    wav = gaussian_sine(n_steps, 300, 100, 31)
    src = Source(1, lo, hi, wav, prof)
    om = [omega_ppw(p) for p in (29, 31, 33)]
    dets = [Detector(1 << 1, (d, d, k_near), (nx - d, ny - d, k_near + 1), om),
            Detector(1 << 1, (d, d, k_far), (nx - d, ny - d, k_far + 1), om)]
    return Workload("C4", nx, ny, nz, n_steps, _inv(eps), [src], dets, pml_cells=d,
                    pml_eps_bg=2.085, loss="phasor_power", loss_detectors=(1,),
                    design_lo=(x0, y0, z0), design_hi=(x0 + 4 * bx, y0 + 4 * by, z0 + 4 * bz), eps=eps)


def c5(n: int, d: int = 10, n_steps: int = 500) -> Workload:
    """configs[4]: throughput sweep; random eps in [1,12.25] on I, extruded into the PML (R9);
    Ez dipole at the centre; loss = sum E^2 over I at the final step."""
    u = np.random.default_rng(5000 + n).random((n, n, n), dtype=np.float32)
    eps = (np.float32(1.0) + np.float32(11.25) * u).astype(np.float32)
    eps = extrude_into_pml(eps, d)
    c = n // 2
    src = Source(2, (c, c, c), (c + 1, c + 1, c + 1), gaussian_sine(n_steps, 40, 12, 20))
    return Workload(f"C5-N{n}", n, n, n, n_steps, _inv(eps), [src], [], pml_cells=d,
                    loss="final_E2_interior", eps=eps)


def tiny_pml(nx=14, ny=13, nz=12, d=3, n_steps=30, seed=7, kappa_max=3.0, alpha_max=0.05,
             with_inv_mu=True) -> Workload:
    """Small CPML grid exercising every term (kappa != 1, alpha != 0, E and H sources, DFT
    detector with two components and two frequencies, random inv_eps and inv_mu)."""
    rng = np.random.default_rng(seed)
    eps = (np.float32(1.0) + np.float32(3.0) * rng.random((nz, ny, nx), dtype=np.float32)).astype(np.float32)
    mu = (np.float32(1.0) + np.float32(0.5) * rng.random((nz, ny, nx), dtype=np.float32)).astype(np.float32)
    wavE = gaussian_sine(n_steps, 8, 3, 7)
    wavH = (0.5 * gaussian_sine(n_steps, 10, 4, 9)).astype(np.float32)
    wide = nx - 2 * d >= 3
    ks = min(d + 2, nz - d - 1)
    lo, hi = (d + 1 if wide else d, d, ks), (nx - d - 1 if wide else nx - d, ny - d, ks + 1)
    prof = (0.5 + rng.random((1, hi[1] - lo[1], hi[0] - lo[0]), dtype=np.float32)).astype(np.float32)
    srcs = [Source(1, lo, hi, wavE, prof),
            Source(3, (nx // 2, ny // 2, nz // 2), (nx // 2 + 1, ny // 2 + 1, nz // 2 + 1), wavH)]
    kd = max(d, nz - d - 2)
    det = Detector((1 << 1) | (1 << 3), (d, d, kd), (nx - d, ny - d, kd + 1),
                   [omega_ppw(7), omega_ppw(9)])
    w = Workload("tiny", nx, ny, nz, n_steps, _inv(eps), srcs, [det], pml_cells=d,
                 pml_kappa_max=kappa_max, pml_alpha_max=alpha_max, loss="phasor_power",
                 loss_detectors=(0,), eps=eps)
    w.meta["inv_mu"] = _inv(mu) if with_inv_mu else None
    return w
