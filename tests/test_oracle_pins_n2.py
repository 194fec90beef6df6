"""Pins for the N2 part of the CPU oracle (Poynting-flux / energy / snapshot detectors, one-directional
TFSF plane source).  As in test_oracle_pins.py each test checks the oracle against
something the mathematics fixes, not against itself or the CUDA path:

N2-a  flux of the exact discrete plane-wave eigenmode (P1) in closed form, with and without Yee co-location
N2-b  flux VJP against central finite differences (the flux is a quadratic form of the phasors: exact)
N2-c  energy of the eigenmode in closed form; energy / snapshot detectors against block-wise stepping
N2-d  gradient of a loss on energy and snapshot outputs against central finite differences (tiny CPML grid)
N2-e  TFSF plane source: nothing behind the interface (to rounding), every (axis, polarisation, direction);
      backward flux <= 1e-12 of the forward flux
"""
import math

import numpy as np
import pytest

from oracle.oracle import Oracle
from paper_2412_12360_b200 import workloads as wl

S = wl.COURANT


def _stag(shape, comp, is_H):
    nz, ny, nx = shape
    off = [0.0, 0.0, 0.0]
    if is_H:
        off[(comp + 1) % 3] = 0.5
        off[(comp + 2) % 3] = 0.5
    else:
        off[comp] = 0.5
    x = np.arange(nx, dtype=np.float64)[None, None, :] + off[0]
    y = np.arange(ny, dtype=np.float64)[None, :, None] + off[1]
    z = np.arange(nz, dtype=np.float64)[:, None, None] + off[2]
    return x, y, z


def _eigenmode(dims, mvec, M, pol_seed):
    """Exact plane-wave eigenmode of the leapfrog (pin P1) whose frequency is exactly 2 pi / M: the permittivity is
    chosen so that sin^2(w/2) = (S^2/eps) sum sin^2(k_a/2) holds with w = 2 pi / M."""
    nx, ny, nz = dims
    shape = (nz, ny, nx)
    k = np.array([2 * math.pi * mvec[0] / nx, 2 * math.pi * mvec[1] / ny, 2 * math.pi * mvec[2] / nz])
    w = 2.0 * math.pi / M
    eps_r = S * S * np.sum(np.sin(k / 2.0) ** 2) / math.sin(w / 2.0) ** 2
    assert eps_r > 1.0
    K = 2.0 * np.sin(k / 2.0)
    r = np.random.default_rng(pol_seed).standard_normal(3)
    A = r - K * (r @ K) / (K @ K)
    Bv = S * np.cross(K, A) / (2.0 * math.sin(w / 2.0))

    def state(n):
        f = np.zeros((6,) + shape)
        for c in range(3):
            x, y, z = _stag(shape, c, False)
            f[c] = A[c] * np.cos(k[0] * x + k[1] * y + k[2] * z - w * n)
            x, y, z = _stag(shape, c, True)
            f[3 + c] = Bv[c] * np.cos(k[0] * x + k[1] * y + k[2] * z - w * (n + 0.5))
        return f

    return shape, k, w, eps_r, A, Bv, state


# ----------------------------------------------------------------------------- N2-a
@pytest.mark.parametrize("dims,mvec,axis,M", [((16, 12, 8), (0, 0, 1), 2, 16), ((16, 12, 8), (1, 0, 1), 2, 16),
                                              ((16, 12, 8), (2, 1, 0), 0, 16), ((10, 12, 8), (1, 2, -1), 1, 12)])
def test_n2a_flux_of_the_exact_plane_wave(dims, mvec, axis, M):
    """For E_c = A_c cos(k.r - w t), H_c = B_c cos(k.r_H - w (t + 1/2)) and a run over whole periods (w N = 2 pi q), the
    DFT phasors are (N/2) A e^{-i theta_E} and (N/2) B e^{-i (theta_H - w/2)} exactly, hence per plane cell
      co-located : 1/2 Re(E_b conj H~_c - E_c conj H~_b) = (N/2)^2 cos(k_a/2) (A_b B_c - A_c B_b) / 2
      raw        :                                         (N/2)^2 cos((k_a - w)/2) (A_b B_c - A_c B_b) / 2
    (E_b and H_c share their in-plane position on the Yee grid; they differ by half a cell along a and half a step)."""
    q = 3
    shape, k, w, eps_r, A, Bv, state = _eigenmode(dims, mvec, M, pol_seed=axis)
    nx, ny, nz = dims
    N = M * q
    a, b, c = axis, (axis + 1) % 3, (axis + 2) % 3
    p = 5
    for interpolate in (True, False):
        lo, hi = [0, 0, 0], [nx, ny, nz]
        lo[a], hi[a] = (p - 1 if interpolate else p), p + 1
        det = wl.Detector((1 << b) | (1 << c) | (1 << (3 + b)) | (1 << (3 + c)), tuple(lo), tuple(hi), [w])
        det.omega = [w]                                       # exact (the dataclass rounds omega to fp32 for the GPU's sake)
        o = Oracle(nx, ny, nz, S, periodic=True)
        f = state(0)
        out = o.forward(f, np.full(shape, 1.0 / eps_r), detectors=[det], n_steps=N)
        assert np.max(np.abs(f - state(N))) < 1e-11            # still the eigenmode (P1)
        flux = o.flux(det, out["phasors"][0], a, interpolate)
        cells = nx * ny * nz // dims[a]
        geom = math.cos(k[a] / 2.0) if interpolate else math.cos((k[a] - w) / 2.0)
        want = cells * (N / 2.0) ** 2 * 0.5 * geom * (A[b] * Bv[c] - A[c] * Bv[b])
        assert abs(want) > 1.0
        assert abs(flux[0] - want) < 1e-10 * abs(want), (interpolate, flux[0], want)
    # sanity of the sign convention: the flux along +a has the sign of k_a (the wave travels along +k)
    assert np.sign(want) == np.sign(k[a])


# ----------------------------------------------------------------------------- N2-b
@pytest.mark.parametrize("interpolate", [False, True])
def test_n2b_flux_vjp_against_finite_differences(interpolate):
    rng = np.random.default_rng(12)
    a = 1
    lo, hi = (2, 3 if interpolate else 4, 1), (7, 5, 5)
    det = wl.Detector(0b111101, lo, hi, [0.31, 0.47])         # Ex, Ez, Hx, Hy, Hz (and the unused Hy): tangential to y = Ex, Ez, Hx, Hz
    o = Oracle(12, 10, 8, S, periodic=True)
    P = rng.standard_normal(det.phasor_shape)
    G = rng.standard_normal(2)
    vjp = o.flux_vjp(det, P, a, interpolate, G)
    assert vjp.shape == P.shape
    h = 1e-5
    idx = [tuple(rng.integers(0, s) for s in P.shape) for _ in range(40)]
    for t in idx:
        Pp, Pm = P.copy(), P.copy()
        Pp[t] += h
        Pm[t] -= h
        fd = float(G @ (o.flux(det, Pp, a, interpolate) - o.flux(det, Pm, a, interpolate))) / (2 * h)
        assert abs(fd - vjp[t]) < 1e-8 * max(1.0, abs(fd)), (t, fd, vjp[t])
    # components that do not enter the flux (the normal ones; E on the lower plane when co-locating) get no cotangent
    comps = [c for c in range(6) if (det.component_mask >> c) & 1]
    assert np.all(vjp[:, comps.index(4)] == 0)                # Hy is normal to the plane
    if interpolate:
        assert np.all(vjp[:, comps.index(0), :, 0] == 0) and np.any(vjp[:, comps.index(3), :, 0] != 0)


# ----------------------------------------------------------------------------- N2-c
def test_n2c_energy_of_the_eigenmode_and_blockwise_consistency():
    """Energy detector: for the plane-wave eigenmode the sum of cos^2 over whole spatial periods is cells/2 for every
    component at every time, so U = (cells/4) (eps |A|^2 + |B|^2) exactly.  Snapshot detector: equals the state reached
    by stepping in blocks."""
    dims, mvec = (16, 12, 8), (1, 0, 1)
    shape, k, w, eps_r, A, Bv, state = _eigenmode(dims, mvec, 16, pol_seed=7)
    nx, ny, nz = dims
    ie = np.full(shape, 1.0 / eps_r)
    td = [wl.TimeDetector("energy", (0, 0, 0), (nx, ny, nz), stride=1),
          wl.TimeDetector("snapshot", (3, 2, 1), (9, 7, 6), stride=5, component_mask=0b100110)]
    o = Oracle(nx, ny, nz, S, periodic=True)
    f = state(0)
    out = o.forward(f, ie, n_steps=23, time_detectors=td)
    U, snap = out["time_outputs"]
    want = nx * ny * nz / 4.0 * (eps_r * (A @ A) + Bv @ Bv)
    assert U.shape == (23,) and np.max(np.abs(U - want)) < 1e-11 * want
    assert snap.shape == (4, 3, 5, 5, 6)
    g = state(0)
    for q in range(4):
        o.forward(g, ie, n_steps=5)
        for ci, c in enumerate((1, 2, 5)):
            assert np.array_equal(snap[q, ci], g[c, 1:6, 2:7, 3:9])


# ----------------------------------------------------------------------------- N2-d
def test_n2d_gradient_through_energy_and_snapshot_detectors():
    """Loss = sum_q a_q U_q + sum W snapshot^2 on the tiny CPML grid (every term: kappa, alpha, inv_mu, E and H sources):
    the time-reversed gradient -- transposed detectors injected into the cotangents, plus the explicit dependence of the
    energy on inv_eps -- against central finite differences of the loss with respect to single inv_eps voxels."""
    w = wl.tiny_pml(n_steps=30)
    d = w.pml_cells
    shape = (w.nz, w.ny, w.nx)
    ie = w.inv_eps.astype(np.float64)
    td = [wl.TimeDetector("energy", (d, d, d), (w.nx - d, w.ny - d, w.nz - d), stride=3),
          wl.TimeDetector("snapshot", (d + 1, d, d + 1), (w.nx - d, w.ny - d - 1, w.nz - d), stride=4, component_mask=0b011011)]
    rng = np.random.default_rng(5)
    aq = rng.standard_normal(td[0].out_shape(w.n_steps))
    Wq = rng.standard_normal(td[1].out_shape(w.n_steps))

    def loss(ie_, want_grad=False):
        o = Oracle(**w.grid_kwargs())
        f = np.zeros((6,) + shape)
        out = o.forward(f, ie_, w.meta["inv_mu"], w.sources, [], w.n_steps, record=want_grad, time_detectors=td)
        U, snap = out["time_outputs"]
        L = float(aq @ U + np.sum(Wq * snap * snap))
        if not want_grad:
            return L
        g, _ = o.backward(f, ie_, w.meta["inv_mu"], w.sources, [], None, None, w.n_steps, out["rec"],
                          time_detectors=td, dL_dtime=[aq, 2.0 * Wq * snap])
        return L, g

    L, g = loss(ie, True)
    scale = np.max(np.abs(g))
    assert scale > 0
    h = 1e-6
    for v in [(w.nz // 2, w.ny // 2, w.nx // 2), (d, d, d), (w.nz - d - 1, w.ny - d - 1, w.nx - d - 1), (d + 1, d + 2, d + 3)]:
        ip, im_ = ie.copy(), ie.copy()
        ip[v] += h
        im_[v] -= h
        fd = (loss(ip) - loss(im_)) / (2 * h)
        assert abs(fd - g[v]) < 2e-6 * scale + 1e-6 * abs(fd), (v, fd, g[v])


# ----------------------------------------------------------------------------- N2-e
@pytest.mark.parametrize("axis,pol", [(0, 1), (0, 2), (1, 0), (1, 2), (2, 0), (2, 1)])
@pytest.mark.parametrize("direction", [1, -1])
def test_n2e_tfsf_plane_source_is_one_directional(axis, pol, direction):
    """The E patch + H patch pair launches a plane wave to one side only: in a periodic uniform box the field behind
    the interface stays at rounding level while the wave in front has the source's amplitude, and the DFT flux behind
    is <= 1e-12 of the flux in front.  (Run shorter than the numerical domain of dependence needs to wrap around.)"""
    n_long, n_steps, p0 = 96, 70, 48
    dims = [6, 5, 4]
    dims[axis] = n_long
    nx, ny, nz = dims
    shape = (nz, ny, nx)
    eps_r, mu_r = 2.25, 1.0
    ppw = 14.0
    base = wl.gaussian_sine(n_steps, 24, 7, ppw).astype(np.float64)
    o = Oracle(nx, ny, nz, S, periodic=True)
    wE, wH, hcomp, hoff = o.tfsf_plane(S, eps_r, mu_r, axis, pol, direction, base)
    lo, hi = [0, 0, 0], [nx, ny, nz]
    lo[axis], hi[axis] = p0, p0 + 1
    srcE = wl.Source(pol, tuple(lo), tuple(hi), wE)
    lo[axis], hi[axis] = p0 + hoff, p0 + hoff + 1
    srcH = wl.Source(hcomp, tuple(lo), tuple(hi), wH)
    b, c = (axis + 1) % 3, (axis + 2) % 3
    mask = (1 << b) | (1 << c) | (1 << (3 + b)) | (1 << (3 + c))
    om = wl.omega_ppw(ppw)

    def plane_det(p):
        lo, hi = [0, 0, 0], [nx, ny, nz]
        lo[axis], hi[axis] = p - 1, p + 1
        return wl.Detector(mask, tuple(lo), tuple(hi), [om])

    dets = [plane_det(p0 + 12 * direction), plane_det(p0 - 12 * direction)]       # in front / behind
    f = np.zeros((6,) + shape)
    out = o.forward(f, np.full(shape, 1.0 / eps_r), None, [srcE, srcH], dets, n_steps)
    ax_np = 3 - axis                                           # numpy axis of `axis` in [c, z, y, x]
    idx = np.arange(n_long)
    behind_E = idx < p0 if direction > 0 else idx > p0
    behind_H = idx < p0 if direction > 0 else idx >= p0
    front = np.max(np.abs(np.compress(~behind_E, f[:3], axis=ax_np)))
    assert front > 0.2 * np.max(np.abs(base))
    assert np.max(np.abs(np.compress(behind_E, f[:3], axis=ax_np))) < 1e-13 * front
    assert np.max(np.abs(np.compress(behind_H, f[3:], axis=ax_np))) < 1e-13 * front
    fl_front = o.flux(dets[0], out["phasors"][0], axis, True)[0]
    fl_back = o.flux(dets[1], out["phasors"][1], axis, True)[0]
    assert fl_front * direction > 0                            # energy flows the way the wave travels
    assert abs(fl_back) <= 1e-12 * abs(fl_front)
    # only the polarisation asked for (and its H partner) is excited
    others = [q for q in range(6) if q not in (pol, hcomp)]
    assert np.max(np.abs(f[others])) == 0.0


# ----------------------------------------------------------------------------- N4
def test_n4_gradient_with_respect_to_inv_mu():
    """SURVEY 8(f) N4 (dL/d inv_mu; Eq. 1): the time-reversed sweep's dL/d inv_mu on the interior against
    central finite differences of the loss with respect to single inv_mu voxels, on the tiny CPML grid with every term
    (kappa, alpha, random inv_eps and inv_mu, E and H sources, DFT loss on Ey and Hx)."""
    w = wl.tiny_pml(n_steps=30)
    d = w.pml_cells
    shape = (w.nz, w.ny, w.nx)
    ie = w.inv_eps.astype(np.float64)
    im0 = w.meta["inv_mu"].astype(np.float64)

    def loss(im_, want_grad=False):
        o = Oracle(**w.grid_kwargs())
        f = np.zeros((6,) + shape)
        out = o.forward(f, ie, im_, w.sources, w.detectors, w.n_steps, record=want_grad)
        P = out["phasors"][0]
        L = float(np.sum(P * P)) + 0.5 * float(np.sum(f[3:] ** 2))
        if not want_grad:
            return L
        dLf = np.zeros_like(f)
        dLf[3:] = f[3:]
        g, _, g_mu = o.backward(f, ie, im_, w.sources, w.detectors, [2.0 * P], dLf, w.n_steps, out["rec"], want_grad_mu=True)
        return L, g_mu

    L, g_mu = loss(im0, True)
    scale = np.max(np.abs(g_mu))
    assert scale > 0
    outside = np.ones(shape, dtype=bool)
    outside[d:w.nz - d, d:w.ny - d, d:w.nx - d] = False
    assert np.all(g_mu[outside] == 0.0)                       # formed on the interior only (R17)
    h = 1e-6
    for v in [(w.nz // 2, w.ny // 2, w.nx // 2), (d, d, d), (w.nz - d - 1, w.ny - d - 1, w.nx - d - 1), (d + 1, d + 2, d + 3),
              (w.nz // 2, w.ny // 2, w.nx // 2 + 1)]:
        ip, im_ = im0.copy(), im0.copy()
        ip[v] += h
        im_[v] -= h
        fd = (loss(ip) - loss(im_)) / (2 * h)
        assert abs(fd - g_mu[v]) < 2e-6 * scale + 1e-6 * abs(fd), (v, fd, g_mu[v])


# ----------------------------------------------------------------------------- N4: lossy media (reading R29)
def test_n4_lossy_eigenmode_decays_as_the_closed_form_says():
    """A plane wave in a uniform conductive medium, periodic box: with K^2 = sum_a 4 sin^2(k_a/2) the lossy leapfrog
    E' = Ca E + Cb S ie curl- H, H' = H - S curl+ E' has the eigenvalue rho of
        rho^2 - (1 + Ca - Cb S^2 ie K^2) rho + Ca = 0        (|rho|^2 = Ca: the decay per step)
    for the transverse mode E^n = Re(rho^n e exp(i k.r_E)), H^{n+1/2} = Re(rho^n h exp(i k.r_H)),
    h = -S rho (K+ x e) / (rho - 1), K+_a = 2 i sin(k_a/2) (staggered positions as in pin P1).  The oracle must follow it
    to rounding; sigma = 0 must reproduce the lossless run bit for bit."""
    nx, ny, nz = 12, 10, 8
    shape = (nz, ny, nx)
    mvec = (2, 1, 1)
    k = np.array([2 * math.pi * mvec[0] / nx, 2 * math.pi * mvec[1] / ny, 2 * math.pi * mvec[2] / nz])
    eps_r, sig = 2.25, 0.07
    ie = 1.0 / eps_r
    beta = 0.5 * sig * S * ie
    Ca, Cb = (1 - beta) / (1 + beta), 1 / (1 + beta)
    K2 = float(np.sum(4 * np.sin(k / 2) ** 2))
    bq = 1 + Ca - Cb * S * S * ie * K2
    rho = (bq + np.sqrt(complex(bq * bq - 4 * Ca))) / 2
    assert abs(abs(rho) ** 2 - Ca) < 1e-14 and abs(rho) < 1
    Kp = 2j * np.sin(k / 2)                       # symbol of the forward difference between the staggered positions
    r = np.random.default_rng(3).standard_normal(3)
    e = r - Kp * (r @ np.conj(Kp)) / K2           # transverse: Kp . e = 0 with the conjugate pairing of the staggered grid
    e = e - np.conj(Kp) * (Kp @ e) / K2
    h = -S * rho * np.cross(Kp, e) / (rho - 1)

    def state(n):
        f = np.zeros((6,) + shape)
        for c in range(3):
            x, y, z = _stag(shape, c, False)
            f[c] = np.real(rho ** n * e[c] * np.exp(1j * (k[0] * x + k[1] * y + k[2] * z)))
            x, y, z = _stag(shape, c, True)
            f[3 + c] = np.real(rho ** n * h[c] * np.exp(1j * (k[0] * x + k[1] * y + k[2] * z)))
        return f

    o = Oracle(nx, ny, nz, S, periodic=True)
    o.set_sigma(np.full(shape, sig))
    f = state(0)
    n = 57
    o.forward(f, np.full(shape, ie), n_steps=n)
    want = state(n)
    assert np.max(np.abs(want)) > 0.05 * np.max(np.abs(state(0)))            # not yet decayed to nothing
    assert np.max(np.abs(f - want)) < 1e-12 * np.max(np.abs(state(0)))
    # sigma = 0: the lossless update, bit for bit
    o0, o1 = Oracle(nx, ny, nz, S, periodic=True), Oracle(nx, ny, nz, S, periodic=True)
    o1.set_sigma(np.zeros(shape))
    f0, f1 = state(0), state(0)
    o0.forward(f0, np.full(shape, ie), n_steps=9)
    o1.forward(f1, np.full(shape, ie), n_steps=9)
    assert np.array_equal(f0, f1)


def test_n4_lossy_gradient_against_finite_differences():
    """Tape-mode gradient with a random conductivity on the tiny CPML grid (every term) against central finite differences
    in single inv_eps voxels (interior, PML, corner); the reversible sweep refuses a lossy medium."""
    w = wl.tiny_pml(n_steps=30)
    d = w.pml_cells
    shape = (w.nz, w.ny, w.nx)
    ie0 = w.inv_eps.astype(np.float64)
    sig = 0.3 * np.random.default_rng(12).random(shape)

    def loss(ie_, want_grad=False):
        o = Oracle(**w.grid_kwargs())
        o.set_sigma(sig)
        f = np.zeros((6,) + shape)
        out = o.forward(f, ie_, w.meta["inv_mu"], w.sources, w.detectors, w.n_steps, record=want_grad, tape=want_grad)
        P = out["phasors"][0]
        L = float(np.sum(P * P)) + 0.5 * float(np.sum(f[:3] ** 2))
        if not want_grad:
            return L
        dLf = np.zeros_like(f)
        dLf[:3] = f[:3]
        g, _ = o.backward_tape(ie_, w.meta["inv_mu"], w.detectors, [2.0 * P], dLf, w.n_steps, out["tape"])
        with pytest.raises(AssertionError):
            o.backward(f, ie_, w.meta["inv_mu"], w.sources, w.detectors, [2.0 * P], dLf, w.n_steps, out["rec"])
        return L, g

    L, g = loss(ie0, True)
    scale = np.max(np.abs(g))
    h = 1e-6
    for v in [(w.nz // 2, w.ny // 2, w.nx // 2), (d, d, d), (1, 2, 3), (0, 0, 0), (w.nz - 1, w.ny - 2, w.nx - 1), (d + 1, d + 2, d + 3)]:
        ip, im_ = ie0.copy(), ie0.copy()
        ip[v] += h
        im_[v] -= h
        fd = (loss(ip) - loss(im_)) / (2 * h)
        assert abs(fd - g[v]) < 2e-6 * scale + 1e-6 * abs(fd), (v, fd, g[v])


# ----------------------------------------------------------------------------- N4: one inv_eps volume per E component (R30)
def test_n4_per_component_inv_eps():
    """(i) Three equal volumes reproduce the scalar run bit for bit and their three gradients sum to the scalar gradient;
    (ii) a uniform diagonal-anisotropic periodic box carries the plane wave k || x, E || y at the speed eps_y alone fixes
    (exact eigenmode, pin P1 with eps -> eps_y) -- eps_x, eps_z must not matter; (iii) tape-mode and time-reversed gradients
    of the three volumes against central finite differences (tiny CPML grid, with a conductivity for the tape mode)."""
    w = wl.tiny_pml(n_steps=30)
    shape = (w.nz, w.ny, w.nx)
    d = w.pml_cells
    ie1 = w.inv_eps.astype(np.float64)
    ie3 = np.stack([ie1, ie1, ie1])

    def run(aniso, ie, sigma=None, mode="reversible"):
        o = Oracle(**w.grid_kwargs())
        if aniso:
            o.set_aniso(True)
        if sigma is not None:
            o.set_sigma(sigma)
        f = np.zeros((6,) + shape)
        out = o.forward(f, ie, w.meta["inv_mu"], w.sources, w.detectors, w.n_steps, record=True, tape=(mode == "tape"))
        P = out["phasors"][0]
        L = float(np.sum(P * P)) + 0.5 * float(np.sum(f[:3] ** 2))
        dLf = np.zeros_like(f)
        dLf[:3] = f[:3]
        fin = f.copy()
        if mode == "tape":
            g, _ = o.backward_tape(ie, w.meta["inv_mu"], w.detectors, [2.0 * P], dLf, w.n_steps, out["tape"])
        elif mode == "reversible":
            g, _ = o.backward(f, ie, w.meta["inv_mu"], w.sources, w.detectors, [2.0 * P], dLf, w.n_steps, out["rec"])
        else:
            g = None
        return L, g, fin

    L1, g1, f1 = run(False, ie1)
    L3, g3, f3 = run(True, ie3)
    assert np.array_equal(f1, f3) and L1 == L3
    assert g3.shape == (3,) + shape and np.max(np.abs(g3.sum(0) - g1)) < 1e-12 * np.max(np.abs(g1))
    # (iii) finite differences in single entries of the three volumes
    rng = np.random.default_rng(4)
    iea = ie3 * (0.8 + 0.4 * rng.random((3,) + shape))
    sig = 0.2 * rng.random(shape)
    for mode, sigma in (("reversible", None), ("tape", sig)):
        L, g, _ = run(True, iea, sigma, mode)
        scale = np.max(np.abs(g))
        h = 1e-6
        cells = [(0, w.nz // 2, w.ny // 2, w.nx // 2), (1, d, d, d), (2, w.nz - d - 1, w.ny - d - 1, w.nx - d - 1), (1, d + 1, d + 2, d + 3)]
        if mode == "tape":
            cells.append((2, 1, 2, 3))                 # a PML cell: only the tape mode has a gradient there
        for v in cells:
            ip, im_ = iea.copy(), iea.copy()
            ip[v] += h
            im_[v] -= h
            fd = (run(True, ip, sigma, None)[0] - run(True, im_, sigma, None)[0]) / (2 * h)
            assert abs(fd - g[v]) < 2e-6 * scale + 1e-6 * abs(fd), (mode, v, fd, g[v])
    # (ii) exact eigenmode with k along x and E along y: only eps_y enters
    nx, ny, nz = 16, 6, 5
    sh = (nz, ny, nx)
    kx = 2 * math.pi * 3 / nx
    eps = np.array([5.0, 2.25, 9.0])
    wq = 2 * math.asin(S / math.sqrt(eps[1]) * math.sin(kx / 2))
    A = 0.7
    Bz = S * (2 * math.sin(kx / 2)) * A / (2 * math.sin(wq / 2))      # P1: B = S (K x A) / (2 sin(w/2)), K = (Kx,0,0), A = (0,A,0)

    def state(n):
        f = np.zeros((6,) + sh)
        x, y, z = _stag(sh, 1, False)
        f[1] = A * np.cos(kx * x - wq * n) + 0 * y + 0 * z
        x, y, z = _stag(sh, 2, True)
        f[5] = Bz * np.cos(kx * x - wq * (n + 0.5)) + 0 * y + 0 * z
        return f

    o = Oracle(nx, ny, nz, S, periodic=True)
    o.set_aniso(True)
    f = state(0)
    o.forward(f, np.stack([np.full(sh, 1.0 / e) for e in eps]), n_steps=41)
    assert np.max(np.abs(f - state(41))) < 1e-12
