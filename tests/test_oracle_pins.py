"""Pins for the CPU oracle (oracle/fdtd_oracle.c): each test checks the oracle against
something the paper or the mathematics fixes, NOT against itself or the CUDA path.

P1  exact discrete plane-wave eigenmode / Yee numerical dispersion relation
P2  exact discrete electromagnetic energy invariant (lossless periodic box)
P3  forward-N / inverse-N recovery ("reversible in time"), incl. NaN-poisoned PML
P4  gradient vs central finite differences (tiny CPML grid, every term exercised)
P5  tape-mode gradient == time-reversed gradient on the interior
P6  adjoint dot-product identity <Jv,w> = <v,J^T w>
P7  discrete Gauss law (div of curl = 0 on the Yee grid)
P8  CPML box vs a much larger box (absorption)
P9  late-time decay / stability in a CPML box
P10 linearity and null tests
P11 the paper's printed step counts (Table 2) => Courant convention
"""
import math

import numpy as np
import pytest

from oracle.oracle import Oracle
from paper_2412_12360_b200 import workloads as wl

S = wl.COURANT


def _rng(seed):
    return np.random.default_rng(seed)


def _stag(shape, comp, is_H):
    """Yee positions (x,y,z arrays broadcastable to shape [nz,ny,nx]) of component comp."""
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


# ----------------------------------------------------------------------------- P1
@pytest.mark.parametrize("dims,mvec,eps_r,pol_seed", [
    ((16, 12, 8), (2, 1, 1), 2.25, 0),
    ((12, 10, 14), (1, 0, 0), 1.0, 1),      # axis-aligned along x
    ((8, 12, 10), (0, 0, 2), 4.0, 2),       # axis-aligned along z
    ((10, 9, 11), (1, -2, 3), 1.7, 3),
])
def test_p1_exact_plane_wave_eigenmode(dims, mvec, eps_r, pol_seed):
    """A_c cos(k.r_E - w n), B_c cos(k.r_H - w (n+1/2)) with sin^2(w/2) = S^2/eps sum sin^2(k_a/2),
    K_a = 2 sin(k_a/2), A perp K, B = S (K x A)/(2 sin(w/2)) is an exact solution of the leapfrog."""
    nx, ny, nz = dims
    shape = (nz, ny, nx)
    k = np.array([2 * math.pi * mvec[0] / nx, 2 * math.pi * mvec[1] / ny, 2 * math.pi * mvec[2] / nz])
    K = 2.0 * np.sin(k / 2.0)
    sin2 = (S * S / eps_r) * np.sum(np.sin(k / 2.0) ** 2)
    assert 0 < sin2 < 1
    w = 2.0 * math.asin(math.sqrt(sin2))
    r = _rng(pol_seed).standard_normal(3)
    A = r - K * (r @ K) / (K @ K)            # A perpendicular to K
    B = S * np.cross(K, A) / (2.0 * math.sin(w / 2.0))

    def state(n):
        f = np.zeros((6,) + shape)
        for c in range(3):
            x, y, z = _stag(shape, c, False)
            f[c] = A[c] * np.cos(k[0] * x + k[1] * y + k[2] * z - w * n)
            x, y, z = _stag(shape, c, True)
            f[3 + c] = B[c] * np.cos(k[0] * x + k[1] * y + k[2] * z - w * (n + 0.5))
        return f

    o = Oracle(nx, ny, nz, S, periodic=True)
    f = state(0)
    ie = np.full(shape, 1.0 / eps_r)
    n_steps = 137
    o.forward(f, ie, n_steps=n_steps)
    ref = state(n_steps)
    assert np.max(np.abs(f - ref)) < 1e-12 * max(1.0, np.max(np.abs(ref)))
    # axis-aligned special case: |H| = sqrt(eps_r) |E| to within the half-step phase
    if sum(1 for v in mvec if v) == 1:
        assert abs(np.linalg.norm(B) / np.linalg.norm(A) - math.sqrt(eps_r)) < 1e-12


def test_p1_dispersion_detects_wrong_courant():
    """The same eigenmode with a Courant number off by 1% must NOT be reproduced (the pin has teeth)."""
    nx, ny, nz = 16, 12, 8
    shape = (nz, ny, nx)
    k = np.array([2 * math.pi * 2 / nx, 2 * math.pi / ny, 2 * math.pi / nz])
    K = 2.0 * np.sin(k / 2.0)
    w = 2.0 * math.asin(math.sqrt(S * S * np.sum(np.sin(k / 2.0) ** 2)))
    A = np.cross(K, [0.3, -1.0, 0.5])
    B = S * np.cross(K, A) / (2.0 * math.sin(w / 2.0))
    f = np.zeros((6,) + shape)
    for c in range(3):
        x, y, z = _stag(shape, c, False)
        f[c] = A[c] * np.cos(k[0] * x + k[1] * y + k[2] * z)
        x, y, z = _stag(shape, c, True)
        f[3 + c] = B[c] * np.cos(k[0] * x + k[1] * y + k[2] * z - w * 0.5)
    o = Oracle(nx, ny, nz, S * 1.01, periodic=True)
    g = f.copy()
    o.forward(g, np.ones(shape), n_steps=137)
    ref = np.zeros_like(f)
    for c in range(3):
        x, y, z = _stag(shape, c, False)
        ref[c] = A[c] * np.cos(k[0] * x + k[1] * y + k[2] * z - w * 137)
    assert np.max(np.abs(g[:3] - ref[:3])) > 1e-3


# ----------------------------------------------------------------------------- P2
def test_p2_exact_energy_invariant():
    """W_n = sum E^n.E^n/ie + sum H^{n+1/2}.H^{n-1/2}/im is conserved to rounding; the naive sum is not."""
    nx, ny, nz = 12, 10, 9
    shape = (nz, ny, nx)
    r = _rng(11)
    ie = 1.0 / (1.0 + 3.0 * r.random(shape))
    im = 1.0 / (1.0 + 0.5 * r.random(shape))
    o = Oracle(nx, ny, nz, S * 0.8, periodic=True)     # S*sqrt(max ie*im) < 1/sqrt(3)
    f = r.standard_normal((6,) + shape)
    W, naive = [], []
    Hprev = f[3:].copy()
    o.forward(f, ie, im, n_steps=1)
    for _ in range(200):
        W.append(np.sum(f[:3] ** 2 / ie) + np.sum(f[3:] * Hprev / im))
        naive.append(np.sum(f[:3] ** 2 / ie) + np.sum(f[3:] ** 2 / im))
        Hprev = f[3:].copy()
        o.forward(f, ie, im, n_steps=1)
    W, naive = np.array(W), np.array(naive)
    assert np.max(np.abs(W - W[0])) < 1e-11 * abs(W[0])
    assert (naive.max() - naive.min()) > 1e-3 * naive.mean()


# ----------------------------------------------------------------------------- P7
def test_p7_discrete_gauss_law():
    """sum_c dm_c (E_c/ie) is time-invariant at every node away from the sources."""
    nx, ny, nz = 11, 12, 10
    shape = (nz, ny, nx)
    r = _rng(5)
    ie = 1.0 / (1.0 + 3.0 * r.random(shape))
    o = Oracle(nx, ny, nz, S, periodic=True)
    f = r.standard_normal((6,) + shape)

    def div(f):
        out = np.zeros(shape)
        for c, ax in ((0, 2), (1, 1), (2, 0)):           # component c varies along numpy axis ax
            D = f[c] / ie
            out += D - np.roll(D, 1, axis=ax)
        return out

    src = wl.Source(2, (5, 6, 4), (6, 7, 5), wl.gaussian_sine(40, 10, 4, 8))
    d0 = div(f)
    o.forward(f, ie, sources=[src], n_steps=40)
    d1 = div(f)
    mask = np.ones(shape, bool)
    mask[4:6, 6, 5] = False                              # the two nodes touching the Ez source cell
    assert np.max(np.abs((d1 - d0)[mask])) < 1e-11
    assert np.max(np.abs((d1 - d0)[~mask])) > 1e-3       # and the source does create charge there


# ----------------------------------------------------------------------------- P3
def test_p3_forward_inverse_recovery_periodic():
    w = wl.c1()
    o = Oracle(**w.grid_kwargs())
    f0 = _rng(3).standard_normal((6, w.nz, w.ny, w.nx)) * 0.1
    f = f0.copy()
    o.forward(f, w.inv_eps, sources=w.sources, n_steps=w.n_steps)
    assert np.max(np.abs(f - f0)) > 0.05
    o.backward(f, w.inv_eps, sources=w.sources, n_steps=w.n_steps)
    assert np.max(np.abs(f - f0)) < 1e-12


def test_p3_interior_recovery_from_recorded_faces_with_poisoned_pml():
    """PML is not invertible: with only the recorded interface values the interior is
    recovered exactly, and nothing outside I is ever read (it is NaN during the reverse sweep)."""
    w = wl.tiny_pml(n_steps=40)
    d = w.pml_cells
    o = Oracle(**w.grid_kwargs())
    shape = (w.nz, w.ny, w.nx)
    f0 = _rng(4).standard_normal((6,) + shape) * 0.1
    f = f0.copy()
    out = o.forward(f, w.inv_eps, w.meta["inv_mu"], w.sources, w.detectors, w.n_steps, record=True)
    inter = (slice(None), slice(d, w.nz - d), slice(d, w.ny - d), slice(d, w.nx - d))
    keep = f[inter].copy()
    f[:] = np.nan
    f[inter] = keep
    g, _ = o.backward(f, w.inv_eps, w.meta["inv_mu"], w.sources, w.detectors, n_steps=w.n_steps,
                      rec=out["rec"])
    assert np.all(np.isfinite(f[inter]))
    assert np.max(np.abs(f[inter] - f0[inter])) < 1e-12
    assert np.all(g == 0)                                 # no cotangent => zero gradient (P10)


# ----------------------------------------------------------------------------- P4 / P5
def _loss_and_cotangents(w, f, phasors, wfield):
    """L = sum_f |P|^2 over the loss detectors + sum wfield * fields^2 (final state)."""
    L = float(np.sum(wfield * f * f))
    dLp = []
    for i, P in enumerate(phasors):
        if i in w.loss_detectors:
            L += float(np.sum(P * P))
            dLp.append(2.0 * P)
        else:
            dLp.append(None)
    return L, dLp, 2.0 * wfield * f


def _run_loss(w, ie, wfield, record=False, tape=False):
    o = Oracle(**w.grid_kwargs())
    f = np.zeros((6, w.nz, w.ny, w.nx))
    out = o.forward(f, ie, w.meta.get("inv_mu"), w.sources, w.detectors, w.n_steps, record=record, tape=tape)
    L, dLp, dLf = _loss_and_cotangents(w, f, out["phasors"], wfield)
    return o, f, out, L, dLp, dLf


def test_p4_p5_gradient_fd_tape_reversible():
    w = wl.tiny_pml(n_steps=30)
    shape = (w.nz, w.ny, w.nx)
    d = w.pml_cells
    ie = w.inv_eps.astype(np.float64)
    wfield = _rng(9).random((6,) + shape)                 # final-field loss over ALL cells, E and H
    o, f, out, L, dLp, dLf = _run_loss(w, ie, wfield, record=True, tape=True)
    g_tape, lam0_t = o.backward_tape(ie, w.meta["inv_mu"], w.detectors, dLp, dLf, w.n_steps, out["tape"])
    g_rev, lam0_r = o.backward(f, ie, w.meta["inv_mu"], w.sources, w.detectors, dLp, dLf, w.n_steps, out["rec"])
    inter = (slice(d, w.nz - d), slice(d, w.ny - d), slice(d, w.nx - d))
    scale = np.max(np.abs(g_tape))
    assert scale > 0
    # P5: identical on I; the reversible gradient is defined to be zero outside I (R17)
    assert np.max(np.abs(g_tape[inter] - g_rev[inter])) < 1e-10 * scale
    outside = np.ones(shape, bool)
    outside[inter] = False
    assert np.all(g_rev[outside] == 0)
    assert np.max(np.abs(lam0_t - lam0_r)) < 1e-10 * max(1.0, np.max(np.abs(lam0_t)))
    # P4: central finite differences on single voxels (interior, PML face, PML corner, source plane)
    h = 1e-6
    voxels = [(w.nz // 2, w.ny // 2, w.nx // 2), (d + 2, d + 1, d + 2), (d, d, d), (w.nz - d - 1, w.ny - d - 1, w.nx - d - 1),
              (1, w.ny // 2, w.nx // 2), (w.nz // 2, w.ny - 2, 2), (0, 0, 0), (w.nz // 2, 1, w.nx // 2)]
    for v in voxels:
        ip, im_ = ie.copy(), ie.copy()
        ip[v] += h
        im_[v] -= h
        Lp = _run_loss(w, ip, wfield)[3]
        Lm = _run_loss(w, im_, wfield)[3]
        fd = (Lp - Lm) / (2 * h)
        assert abs(fd - g_tape[v]) < 2e-6 * scale + 1e-6 * abs(fd), (v, fd, g_tape[v])


def test_p5_tape_equals_reversible_periodic_c1():
    w = wl.c1()
    ie = w.inv_eps.astype(np.float64)
    o = Oracle(**w.grid_kwargs())
    f = np.zeros((6, w.nz, w.ny, w.nx))
    out = o.forward(f, ie, sources=w.sources, n_steps=w.n_steps, tape=True)
    dLf = np.zeros_like(f)
    dLf[:3] = 2 * f[:3]
    g_t, _ = o.backward_tape(ie, dL_dfields=dLf, n_steps=w.n_steps, tape=out["tape"])
    g_r, _ = o.backward(f, ie, sources=w.sources, dL_dfields=dLf, n_steps=w.n_steps)
    assert np.max(np.abs(g_t - g_r)) < 1e-10 * np.max(np.abs(g_t))
    assert np.max(np.abs(f)) < 1e-12                      # state 0 (all zero) recovered


# ----------------------------------------------------------------------------- P6
def test_p6_adjoint_dot_product_single_steps_with_psi():
    """One E update and one H update, psi included in the vectors: <J v, w> = <v, J^T w>."""
    nx, ny, nz, d = 11, 10, 9, 3
    shape = (nz, ny, nx)
    r = _rng(21)
    ie = 1.0 / (1.0 + 3.0 * r.random(shape))
    im = 1.0 / (1.0 + 0.5 * r.random(shape))
    o = Oracle(nx, ny, nz, S, pml_cells=d, pml_kappa_max=3.0, pml_alpha_max=0.05)
    for is_H, step, adj, med in ((0, o.step_E, o.adj_E, ie), (1, o.step_H, o.adj_H, im)):
        v = r.standard_normal((6,) + shape)
        vpsi = r.standard_normal((3, 2) + shape)
        wv = r.standard_normal((6,) + shape)
        wpsi = r.standard_normal((3, 2) + shape)
        o.zero_psi(); o.zero_lpsi()
        f = v.copy()
        for c in range(3):
            for s in range(2):
                o.psi(is_H, c, s)[:] = vpsi[c, s]
        step(f, med)
        Jpsi = np.array([[o.psi(is_H, c, s).copy() for s in range(2)] for c in range(3)])
        lhs = np.sum(f * wv) + np.sum(Jpsi * wpsi)
        lam = wv.copy()
        for c in range(3):
            for s in range(2):
                o.lpsi(is_H, c, s)[:] = wpsi[c, s]
        adj(lam, med)
        JTpsi = np.array([[o.lpsi(is_H, c, s).copy() for s in range(2)] for c in range(3)])
        rhs = np.sum(v * lam) + np.sum(vpsi * JTpsi)
        assert abs(lhs - rhs) < 1e-11 * max(abs(lhs), 1.0), (is_H, lhs, rhs)


@pytest.mark.parametrize("periodic", [True, False])
def test_p6_adjoint_dot_product_n_steps(periodic):
    nx, ny, nz = 11, 10, 9
    d = 0 if periodic else 3
    shape = (nz, ny, nx)
    r = _rng(22)
    ie = 1.0 / (1.0 + 3.0 * r.random(shape))
    im = 1.0 / (1.0 + 0.5 * r.random(shape))
    o = Oracle(nx, ny, nz, S * 0.8, periodic=periodic, pml_cells=d, pml_kappa_max=3.0, pml_alpha_max=0.05)
    v = r.standard_normal((6,) + shape)
    wv = r.standard_normal((6,) + shape)
    f = v.copy()
    n = 25
    out = o.forward(f, ie, im, n_steps=n, tape=True)
    _, lam0 = o.backward_tape(ie, im, dL_dfields=wv, n_steps=n, tape=out["tape"])
    lhs, rhs = np.sum(f * wv), np.sum(v * lam0)
    assert abs(lhs - rhs) < 1e-11 * max(abs(lhs), 1.0)


# ----------------------------------------------------------------------------- P8 / P9
@pytest.mark.parametrize("kappa,alpha,tol", [(0.0, 0.0, 5e-5), (3.0, 0.05, 1.5e-4)])
def test_p8_cpml_matches_big_box(kappa, alpha, tol):
    """Same dipole in a 40^3/d=10 CPML box and in a 96^3 box whose walls are out of causal reach
    (125 steps * S < 48-20 cells): the interiors agree to the PML's reflection level, measured
    against the peak field seen in the interior during the run; hard walls are >1000x worse."""
    n_small, n_big, d, steps = 40, 96, 10, 125
    wav = wl.gaussian_sine(steps, 30, 10, 12)

    def run(n, dd, pml):
        o = Oracle(n, n, n, S, pml_cells=dd if pml else 0, pml_kappa_max=kappa, pml_alpha_max=alpha)
        f = np.zeros((6, n, n, n))
        c = n // 2
        peak = 0.0
        for b in range(0, steps, 25):                      # 25-step blocks only to track the peak
            src = [wl.Source(2, (c, c, c), (c + 1, c + 1, c + 1), np.roll(wav, -b))]
            o.forward(f, np.ones((n, n, n)), sources=src, n_steps=25, reset_psi=(b == 0))
            peak = max(peak, float(np.max(np.abs(f[:, dd:n - dd, dd:n - dd, dd:n - dd]))))
        return f, peak

    fs, peak = run(n_small, d, True)
    fb, _ = run(n_big, 0, False)
    f0, _ = run(n_small, d, False)                         # same box, hard (zero-pad) walls
    off = (n_big - n_small) // 2
    sl_s = (slice(None),) + (slice(d, n_small - d),) * 3
    sl_b = (slice(None),) + (slice(off + d, off + n_small - d),) * 3
    assert peak > 0.1
    err_pml = np.max(np.abs(fs[sl_s] - fb[sl_b]))
    err_wall = np.max(np.abs(f0[sl_s] - fb[sl_b]))
    assert err_pml < tol * peak
    assert err_wall > 100 * err_pml                        # the wave did reach the boundary


def test_p9_late_time_decay_in_cpml_box():
    """6000 steps in a CPML box with a strongly heterogeneous medium extruded into the PML (R9):
    after the source stops, the exact discrete energy W (the P2 invariant) never increases -- the
    CPML only removes energy -- and the run stays finite.  (A soft Ez dipole leaves a static charge
    behind, so W settles on the electrostatic energy instead of zero.)"""
    n, d = 24, 6
    rng = _rng(31)
    eps = wl.extrude_into_pml(1.0 + 11.25 * rng.random((n, n, n)), d)
    ie = 1.0 / eps
    o = Oracle(n, n, n, S, pml_cells=d)
    f = np.zeros((6, n, n, n))
    c = n // 2
    wav = wl.gaussian_sine(6000, 40, 12, 20)
    src = [wl.Source(2, (c, c, c), (c + 1, c + 1, c + 1), wav)]
    o.forward(f, ie, sources=src, n_steps=200)
    W = []
    for blk in range(29):                                  # 200-step blocks up to 6000 steps
        o.forward(f, ie, n_steps=199, reset_psi=False)
        Hprev = f[3:].copy()
        o.forward(f, ie, n_steps=1, reset_psi=False)
        W.append(np.sum(f[:3] ** 2 / ie) + np.sum(f[3:] * Hprev))
    W = np.array(W)
    assert np.all(np.isfinite(W)) and W[0] > 0
    assert np.all(np.diff(W) <= 1e-12 * W[0])
    assert W[-1] < 0.3 * W[0]


# ----------------------------------------------------------------------------- P10
def test_p10_linearity_and_null():
    w = wl.tiny_pml(n_steps=25)
    shape = (6, w.nz, w.ny, w.nx)
    o = Oracle(**w.grid_kwargs())
    z = np.zeros(shape)
    out = o.forward(z, w.inv_eps, w.meta["inv_mu"], [], w.detectors, w.n_steps)
    assert np.all(z == 0) and all(np.all(P == 0) for P in out["phasors"])

    def run(srcs):
        f = np.zeros(shape)
        out = o.forward(f, w.inv_eps, w.meta["inv_mu"], srcs, w.detectors, w.n_steps)
        return f, out["phasors"][0]

    s1, s2 = w.sources
    f1, p1 = run([s1])
    f2, p2 = run([s2])
    a, b = 0.7, -1.3
    sa = wl.Source(s1.component, s1.lo, s1.hi, (a * s1.waveform.astype(np.float64)), s1.profile)
    sb = wl.Source(s2.component, s2.lo, s2.hi, (b * s2.waveform.astype(np.float64)), s2.profile)
    f12, p12 = run([sa, sb])
    assert np.max(np.abs(f12 - (a * f1 + b * f2))) < 1e-12
    assert np.max(np.abs(p12 - (a * p1 + b * p2))) < 1e-12


def test_p10_detector_is_plain_dft_of_the_time_series():
    """Phasor == sum_n F^{n+1} exp(-i omega (n+1)) built from per-step snapshots (reading R13)."""
    w = wl.tiny_pml(n_steps=20)
    o = Oracle(**w.grid_kwargs())
    f = np.zeros((6, w.nz, w.ny, w.nx))
    det = w.detectors[0]
    acc = np.zeros(det.phasor_shape[:-1], dtype=complex)
    comps = [c for c in range(6) if (det.component_mask >> c) & 1]
    for n in range(w.n_steps):
        s = [wl.Source(q.component, q.lo, q.hi, np.roll(q.waveform, -n), q.profile) for q in w.sources]
        o.forward(f, w.inv_eps, w.meta["inv_mu"], s, [], 1, reset_psi=(n == 0))
        for fi, om in enumerate(det.omega):
            for ci, c in enumerate(comps):
                box = f[c, det.lo[2]:det.hi[2], det.lo[1]:det.hi[1], det.lo[0]:det.hi[0]]
                acc[fi, ci] += box * np.exp(-1j * om * (n + 1))
    f2 = np.zeros_like(f)
    P = o.forward(f2, w.inv_eps, w.meta["inv_mu"], w.sources, w.detectors, w.n_steps)["phasors"][0]
    assert np.max(np.abs(f - f2)) < 1e-14
    assert np.max(np.abs(P[..., 0] - acc.real)) < 1e-12 and np.max(np.abs(P[..., 1] - acc.imag)) < 1e-12


# ----------------------------------------------------------------------------- P11
def test_p11_paper_step_counts_fix_the_courant_convention(golden_dir):
    """Table 2 / sections 3.2-3.3 step counts are reproduced by dt = S dx / c with S = 0.99/sqrt(3)
    and steps = round(T/dt) -- and by no other reading (S = 0.99, or ceil/floor)."""
    c0 = 299792458.0
    rows = [l.split() for l in (golden_dir / "paper_table2_steps.txt").read_text().splitlines()
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 6
    for T_fs, res_nm, steps in rows:
        ratio = float(T_fs) * 1e-15 * c0 / (wl.COURANT * float(res_nm) * 1e-9)
        assert round(ratio) == int(steps), (T_fs, res_nm, ratio)
        wrong = float(T_fs) * 1e-15 * c0 / (0.99 * float(res_nm) * 1e-9)
        assert round(wrong) != int(steps)
    # 300 fs @ 100 nm is 1573.50 -> 1574: round, not floor
    r = 300e-15 * c0 / (wl.COURANT * 100e-9)
    assert math.floor(r) == 1573 and round(r) == 1574


# ----------------------------------------------------------------------------- tables
def test_cpml_tables_structure():
    """Interior: a=0, ik=1 (update reduces to the plain curl, hence exactly invertible);
    PML: 0<b<1, a<0, ik<=1, monotone in depth; E tables at p, H tables at p+1/2 (mirror symmetry)."""
    n, d = 30, 8
    o = Oracle(n, n, n, S, pml_cells=d, pml_kappa_max=3.0, pml_alpha_max=0.05)
    bE, aE, kE = o.cpml_table(0, 0)
    bH, aH, kH = o.cpml_table(0, 1)
    assert np.all(aE[d:n - d + 1] == 0) and np.all(kE[d:n - d + 1] == 1)
    assert np.all(aH[d:n - d] == 0) and np.all(kH[d:n - d] == 1)
    assert np.all(aE[:d] < 0) and np.all(aE[n - d + 1:] < 0) and np.all(aH[:d] < 0) and np.all(aH[n - d:] < 0)
    assert np.all((bE[:d] > 0) & (bE[:d] < 1))
    assert np.all(np.diff(kE[:d + 1]) > 0) and np.all(np.diff(bE[:d]) > 0)
    # mirror symmetry: E position p mirrors to n-p, H position p+1/2 mirrors to n-1-p+1/2
    assert np.allclose(bE[1:], bE[1:][::-1]) and np.allclose(aH, aH[::-1]) and np.allclose(kH, kH[::-1])
    # defaults (R8): kappa=1, alpha=0 => a = b-1, sigma_max = 0.8*(m+1)/sqrt(eps_bg), m=3
    o2 = Oracle(n, n, n, S, pml_cells=d, pml_eps_bg=2.085)
    b2, a2, k2 = o2.cpml_table(2, 0)
    assert np.all(k2 == 1) and np.allclose(a2[:d], b2[:d] - 1)
    assert math.isclose(b2[0], math.exp(-(3.2 / math.sqrt(2.085)) * S), rel_tol=1e-14)


# ----------------------------------------------------------------------------- CPML coefficients a, b
def _cpml_profile(n, d, half, m=3.0, sigma_max=0.8 * 4.0, kappa_max=3.0, alpha_max=0.05, alpha_m=1.0):
    """sigma~, kappa, alpha~ of reading R8 at the table positions (x = p, or p + 1/2 when `half`), recomputed here."""
    x = np.arange(n, dtype=np.float64) + (0.5 if half else 0.0)
    rho = np.maximum(0.0, np.maximum(d - x, x - (n - d)))
    r = rho / d
    inside = rho > 0
    sig = np.where(inside, sigma_max * r ** m, 0.0)
    kap = np.where(inside, 1.0 + (kappa_max - 1.0) * r ** m, 1.0)
    alp = np.where(inside, alpha_max * (1.0 - r) ** alpha_m, 0.0)
    return inside, sig, kap, alp


@pytest.mark.parametrize("kappa_max,alpha_max", [(3.0, 0.05), (1.0, 0.0), (2.0, 0.3)])
def test_cpml_zero_frequency_limit_of_the_stretch_factor(kappa_max, alpha_max):
    """PAPER.md L72 (CPML, ref. 7): the stretched derivative is d/s with s(w) = kappa + sigma/(alpha + i w eps0).
    A constant input d drives psi to a d/(1-b), so the recursion's DC gain 1/kappa + a/(1-b) must equal
    1/s(0) = 1/(kappa + sigma~/alpha~) = alpha~/(sigma~ + kappa alpha~)  (0 where alpha~ = 0), at every PML position
    of both staggerings.  A kappa dropped from a's denominator, or a sign slip, fails this."""
    n, d = 30, 8
    o = Oracle(n, n + 2, n + 4, S, pml_cells=d, pml_kappa_max=kappa_max, pml_alpha_max=alpha_max)
    seen_alpha_zero = seen_alpha_pos = False
    for axis, na in enumerate((n, n + 2, n + 4)):
        for half in (0, 1):
            b, a, ik = o.cpml_table(axis, half)
            inside, sig, kap, alp = _cpml_profile(na, d, half, kappa_max=kappa_max, alpha_max=alpha_max)
            assert inside.sum() in (2 * d, 2 * d - 1)
            dc = ik + np.where(inside, a / np.where(inside, 1.0 - b, 1.0), 0.0)
            want = np.where(inside, alp / np.where(inside, sig + kap * alp, 1.0), 1.0)
            assert np.max(np.abs(dc - want)) < 1e-13, (axis, half)
            seen_alpha_zero |= bool(np.any(inside & (alp == 0)))
            seen_alpha_pos |= bool(np.any(inside & (alp > 0)))
    assert seen_alpha_zero and (seen_alpha_pos or alpha_max == 0)


def test_cpml_coefficients_are_the_integrated_impulse_response():
    """Ref. 7's recursive convolution: 1/s(w) = 1/kappa + FT[zeta], zeta(t) = -(sigma~ S/kappa^2) exp(-(sigma~/kappa + alpha~) S t)
    (t in steps; (sigma/eps0) dt = sigma~ S), and psi_n = sum_m Z(m) d_{n-m} with Z(m) the integral of zeta over [m, m+1].
    The tables must satisfy a = Z(0) and a b = Z(1): checked by Gauss-Legendre quadrature of zeta, which pins a and b
    (exponent, the factor S, kappa in both places) without retyping their closed forms."""
    n, d, kmax, amax = 26, 7, 3.0, 0.05
    o = Oracle(n, n, n, S, pml_cells=d, pml_kappa_max=kmax, pml_alpha_max=amax, pml_eps_bg=2.085)
    xg, wg = np.polynomial.legendre.leggauss(24)
    for half in (0, 1):
        b, a, ik = o.cpml_table(1, half)
        inside, sig, kap, alp = _cpml_profile(n, d, half, sigma_max=0.8 * 4.0 / math.sqrt(2.085), kappa_max=kmax, alpha_max=amax)
        for p in np.nonzero(inside)[0]:
            zeta = lambda t: -(sig[p] * S / kap[p] ** 2) * np.exp(-(sig[p] / kap[p] + alp[p]) * S * t)
            Z0 = 0.5 * np.sum(wg * zeta(0.5 * (xg + 1.0)))
            Z1 = 0.5 * np.sum(wg * zeta(1.0 + 0.5 * (xg + 1.0)))
            assert abs(a[p] - Z0) < 1e-13 and abs(a[p] * b[p] - Z1) < 1e-13, (half, p, a[p], Z0)
            assert abs(ik[p] - 1.0 / kap[p]) < 1e-15


# ----------------------------------------------------------------------------- B6
def test_b6_rho_chain_rule_against_finite_differences():
    """SURVEY 8(a) B6 / reading R20: eps = eps_bg + delta_eps rho on a design box, solver input inv_eps = 1/eps.
    dL/drho from the oracle (time-reversed gradient, then orc_grad_rho) against central finite differences of the
    loss with respect to single rho voxels on the tiny CPML grid (box offset from the origin, inside I)."""
    w = wl.tiny_pml(n_steps=30)
    shape = (w.nz, w.ny, w.nx)
    d = w.pml_cells
    lo, hi = (d + 1, d + 1, d + 1), (w.nx - d - 1, w.ny - d, w.nz - d - 1)          # (i,j,k), inside I = [d, N-d)
    box = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
    eps_bg, delta_eps = 1.5, 2.5
    rho = _rng(17).random((hi[2] - lo[2], hi[1] - lo[1], hi[0] - lo[0]))
    wfield = _rng(18).random((6,) + shape)

    def inv_eps_of(rho_):
        ie = w.inv_eps.astype(np.float64).copy()
        ie[box] = 1.0 / (eps_bg + delta_eps * rho_)
        return ie

    ie = inv_eps_of(rho)
    o, f, out, L, dLp, dLf = _run_loss(w, ie, wfield, record=True)
    g, _ = o.backward(f, ie, w.meta["inv_mu"], w.sources, w.detectors, dLp, dLf, w.n_steps, out["rec"])
    dL_drho = o.grad_rho(g, ie, delta_eps, lo, hi)
    assert dL_drho.shape == rho.shape
    scale = np.max(np.abs(dL_drho))
    assert scale > 0
    h = 1e-6
    for v in [(0, 0, 0), (1, 2, 3), (rho.shape[0] - 1, rho.shape[1] - 1, rho.shape[2] - 1), (2, 0, 1)]:
        rp, rm = rho.copy(), rho.copy()
        rp[v] += h
        rm[v] -= h
        fd = (_run_loss(w, inv_eps_of(rp), wfield)[3] - _run_loss(w, inv_eps_of(rm), wfield)[3]) / (2 * h)
        assert abs(fd - dL_drho[v]) < 2e-6 * scale + 1e-6 * abs(fd), (v, fd, dL_drho[v])
