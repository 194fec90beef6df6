"""GPU parity for SURVEY 8(f) N2: time-domain snapshot / energy detectors and their
transposes, Poynting flux from phasors with and without Yee co-location and its VJP, the one-directional TFSF plane
source -- the CUDA path through the C ABI against the fp64 oracle on the same seeded inputs (readings R23-R25).
Tolerances as in test_gpu_parity.py: fields 1e-5, phasor-level quantities 1e-4, gradients 1e-3 (R19 metric)."""
import numpy as np
import pytest

from paper_2412_12360_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_FIELD, TOL_PHASOR, TOL_GRAD = 1e-5, 1e-4, 1e-3


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2412_12360_b200 import binding
    return binding


def relerr(x, ref):
    ref = np.asarray(ref, dtype=np.float64)
    x = np.asarray(x, dtype=np.float64)
    den = np.max(np.abs(ref))
    return float(np.max(np.abs(x - ref)) / den) if den > 0 else float(np.max(np.abs(x)))


def _time_detector_case(B, w, path, td, record_mode=1, grad_box=None):
    """Forward with time-domain detectors, loss linear in their outputs (fixed seeded weights), backward."""
    import torch
    from oracle.oracle import Oracle
    rng = np.random.default_rng(11)
    cots = [rng.standard_normal(t.out_shape(w.n_steps)).astype(np.float32) for t in td]
    im = w.meta.get("inv_mu")
    # oracle
    o = Oracle(**w.grid_kwargs())
    fr = np.zeros((6, w.nz, w.ny, w.nx))
    out = o.forward(fr, w.inv_eps, im, w.sources, [], w.n_steps, record=True, time_detectors=td)
    g_ref, lam_ref = o.backward(fr, w.inv_eps, im, w.sources, [], None, None, w.n_steps, out["rec"],
                                time_detectors=td, dL_dtime=cots)
    # GPU
    kw = w.grid_kwargs()
    kw.update(max_steps=w.n_steps, record=record_mode, path=path)
    if grad_box:
        kw.update(grad_lo=grad_box[0], grad_hi=grad_box[1])
    g = B.Grid(**kw)
    f = torch.zeros((6, w.nz, w.ny, w.nx), device="cuda")
    ie = torch.as_tensor(w.inv_eps).cuda()
    imt = None if im is None else torch.as_tensor(im).cuda()
    g.forward(f, ie, imt, w.sources, [], w.n_steps, time_detectors=td)
    torch.cuda.synchronize()
    for t, got, want in zip(td, g.time_outputs, out["time_outputs"]):
        e = relerr(got.cpu().numpy(), want)
        assert e <= (TOL_PHASOR if t.kind == "energy" else TOL_FIELD), (t.kind, e)
    grad, lam0 = g.backward(f, ie, imt, w.sources, [], None, None, w.n_steps, want_dL_dfields0=True,
                            time_detectors=td, dL_dtime=[torch.as_tensor(c).cuda() for c in cots])
    torch.cuda.synchronize()
    info = g.info()
    gg, ll = grad.cpu().numpy(), lam0.cpu().numpy()
    g.close()
    if grad_box:
        lo, hi = grad_box
        mask = np.zeros_like(g_ref, dtype=bool)
        mask[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] = True
        g_ref = np.where(mask, g_ref, 0.0)
    eg, el = relerr(gg, g_ref), relerr(ll, lam_ref)
    assert eg <= TOL_GRAD and el <= TOL_GRAD, (eg, el)
    return info


def test_time_detectors_tiny_every_term(B):
    """Tiny CPML grid with kappa, alpha, inv_mu, E and H sources (generic kernels: nx % 4 != 0)."""
    w = wl.tiny_pml(n_steps=30)
    d = w.pml_cells
    td = [wl.TimeDetector("energy", (d, d, d), (w.nx - d, w.ny - d, w.nz - d), stride=3),
          wl.TimeDetector("snapshot", (d + 1, d, d + 1), (w.nx - d, w.ny - d - 1, w.nz - d), stride=4, component_mask=0b011011)]
    _time_detector_case(B, w, B.FDTD_PATH_GENERIC, td)


@pytest.mark.parametrize("with_mu", [False, True])
@pytest.mark.parametrize("record_mode", [1, 2])
def test_time_detectors_on_the_fused_path(B, with_mu, record_mode):
    """C3 miniature on the fused kernels (ping-pong volumes, im lamH carried by the sweep when inv_mu is given):
    an energy detector inside the reconstruction box, a snapshot detector that reaches into the PML."""
    w = wl.c3_mini(n_steps=90)
    if with_mu:
        rng = np.random.default_rng(5)
        w.meta["inv_mu"] = (1.0 / (1.0 + 0.5 * rng.random((w.nz, w.ny, w.nx), dtype=np.float32))).astype(np.float32)
    lo, hi = w.design_lo, w.design_hi
    td = [wl.TimeDetector("energy", lo, hi, stride=7),
          wl.TimeDetector("snapshot", (2, 3, lo[2]), (w.nx - 6, w.ny - 2, lo[2] + 2), stride=10, component_mask=0b101101)]
    info = _time_detector_case(B, w, B.FDTD_PATH_FUSED, td, record_mode=record_mode, grad_box=(lo, hi))
    assert info.path == B.FDTD_PATH_FUSED


def _flux_detector(w, axis, p, thick):
    d = w.pml_cells
    lo, hi = [d, d, d], [w.nx - d, w.ny - d, w.nz - d]
    lo[axis], hi[axis] = p - (thick - 1), p + 1
    b, c = (axis + 1) % 3, (axis + 2) % 3
    mask = (1 << b) | (1 << c) | (1 << (3 + b)) | (1 << (3 + c)) | (1 << axis)      # one extra component: slots are not 0..3
    return wl.Detector(mask, tuple(lo), tuple(hi), [wl.omega_ppw(12), wl.omega_ppw(17)])


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("interpolate", [False, True])
def test_flux_and_its_vjp(B, axis, interpolate):
    """Flux through a plane normal to every axis from the phasors the GPU accumulated, and the VJP that turns
    dL/dflux into the phasor cotangent, against the oracle's statement of reading R24 on the same phasors."""
    import torch
    from oracle.oracle import Oracle
    w = wl.c3_mini(nx=40, ny=36, nz=32, d=6, n_steps=80)
    det = _flux_detector(w, axis, [26, 22, 20][axis], 2 if interpolate else 1)
    g = B.Grid(**{**w.grid_kwargs(), "max_steps": w.n_steps})
    f = torch.zeros((6, w.nz, w.ny, w.nx), device="cuda")
    ie = torch.as_tensor(w.inv_eps).cuda()
    ph = g.forward(f, ie, None, w.sources, [det], w.n_steps)[0]
    fl = g.flux(det, ph, axis, interpolate)
    Gf = np.array([0.7, -1.3], dtype=np.float32)
    dP = g.flux_vjp(det, ph, axis, interpolate, Gf)
    torch.cuda.synchronize()
    o = Oracle(**w.grid_kwargs())
    P = ph.cpu().numpy().astype(np.float64)
    fl_ref = o.flux(det, P, axis, interpolate)
    dP_ref = o.flux_vjp(det, P, axis, interpolate, Gf.astype(np.float64))
    g.close()
    assert np.max(np.abs(fl_ref)) > 0
    # the flux is a difference of two products summed over the plane: error relative to the sum of magnitudes' scale
    assert relerr(fl.cpu().numpy(), fl_ref) <= TOL_PHASOR, (fl.cpu().numpy(), fl_ref)
    assert relerr(dP.cpu().numpy(), dP_ref) <= TOL_FIELD


def test_flux_rejects_a_detector_without_the_tangential_components(B):
    import torch
    w = wl.c3_mini(nx=40, ny=36, nz=32, d=6, n_steps=4)
    det = wl.Detector(0b000011, (6, 6, 20), (34, 30, 21), [0.3])
    g = B.Grid(**{**w.grid_kwargs(), "max_steps": 4})
    ph = torch.zeros(det.phasor_shape, device="cuda")
    with pytest.raises(B.FdtdError) as e:
        g.flux(det, ph, 2, False)
    assert e.value.code == B.FDTD_EINVAL
    det2 = _flux_detector(w, 2, 20, 1)
    with pytest.raises(B.FdtdError):
        g.flux(det2, torch.zeros(det2.phasor_shape, device="cuda"), 2, True)       # needs two planes
    g.close()


@pytest.mark.parametrize("axis,pol,direction", [(2, 1, 1), (2, 0, -1), (0, 2, 1), (1, 0, -1)])
def test_tfsf_plane_source(B, axis, pol, direction):
    """The helper's two waveforms against the oracle's auxiliary grid, then the pair of patches in a 3-D run on the
    GPU: fields equal the oracle's run, the wave leaves to one side only (backward flux <= 1e-5 of the forward flux;
    fp32 rounding in place of the oracle's 1e-12)."""
    import torch
    from oracle.oracle import Oracle
    n_long, n_steps, p0 = 96, 70, 48
    dims = [8, 6, 5]
    dims[axis] = n_long
    if axis != 0:
        dims[0] = 8
    nx, ny, nz = dims
    eps_r, mu_r, ppw = 2.25, 1.0, 14.0
    base = wl.gaussian_sine(n_steps, 24, 7, ppw)
    o = Oracle(nx, ny, nz, wl.COURANT, periodic=True)
    wE_r, wH_r, hc_r, off_r = o.tfsf_plane(wl.COURANT, eps_r, mu_r, axis, pol, direction, base.astype(np.float64))
    g = B.Grid(nx=nx, ny=ny, nz=nz, courant=wl.COURANT, periodic=True, max_steps=n_steps)
    wE, wH, hc, off = g.tfsf_plane(eps_r, mu_r, axis, pol, direction, base)
    torch.cuda.synchronize()
    assert (hc, off) == (hc_r, off_r)
    assert relerr(wE.cpu().numpy(), wE_r) <= TOL_FIELD and relerr(wH.cpu().numpy(), wH_r) <= TOL_FIELD

    def patches(we, wh):
        lo, hi = [0, 0, 0], [nx, ny, nz]
        lo[axis], hi[axis] = p0, p0 + 1
        sE = wl.Source(pol, tuple(lo), tuple(hi), we)
        lo[axis], hi[axis] = p0 + off, p0 + off + 1
        return [sE, wl.Source(hc, tuple(lo), tuple(hi), wh)]

    b, c = (axis + 1) % 3, (axis + 2) % 3
    mask = (1 << b) | (1 << c) | (1 << (3 + b)) | (1 << (3 + c))

    def plane_det(p):
        lo, hi = [0, 0, 0], [nx, ny, nz]
        lo[axis], hi[axis] = p - 1, p + 1
        return wl.Detector(mask, tuple(lo), tuple(hi), [wl.omega_ppw(ppw)])

    dets = [plane_det(p0 + 12 * direction), plane_det(p0 - 12 * direction)]
    ie = np.full((nz, ny, nx), 1.0 / eps_r, dtype=np.float32)
    fr = np.zeros((6, nz, ny, nx))
    o.forward(fr, ie, None, patches(wE_r.astype(np.float32), wH_r.astype(np.float32)), dets, n_steps)
    f = torch.zeros((6, nz, ny, nx), device="cuda")
    ph = g.forward(f, torch.as_tensor(ie).cuda(), None, patches(wE, wH), dets, n_steps)
    fl_front = float(g.flux(dets[0], ph[0], axis, True)[0])
    fl_back = float(g.flux(dets[1], ph[1], axis, True)[0])
    torch.cuda.synchronize()
    fg = f.cpu().numpy()
    g.close()
    assert relerr(fg[:3], fr[:3]) <= TOL_FIELD and relerr(fg[3:], fr[3:]) <= TOL_FIELD
    assert fl_front * direction > 0 and abs(fl_back) <= 1e-5 * abs(fl_front), (fl_front, fl_back)
    idx = np.arange(n_long)
    behind = idx < p0 - 1 if direction > 0 else idx > p0 + 1
    front = np.max(np.abs(fg[:3]))
    assert np.max(np.abs(np.compress(behind, fg, axis=3 - axis))) <= 1e-5 * front


# ----------------------------------------------------------------------------------------------------------- N4
@pytest.mark.parametrize("case", ["tiny-generic", "mini-generic", "mini-fused", "mini-nomu-odd-fused"])
def test_gradient_with_respect_to_inv_mu(B, case):
    """dL/d inv_mu through fdtd_backward_mu against the oracle (loss on phasors and on the final H, so the
    cotangent of H is seeded; every CPML term on the tiny grid; the fused sweep carries im lamH)."""
    import torch
    from oracle.oracle import Oracle
    if case.startswith("tiny"):
        w = wl.tiny_pml(n_steps=30)
    else:
        ns = 121 if "odd" in case else 120
        w = wl.c3_mini(n_steps=ns, kappa_max=3.0, alpha_max=0.05)
        rng = np.random.default_rng(5)
        w.meta["inv_mu"] = None if "nomu" in case else (1.0 / (1.0 + 0.5 * rng.random((w.nz, w.ny, w.nx), dtype=np.float32))).astype(np.float32)
        w.sources.append(wl.Source(4, (20, 12, 22), (60, 40, 23), (0.3 * wl.gaussian_sine(ns, 40, 12, 11)).astype(np.float32)))
    path = B.FDTD_PATH_FUSED if case.endswith("fused") else B.FDTD_PATH_GENERIC
    im = w.meta["inv_mu"]
    o = Oracle(**w.grid_kwargs())
    fr = np.zeros((6, w.nz, w.ny, w.nx))
    out = o.forward(fr, w.inv_eps, im, w.sources, w.detectors, w.n_steps, record=True)
    dLf_r = np.zeros_like(fr)
    dLf_r[3:] = fr[3:]
    g_r, lam_r, gmu_r = o.backward(fr, w.inv_eps, im, w.sources, w.detectors, [2.0 * P for P in out["phasors"]], dLf_r,
                                   w.n_steps, out["rec"], want_grad_mu=True)
    kw = w.grid_kwargs()
    kw.update(max_steps=w.n_steps, record=1, path=path)
    g = B.Grid(**kw)
    f = torch.zeros((6, w.nz, w.ny, w.nx), device="cuda")
    ie, imt = torch.as_tensor(w.inv_eps).cuda(), (None if im is None else torch.as_tensor(im).cuda())
    ph = g.forward(f, ie, imt, w.sources, w.detectors, w.n_steps)
    dLf = torch.zeros_like(f)
    dLf[3:] = f[3:]
    gmu = torch.empty((w.nz, w.ny, w.nx), device="cuda")
    grad, lam0 = g.backward(f, ie, imt, w.sources, w.detectors, [2.0 * P for P in ph], dLf, w.n_steps,
                            want_dL_dfields0=True, grad_mu=gmu)
    torch.cuda.synchronize()
    info = g.info()
    assert info.path == path
    # fused: dL/d inv_mu is formed inside the fused inverse step (one launch per reverse step, and inverse step 0)
    assert info.fused_inverse_launches == (w.n_steps if path == B.FDTD_PATH_FUSED else 0)
    e = (relerr(gmu.cpu().numpy(), gmu_r), relerr(grad.cpu().numpy(), g_r), relerr(lam0.cpu().numpy(), lam_r))
    g.close()
    assert np.max(np.abs(gmu_r)) > 0
    assert max(e) <= TOL_GRAD, e


@pytest.mark.parametrize("case", ["tiny-generic", "mini-generic", "mini-fused", "mini-fused-odd"])
def test_checkpointed_reverse_sweep(B, case):
    """SURVEY 8(f) N4 / PAPER.md L82: record=3, the reverse sweep from checkpoints (no inverse step).  Its gradient is the
    plain reverse-mode derivative on EVERY cell, PML included: compared with the oracle's tape mode (which stores every E-update
    bracket) on the whole grid, and with the time-reversed sweep on the interior."""
    import torch
    from oracle.oracle import Oracle
    if case.startswith("tiny"):
        w = wl.tiny_pml(n_steps=30)
        K = 7
    else:
        n = 61 if case.endswith("odd") else 60
        w = wl.c3_mini(n_steps=n, kappa_max=3.0, alpha_max=0.05)
        rng = np.random.default_rng(5)
        w.meta["inv_mu"] = (1.0 / (1.0 + 0.5 * rng.random((w.nz, w.ny, w.nx), dtype=np.float32))).astype(np.float32)
        # an E source inside the gradient box (its contribution to E' - E is not part of the bracket) and an H source
        w.sources.append(wl.Source(2, (30, 20, 20), (50, 30, 22), (0.4 * wl.gaussian_sine(n, 20, 7, 10)).astype(np.float32)))
        w.sources.append(wl.Source(4, (20, 12, 22), (60, 40, 23), (0.3 * wl.gaussian_sine(n, 25, 9, 11)).astype(np.float32)))
        K = 0 if case.endswith("odd") else 16
    path = B.FDTD_PATH_FUSED if "fused" in case else B.FDTD_PATH_GENERIC
    im = w.meta["inv_mu"]
    o = Oracle(**w.grid_kwargs())
    fr = np.zeros((6, w.nz, w.ny, w.nx))
    out = o.forward(fr, w.inv_eps, im, w.sources, w.detectors, w.n_steps, record=True, tape=True)
    dLf_r = np.zeros_like(fr)
    dLf_r[:3] = 0.5 * fr[:3]
    dLp_r = [2.0 * P for P in out["phasors"]]
    g_tape, lam_tape = o.backward_tape(w.inv_eps, im, w.detectors, dLp_r, dLf_r, w.n_steps, out["tape"])
    kw = w.grid_kwargs()
    kw.update(max_steps=w.n_steps, record=3, path=path, checkpoint_every=K)
    g = B.Grid(**kw)
    f = torch.zeros((6, w.nz, w.ny, w.nx), device="cuda")
    ie, imt = torch.as_tensor(w.inv_eps).cuda(), torch.as_tensor(im).cuda()
    ph = g.forward(f, ie, imt, w.sources, w.detectors, w.n_steps)
    torch.cuda.synchronize()
    assert relerr(f.cpu().numpy()[:3], fr[:3]) <= TOL_FIELD
    dLf = torch.zeros_like(f)
    dLf[:3] = 0.5 * f[:3]
    grad, lam0 = g.backward(f, ie, imt, w.sources, w.detectors, [2.0 * P for P in ph], dLf, w.n_steps, want_dL_dfields0=True)
    torch.cuda.synchronize()
    info = g.info()
    g.close()
    assert info.path == path and info.recorder_bytes > 0
    gg = grad.cpu().numpy()
    d = w.pml_cells
    pml = np.ones_like(g_tape, dtype=bool)
    pml[d:w.nz - d, d:w.ny - d, d:w.nx - d] = False
    assert np.max(np.abs(g_tape[pml])) > 1e-3 * np.max(np.abs(g_tape))          # the PML cells do carry gradient
    assert relerr(gg, g_tape) <= TOL_GRAD and relerr(gg[pml], g_tape[pml]) <= TOL_GRAD, (relerr(gg, g_tape), relerr(gg[pml], g_tape[pml]))
    assert relerr(lam0.cpu().numpy(), lam_tape) <= TOL_GRAD


@pytest.mark.parametrize("case", ["tiny", "mini-generic", "mini-fused", "mini-fused-mu"])
def test_lossy_medium_forward_and_checkpointed_gradient(B, case):
    """SURVEY 8(f) N4, reading R29: a random conductivity volume.  Forward fields and phasors against the oracle's lossy
    update; the gradient from the checkpointed sweep (record=3; the only route: a lossy step cannot be time-reversed) and the
    cotangent of state 0 against the oracle's tape mode, PML cells included.  Both kernel paths (the fused step kernels read
    the conductivity at a thread's own cells; the fused adjoint step leaves lamE' before its scaling by Ca in scratch volumes)."""
    import torch
    from oracle.oracle import Oracle
    path = B.FDTD_PATH_FUSED if "fused" in case else B.FDTD_PATH_GENERIC
    if case == "tiny":
        w = wl.tiny_pml(n_steps=30)
    else:
        w = wl.c3_mini(n_steps=70, kappa_max=3.0, alpha_max=0.05)
        if not case.endswith("mu"):
            w.meta["inv_mu"] = None
        else:
            w.meta["inv_mu"] = (1.0 / (1.0 + 0.5 * np.random.default_rng(8).random((w.nz, w.ny, w.nx), dtype=np.float32))).astype(np.float32)
    shape = (w.nz, w.ny, w.nx)
    sig = (0.25 * np.random.default_rng(12).random(shape, dtype=np.float32)).astype(np.float32)
    im = w.meta["inv_mu"]
    o = Oracle(**w.grid_kwargs())
    o.set_sigma(sig)
    fr = np.zeros((6,) + shape)
    out = o.forward(fr, w.inv_eps, im, w.sources, w.detectors, w.n_steps, tape=True)
    dLf_r = np.zeros_like(fr)
    dLf_r[:3] = 0.5 * fr[:3]
    g_tape, lam_tape = o.backward_tape(w.inv_eps, im, w.detectors, [2.0 * P for P in out["phasors"]], dLf_r, w.n_steps, out["tape"])
    o0 = Oracle(**w.grid_kwargs())
    f0 = np.zeros((6,) + shape)
    o0.forward(f0, w.inv_eps, im, w.sources, w.detectors, w.n_steps)
    assert relerr(fr[:3], f0[:3]) > 1e-2                      # the loss does change the fields
    kw = w.grid_kwargs()
    kw.update(max_steps=w.n_steps, record=3, checkpoint_every=9, path=path)
    g = B.Grid(**kw)
    assert g.info().path == path
    g.set_conductivity(sig)
    f = torch.zeros((6,) + shape, device="cuda")
    ie = torch.as_tensor(w.inv_eps).cuda()
    imt = None if im is None else torch.as_tensor(im).cuda()
    ph = g.forward(f, ie, imt, w.sources, w.detectors, w.n_steps)
    torch.cuda.synchronize()
    fg = f.cpu().numpy()
    assert relerr(fg[:3], fr[:3]) <= TOL_FIELD and relerr(fg[3:], fr[3:]) <= TOL_FIELD
    for P, Pr in zip(ph, out["phasors"]):
        assert relerr(P.cpu().numpy(), Pr) <= TOL_PHASOR
    dLf = torch.zeros_like(f)
    dLf[:3] = 0.5 * f[:3]
    grad, lam0 = g.backward(f, ie, imt, w.sources, w.detectors, [2.0 * P for P in ph], dLf, w.n_steps, want_dL_dfields0=True)
    torch.cuda.synchronize()
    info = g.info()
    g.close()
    # forward + replayed forward + adjoint sweep, each w.n_steps launches of the fused step kernel
    assert info.fused_step_launches == (3 * w.n_steps if path == B.FDTD_PATH_FUSED else 0)
    assert relerr(grad.cpu().numpy(), g_tape) <= TOL_GRAD and relerr(lam0.cpu().numpy(), lam_tape) <= TOL_GRAD
    # record = 0: forward and the adjoint sweep alone (no gradient, nothing to reverse) take the lossy medium as well
    g0 = B.Grid(**{**w.grid_kwargs(), "max_steps": w.n_steps, "record": 0, "path": path})
    g0.set_conductivity(sig)
    f0g = torch.zeros((6,) + shape, device="cuda")
    ph0 = g0.forward(f0g, ie, imt, w.sources, w.detectors, w.n_steps)
    dLf0 = torch.zeros_like(f0g)
    dLf0[:3] = 0.5 * f0g[:3]
    _, lam00 = g0.backward(f0g, ie, imt, w.sources, w.detectors, [2.0 * P for P in ph0], dLf0, w.n_steps, want_grad=False)
    torch.cuda.synchronize()
    info0 = g0.info()
    g0.close()
    assert info0.fused_step_launches == (2 * w.n_steps if path == B.FDTD_PATH_FUSED else 0)
    assert relerr(f0g.cpu().numpy(), fr) <= TOL_FIELD and relerr(lam00.cpu().numpy(), lam_tape) <= TOL_GRAD
    # a recording grid refuses a lossy medium
    g1 = B.Grid(**{**w.grid_kwargs(), "max_steps": 4, "record": 1})
    with pytest.raises(B.FdtdError) as e:
        g1.set_conductivity(sig)
    assert e.value.code == B.FDTD_ESTATE
    g1.close()


@pytest.mark.parametrize("case", ["tiny-reversible", "mini-reversible", "mini-checkpointed-lossy", "mini-fused-reversible",
                                  "mini-fused-checkpointed-lossy", "mini-fused-reversible-box"])
def test_per_component_inv_eps(B, case):
    """SURVEY 8(f) N4, reading R30 (FDTD_FLAG_ANISO_EPS): three inv_eps volumes, three gradient volumes.  Fields, phasors and the
    time-reversed gradient against the oracle; with a conductivity, the checkpointed gradient against the oracle's tape mode."""
    import torch
    from oracle.oracle import Oracle
    w = wl.tiny_pml(n_steps=30) if case.startswith("tiny") else wl.c3_mini(n_steps=70, kappa_max=3.0, alpha_max=0.05)
    shape = (w.nz, w.ny, w.nx)
    rng = np.random.default_rng(4)
    ie3 = (np.stack([w.inv_eps] * 3) * (0.8 + 0.4 * rng.random((3,) + shape, dtype=np.float32))).astype(np.float32)
    lossy = case.endswith("lossy")
    sig = (0.2 * rng.random(shape, dtype=np.float32)).astype(np.float32) if lossy else None
    im = w.meta.get("inv_mu")
    o = Oracle(**w.grid_kwargs())
    o.set_aniso(True)
    if lossy:
        o.set_sigma(sig)
    fr = np.zeros((6,) + shape)
    out = o.forward(fr, ie3, im, w.sources, w.detectors, w.n_steps, record=not lossy, tape=lossy)
    dLf_r = np.zeros_like(fr)
    dLf_r[:3] = 0.5 * fr[:3]
    dLp_r = [2.0 * P for P in out["phasors"]]
    fin = fr.copy()
    if lossy:
        g_r, lam_r = o.backward_tape(ie3, im, w.detectors, dLp_r, dLf_r, w.n_steps, out["tape"])
    else:
        g_r, lam_r = o.backward(fr, ie3, im, w.sources, w.detectors, dLp_r, dLf_r, w.n_steps, out["rec"])
    kw = w.grid_kwargs()
    path = B.FDTD_PATH_FUSED if "fused" in case else B.FDTD_PATH_GENERIC
    kw.update(max_steps=w.n_steps, record=3 if lossy else 1, flags=B.FDTD_FLAG_ANISO_EPS, path=path)
    if case.endswith("box"):            # the design-box recorder (record=2): the fused inverse step masks the box edges
        kw.update(record=2, grad_lo=w.design_lo, grad_hi=w.design_hi)
    g = B.Grid(**kw)
    assert g.info().path == path
    if lossy:
        g.set_conductivity(sig)
    f = torch.zeros((6,) + shape, device="cuda")
    ie = torch.as_tensor(ie3).cuda()
    imt = None if im is None else torch.as_tensor(im).cuda()
    ph = g.forward(f, ie, imt, w.sources, w.detectors, w.n_steps)
    torch.cuda.synchronize()
    fg = f.cpu().numpy()
    assert relerr(fg[:3], fin[:3]) <= TOL_FIELD and relerr(fg[3:], fin[3:]) <= TOL_FIELD
    for P, Pr in zip(ph, out["phasors"]):
        assert relerr(P.cpu().numpy(), Pr) <= TOL_PHASOR
    dLf = torch.zeros_like(f)
    dLf[:3] = 0.5 * f[:3]
    grad, lam0 = g.backward(f, ie, imt, w.sources, w.detectors, [2.0 * P for P in ph], dLf, w.n_steps, want_dL_dfields0=True)
    torch.cuda.synchronize()
    info = g.info()
    g.close()
    if path == B.FDTD_PATH_FUSED:
        assert info.fused_step_launches == (3 if lossy else 2) * w.n_steps
        assert info.fused_inverse_launches == (0 if lossy else w.n_steps)
    else:
        assert info.fused_step_launches == 0
    assert tuple(grad.shape) == (3,) + shape
    gg = grad.cpu().numpy()
    for c in range(3):
        assert np.max(np.abs(g_r[c])) > 0
    if case.endswith("box"):
        lo, hi = w.design_lo, w.design_hi
        box = (slice(None), slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
        assert np.max(np.abs(g_r[box])) > 0
        assert relerr(gg[box], g_r[box]) <= TOL_GRAD
    else:
        assert relerr(gg, g_r) <= TOL_GRAD
    assert relerr(lam0.cpu().numpy(), lam_r) <= TOL_GRAD


def test_bandwidth_probe_touches_every_cell(B):
    """bench.py --probe: the probe kernels (include/fdtd.h fdtd_probe_bandwidth) must move ALL of the 7 + 6 volumes, or the rate they
    report is not the rate of the step kernel's bytes: out[c] = in[c] + 0.5 * in[6] * in[(c + 1) % 6] on every cell, for the
    streaming pattern and for the tile-column traversal with a ragged last tile column, ragged runs and every unroll."""
    import torch
    nx, ny, nz = 40, 23, 19
    vin = torch.rand((7, nz, ny, nx), device="cuda")
    want = torch.stack([vin[c] + 0.5 * vin[6] * vin[(c + 1) % 6] for c in range(6)])
    st = torch.cuda.current_stream().cuda_stream
    for pattern, ty, runs, unroll, blocks, threads in ((0, 0, 1, 1, 7, 64), (0, 0, 3, 1, 300, 256), (1, 7, 5, 1, 0, 96), (1, 7, 4, 2, 0, 384),
                                                       (1, 5, 19, 4, 0, 64), (1, 30, 1, 2, 0, 512)):
        vout = torch.full((6, nz, ny, nx), float("nan"), device="cuda")
        gbs = B.fdtd_probe_bandwidth(pattern, nx, ny, nz, ty, runs, unroll, blocks, threads, 2, vin, vout, st)
        assert gbs > 0
        assert torch.allclose(vout, want, rtol=1e-6, atol=1e-7), (pattern, ty, runs, unroll)     # fused multiply-add vs two roundings; NaN = not written
    # patterns 2 / 3: the same traversal on ping-pong volumes (the first six volumes of `in` and `out` swap roles with every
    # launch, plain copies), upwards every time or with the direction alternating: every cell of both sets is written
    keep = vin.clone()
    for pattern, ty, runs, unroll, threads in ((2, 7, 5, 2, 96), (3, 7, 4, 1, 384), (3, 5, 19, 4, 64), (3, 30, 1, 2, 512)):
        vout = torch.full((6, nz, ny, nx), float("nan"), device="cuda")
        vin[:6] = keep[:6] + 0.0
        gbs = B.fdtd_probe_bandwidth(pattern, nx, ny, nz, ty, runs, unroll, 0, threads, 2, vin, vout, st)
        assert gbs > 0
        assert torch.equal(vout, keep[:6]) and torch.equal(vin, keep), (pattern, ty, runs, unroll)
    for bad in (dict(nx=42), dict(threads=100), dict(pattern=4), dict(pattern=1, unroll=3), dict(pattern=1, runs=nz + 1), dict(pattern=0, blocks=0)):
        a = dict(pattern=0, nx=nx, ny=ny, nz=nz, tile_y=7, runs=2, unroll=1, blocks=8, threads=128)
        a.update(bad)
        with pytest.raises(B.FdtdError) as e:
            B.fdtd_probe_bandwidth(a["pattern"], a["nx"], a["ny"], a["nz"], a["tile_y"], a["runs"], a["unroll"], a["blocks"], a["threads"], 1, vin,
                                   torch.empty_like(want), st)
        assert e.value.code == B.FDTD_EINVAL
