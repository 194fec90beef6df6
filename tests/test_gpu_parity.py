"""GPU parity: the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element on
the same seeded fp32 inputs.  Error metric (reading R19): max-norm relative per group,
max|x_gpu - x_ref| / max|x_ref|.  Tolerances (BASELINE.json north_star / SURVEY 8(c)):
fields <= 1e-5 after 100 fp32 steps, phasors <= 1e-4, gradient <= 1e-3.
"""
import os

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


def paths(B, w):
    """Kernel paths to test on this workload."""
    out = [B.FDTD_PATH_GENERIC]
    d = w.pml_cells
    d4 = (d + 3) // 4 * 4
    # the fused TMA kernels take non-periodic grids with nx % 4 == 0 whose interior leaves room for a tile
    # that touches at most one CPML slab per axis (include/fdtd.h, FDTD_PATH_FUSED)
    fused_ok = not w.periodic and w.nx % 4 == 0 and (d == 0 or (w.nx - 2 * d4 >= 8 and w.ny - 2 * d >= 3))
    if fused_ok and os.environ.get("FDTD_TEST_PATHS", "all") != "generic":
        out.append(B.FDTD_PATH_FUSED)
    return out


def loss_cotangents(w, fields, phasors, interior_only=False):
    """Returns (dL_dphasor list | None, dL_dfields | None) for the workload's loss; works on numpy
    (oracle, fp64) and on torch tensors (GPU) alike."""
    if w.loss == "phasor_power":
        return [2.0 * P if i in w.loss_detectors else None for i, P in enumerate(phasors)], None
    if w.loss in ("final_E2", "final_E2_interior"):
        dLf = fields * 0
        if w.loss == "final_E2":
            dLf[:3] = 2.0 * fields[:3]
        else:
            d = w.pml_cells
            sl = (slice(0, 3), slice(d, w.nz - d), slice(d, w.ny - d), slice(d, w.nx - d))
            dLf[sl] = 2.0 * fields[sl]
        return None, dLf
    return None, None


def run_oracle(w, n_steps=None, backward=True, f0=None, dtype=np.float64):
    from oracle.oracle import Oracle
    n = w.n_steps if n_steps is None else n_steps
    o = Oracle(**w.grid_kwargs(), dtype=dtype)
    f = np.zeros((6, w.nz, w.ny, w.nx), dtype=dtype) if f0 is None else f0.astype(dtype).copy()
    out = o.forward(f, w.inv_eps, w.meta.get("inv_mu"), w.sources, w.detectors, n, record=backward and w.pml_cells > 0)
    res = {"fields": f.copy(), "phasors": out["phasors"]}
    if backward:
        dLp, dLf = loss_cotangents(w, f, out["phasors"])
        g, lam0 = o.backward(f, w.inv_eps, w.meta.get("inv_mu"), w.sources, w.detectors, dLp, dLf, n, out["rec"])
        res.update(grad=g, lam0=lam0, state0=f)
    return res


def run_gpu(B, w, path, n_steps=None, backward=True, f0=None, grad_box=None, record_mode=1, rho_box=None, flags=0):
    import torch
    n = w.n_steps if n_steps is None else n_steps
    kw = w.grid_kwargs()
    kw.update(max_steps=n, record=record_mode if (backward and w.pml_cells > 0) else 0, path=path, flags=flags)
    if grad_box:
        kw.update(grad_lo=grad_box[0], grad_hi=grad_box[1])
    g = B.Grid(**kw)
    f = torch.zeros((6, w.nz, w.ny, w.nx), dtype=torch.float32, device="cuda")
    if f0 is not None:
        f.copy_(torch.as_tensor(f0, dtype=torch.float32))
    ie = torch.as_tensor(w.inv_eps).cuda()
    im = None if w.meta.get("inv_mu") is None else torch.as_tensor(w.meta["inv_mu"]).cuda()
    ph = g.forward(f, ie, im, w.sources, w.detectors, n)
    torch.cuda.synchronize()
    res = {"fields": f.cpu().numpy(), "phasors": [p.cpu().numpy() for p in ph], "info": g.info()}
    if backward:
        dLp, dLf = loss_cotangents(w, f, ph)
        grad, lam0 = g.backward(f, ie, im, w.sources, w.detectors, dLp, dLf, n, want_dL_dfields0=True)
        if rho_box is not None:            # B6 through the ABI: dL/drho on the design box
            lo, hi = rho_box
            drho = torch.empty((hi[2] - lo[2], hi[1] - lo[1], hi[0] - lo[0]), dtype=torch.float32, device="cuda")
            B.fdtd_grad_rho(g.h, grad, ie, float(w.meta["delta_eps"]), lo, hi, drho, g.stream())
            res["dL_drho"] = drho.cpu().numpy()
        torch.cuda.synchronize()
        res.update(grad=grad.cpu().numpy(), lam0=lam0.cpu().numpy(), state0=f.cpu().numpy(), info=g.info())
    g.close()
    return res


def interior(w, a):
    d = w.pml_cells
    return a[..., d:w.nz - d, d:w.ny - d, d:w.nx - d]


def compare(w, gpu, ref, backward=True, tol_field=TOL_FIELD):
    errs = {"E": relerr(gpu["fields"][:3], ref["fields"][:3]), "H": relerr(gpu["fields"][3:], ref["fields"][3:])}
    assert errs["E"] <= tol_field and errs["H"] <= tol_field, errs
    for i, (P, Pr) in enumerate(zip(gpu["phasors"], ref["phasors"])):
        errs[f"P{i}"] = relerr(P, Pr)
        assert errs[f"P{i}"] <= TOL_PHASOR, errs
    if backward:
        errs["grad"] = relerr(gpu["grad"], ref["grad"])
        errs["lam0"] = relerr(gpu["lam0"], ref["lam0"])
        assert errs["grad"] <= TOL_GRAD and errs["lam0"] <= TOL_GRAD, errs
        # reconstructed state 0 on I: absolute residue against the largest field seen at state n
        scale = max(np.max(np.abs(ref["fields"])), 1e-30)
        errs["state0"] = float(np.max(np.abs(interior(w, gpu["state0"]) - interior(w, ref["state0"]))) / scale)
        assert errs["state0"] <= 1e-4, errs
    return errs


# ------------------------------------------------------------------------------------------------
def test_c1_periodic_forward_and_gradient(B):
    """configs[0]: 16^3 periodic, 100 steps, loss = sum E^2, gradient wrt inv_eps (all 4096 voxels)."""
    w = wl.c1()
    ref = run_oracle(w)
    gpu = run_gpu(B, w, B.FDTD_PATH_GENERIC)
    errs = compare(w, gpu, ref)
    assert gpu["info"].path == B.FDTD_PATH_GENERIC
    assert np.max(np.abs(gpu["state0"])) < 1e-4 * np.max(np.abs(ref["fields"]))   # state 0 was all zero
    print("C1", errs)


@pytest.mark.parametrize("kappa,alpha,with_mu", [(3.0, 0.05, True), (0.0, 0.0, False)])
def test_tiny_pml_every_term(B, kappa, alpha, with_mu):
    """14x13x12, d=3: kappa/alpha CPML, E and H sources, inv_mu, 2 components x 2 frequencies.
    nx is not a multiple of 4, so this is the generic path only."""
    w = wl.tiny_pml(n_steps=60, kappa_max=kappa, alpha_max=alpha, with_inv_mu=with_mu)
    ref = run_oracle(w)
    gpu = run_gpu(B, w, B.FDTD_PATH_GENERIC)
    print("tiny", compare(w, gpu, ref))


@pytest.mark.parametrize("kappa,alpha", [(0.0, 0.0), (3.0, 0.05)])
def test_c3_mini_all_paths(B, kappa, alpha):
    """88x52x44 miniature of the graded config: several tiles and ragged tails on every axis;
    forward fields + phasors + reversible gradient + cotangent of state 0, every kernel path."""
    w = wl.c3_mini(kappa_max=kappa, alpha_max=alpha)
    ref = run_oracle(w)
    # conditioning of the workload itself: the fp32 build of the oracle against its fp64 build (the pulse has
    # crossed the detector plane by the end of the run, so the gradient is not dominated by cancellation)
    ref32 = run_oracle(w, dtype=np.float32)
    cond = relerr(ref32["grad"], ref["grad"])
    print("c3-mini oracle fp32 vs fp64: gradient", cond, "phasor", relerr(ref32["phasors"][0], ref["phasors"][0]))
    assert cond <= 1e-4
    assert np.max(np.abs(ref["phasors"][0])) > 0.2 * np.max(np.abs(ref["fields"]))      # the pulse did reach the detector
    for path in paths(B, w):
        gpu = run_gpu(B, w, path)
        assert gpu["info"].path == path
        if path == B.FDTD_PATH_FUSED:
            assert gpu["info"].fused_step_launches == 2 * w.n_steps and gpu["info"].fused_inverse_launches >= w.n_steps
        print("c3-mini path", path, compare(w, gpu, ref))


def test_c3_mini_with_inv_mu_and_h_source(B):
    w = wl.c3_mini(nx=64, ny=40, nz=36, d=6, n_steps=80)
    rng = np.random.default_rng(5)
    w.meta["inv_mu"] = (np.float32(1) / (np.float32(1) + np.float32(0.5) * rng.random((w.nz, w.ny, w.nx), dtype=np.float32))).astype(np.float32)
    w.sources.append(wl.Source(3, (20, 12, 14), (30, 20, 16), (0.3 * wl.gaussian_sine(80, 20, 8, 10)).astype(np.float32)))
    ref = run_oracle(w)
    for path in paths(B, w):
        gpu = run_gpu(B, w, path)
        print("c3-mini mu", path, compare(w, gpu, ref))
        if path == B.FDTD_PATH_FUSED:       # inv_mu goes through the fused adjoint and inverse kernels, not the generic ones
            assert gpu["info"].pipelined_inverse_ctas > 0
            assert gpu["info"].fused_step_launches == 2 * w.n_steps and gpu["info"].fused_inverse_launches == w.n_steps
    # the same with an E-only loss detector: the pipelined (grouped) reverse sweep carries inv_mu too
    w.detectors[0] = wl.Detector(1 << 1, w.detectors[0].lo, w.detectors[0].hi, w.detectors[0].omega)
    ref = run_oracle(w)
    gpu = run_gpu(B, w, B.FDTD_PATH_FUSED)
    print("c3-mini mu, pipelined", compare(w, gpu, ref))
    assert gpu["info"].fused_inverse_launches == w.n_steps + 1      # step n_steps (empty) .. 1 in the groups, step 0 after the loop


def test_fused_inverse_subtracts_h_sources(B):
    """SURVEY B3 (`H' - srcH_n`): an H-component source inside the interior, inv_mu = NULL and an E-only loss
    detector, so the whole reverse sweep runs in the fused kernels (pipelined groups): k_inverse has to take the
    H source out again before it inverts the H update."""
    w = wl.c3_mini(nx=64, ny=40, nz=36, d=6, n_steps=90)
    w.detectors[0] = wl.Detector(1 << 1, w.detectors[0].lo, w.detectors[0].hi, w.detectors[0].omega)
    w.sources.append(wl.Source(4, (18, 10, 12), (31, 19, 15), (0.4 * wl.gaussian_sine(90, 25, 8, 10)).astype(np.float32)))
    w.sources.append(wl.Source(5, (40, 22, 20), (41, 23, 21), (0.3 * wl.gaussian_sine(90, 20, 7, 9)).astype(np.float32)))
    ref = run_oracle(w)
    for path in paths(B, w):
        gpu = run_gpu(B, w, path)
        print("H sources", path, compare(w, gpu, ref))
        if path == B.FDTD_PATH_FUSED:
            assert gpu["info"].fused_inverse_launches == w.n_steps + 1
    # teeth: without the H sources the reconstructed state differs by far more than the tolerance
    w0 = wl.c3_mini(nx=64, ny=40, nz=36, d=6, n_steps=90)
    w0.detectors[0] = w.detectors[0]
    assert relerr(run_oracle(w0)["fields"], ref["fields"]) > 1e-2


def test_fused_path_with_prime_ny_nz(B):
    """Ragged tails with no common factor with any tile height: ny = 53, nz = 47 (nx = 88 as the float4 rows need)."""
    w = wl.c3_mini(nx=88, ny=53, nz=47, d=8, n_steps=100, kappa_max=3.0, alpha_max=0.05)
    ref = run_oracle(w)
    for path in paths(B, w):
        gpu = run_gpu(B, w, path)
        assert gpu["info"].path == path
        print("prime ny nz", path, compare(w, gpu, ref))


def test_more_descriptors_than_the_fused_kernels_hold(B):
    """include/fdtd.h "Kernel paths": 5 sources and 5 detectors on a grid that qualifies for the fused kernels.  Under
    FDTD_PATH_AUTO the forward call runs on the generic kernels and the reverse sweep degrades per feature; the
    result matches the oracle.  FDTD_PATH_FUSED refuses the call with EINVAL."""
    w = wl.c3_mini(nx=64, ny=40, nz=36, d=6, n_steps=70)
    d0 = w.detectors[0]
    for q in range(4):
        w.sources.append(wl.Source(q % 3, (10 + 9 * q, 9 + 3 * q, 9 + 4 * q), (14 + 9 * q, 12 + 3 * q, 10 + 4 * q),
                                   (0.2 * wl.gaussian_sine(70, 15 + 3 * q, 6, 9 + q)).astype(np.float32)))
        w.detectors.append(wl.Detector(1 << (q % 3), (8, 8, 12 + 3 * q), (56, 32, 13 + 3 * q), [wl.omega_ppw(11 + q)]))
    w.loss_detectors = (0, 2, 4)
    assert len(w.sources) == 5 and len(w.detectors) == 5
    ref = run_oracle(w)
    gpu = run_gpu(B, w, B.FDTD_PATH_AUTO)
    assert gpu["info"].path == B.FDTD_PATH_FUSED          # the grid itself is a fused grid
    print("5 sources, 5 detectors", compare(w, gpu, ref))
    with pytest.raises(B.FdtdError) as ei:
        run_gpu(B, w, B.FDTD_PATH_FUSED)
    assert ei.value.code == B.FDTD_EINVAL


def test_b6_grad_rho_parity(B):
    """SURVEY 8(a) B6 / R20 through the ABI: fdtd_grad_rho on the design box (offset from the origin) against the
    oracle's orc_grad_rho applied to the oracle's gradient, element by element, every kernel path."""
    w = wl.c3_mini()
    lo, hi = w.design_lo, w.design_hi
    assert min(lo) > 0
    from oracle.oracle import Oracle
    ref = run_oracle(w)
    ref_drho = Oracle(**w.grid_kwargs()).grad_rho(ref["grad"], w.inv_eps, w.meta["delta_eps"], lo, hi)
    assert ref_drho.shape == w.meta["rho"].shape and np.max(np.abs(ref_drho)) > 0
    for path in paths(B, w):
        for rmode, gbox in ((1, None), (2, (lo, hi))):
            gpu = run_gpu(B, w, path, rho_box=(lo, hi), grad_box=gbox, record_mode=rmode)
            e = relerr(gpu["dL_drho"], ref_drho)
            print("B6 dL/drho", path, "record", rmode, e)
            assert gpu["dL_drho"].shape == ref_drho.shape and e <= TOL_GRAD


def test_c2_fields_at_100_200_and_phasor_at_1000(B):
    """configs[1]: 64^3, d=10, eps block, Ey plane source, Ey DFT plane; forward only."""
    w = wl.c2()
    for n in (100, 200):
        ref = run_oracle(w, n_steps=n, backward=False)
        for path in paths(B, w):
            print("C2", n, path, compare(w, run_gpu(B, w, path, n_steps=n, backward=False), ref, backward=False))
    ref = run_oracle(w, n_steps=1000, backward=False)
    for path in paths(B, w):
        gpu = run_gpu(B, w, path, n_steps=1000, backward=False)
        e = relerr(gpu["phasors"][0], ref["phasors"][0])
        assert e <= TOL_PHASOR, e
        print("C2 phasor", path, e)


def test_c5_small_sweep_point(B):
    """configs[4] at N=64 (d=10, random eps extruded into the PML, dipole, loss = sum E^2 over I)."""
    w = wl.c5(64, n_steps=150)
    ref = run_oracle(w)
    for path in paths(B, w):
        print("C5-64", path, compare(w, run_gpu(B, w, path), ref))


# ------------------------------------------------------------------------------------------------ edge cases
def test_zero_steps_and_walls_without_pml(B):
    import torch
    w = wl.c3_mini(nx=24, ny=20, nz=16, d=0, n_steps=40)
    w.loss, w.loss_detectors = "final_E2", ()
    ref = run_oracle(w)
    for path in paths(B, w):
        print("walls", path, compare(w, run_gpu(B, w, path), ref))
    # n_steps = 0: fields untouched, gradient zero
    f0 = np.random.default_rng(1).standard_normal((6, w.nz, w.ny, w.nx)).astype(np.float32)
    gpu = run_gpu(B, w, B.FDTD_PATH_GENERIC, n_steps=0, f0=f0)
    assert np.array_equal(gpu["fields"], f0) and np.all(gpu["grad"] == 0)
    assert np.array_equal(gpu["lam0"][:3], 2 * f0[:3])


def test_minimum_grid_2d_plus_2(B):
    d = 3
    w = wl.tiny_pml(nx=2 * d + 2, ny=2 * d + 2, nz=2 * d + 2, d=d, n_steps=25, with_inv_mu=False)
    ref = run_oracle(w)
    for path in paths(B, w):
        print("min grid", path, compare(w, run_gpu(B, w, path), ref))


def test_nonzero_initial_state(B):
    w = wl.c3_mini(nx=40, ny=36, nz=32, d=6, n_steps=50)
    f0 = (0.1 * np.random.default_rng(2).standard_normal((6, w.nz, w.ny, w.nx))).astype(np.float32)
    ref = run_oracle(w, f0=f0)
    for path in paths(B, w):
        print("f0", path, compare(w, run_gpu(B, w, path, f0=f0), ref))


def test_grad_box_restricts_the_gradient(B):
    w = wl.c3_mini(nx=40, ny=36, nz=32, d=6, n_steps=50)
    ref = run_oracle(w)
    lo, hi = w.design_lo, w.design_hi
    for path in paths(B, w):
        gpu = run_gpu(B, w, path, grad_box=(lo, hi))
        box = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
        assert relerr(gpu["grad"][box], ref["grad"][box]) <= TOL_GRAD
        mask = np.ones_like(gpu["grad"], bool)
        mask[box] = False
        assert np.all(gpu["grad"][mask] == 0)


def test_gradient_box_recorder(B):
    """record=2: only the faces of the gradient box are recorded and only that box is
    reconstructed; gradient, cotangent of state 0 and the reconstructed state 0 on the box match the oracle,
    whose recorder still works on the whole interior."""
    for kappa, alpha, odd in [(0.0, 0.0, 0), (3.0, 0.05, 1)]:
        w = wl.c3_mini(nx=40, ny=36, nz=32, d=6, n_steps=50 + odd, kappa_max=kappa, alpha_max=alpha)
        ref = run_oracle(w)
        lo, hi = w.design_lo, w.design_hi
        box = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
        scale = np.max(np.abs(ref["fields"]))
        for path in paths(B, w):
            gpu = run_gpu(B, w, path, grad_box=(lo, hi), record_mode=2)
            assert gpu["info"].record_floats_per_step < run_gpu(B, w, path, grad_box=(lo, hi))["info"].record_floats_per_step
            assert relerr(gpu["grad"][box], ref["grad"][box]) <= TOL_GRAD
            assert relerr(gpu["lam0"], ref["lam0"]) <= TOL_GRAD
            for c in range(6):
                assert np.max(np.abs(gpu["state0"][c][box] - ref["state0"][c][box])) / scale <= 1e-4, (path, c)
            mask = np.ones_like(gpu["grad"], bool)
            mask[box] = False
            assert np.all(gpu["grad"][mask] == 0)


@pytest.mark.parametrize("record_mode", [1, 2])
def test_reduced_precision_recorder(B, record_mode):
    """SURVEY 8(f) N1, reduced-precision recorder (FDTD_FLAG_RECORDER_FP16): half the recorder bytes; the interface
    values re-imposed in the reverse sweep carry fp16 rounding (2^-11 relative), so the reconstructed fields and the
    gradient are approximate.  The gradient must stay within the north-star 1e-3 of the fp64 oracle on the C3
    miniature (both kernel paths); the measured error is printed beside the fp32 recorder's."""
    w = wl.c3_mini(n_steps=200)
    ref = run_oracle(w)
    box = (w.design_lo, w.design_hi)
    gref = np.zeros_like(ref["grad"])
    sl = (slice(box[0][2], box[1][2]), slice(box[0][1], box[1][1]), slice(box[0][0], box[1][0]))
    gref[sl] = ref["grad"][sl]
    for path in paths(B, w):
        e32 = relerr(run_gpu(B, w, path, grad_box=box, record_mode=record_mode)["grad"], gref)
        r16 = run_gpu(B, w, path, grad_box=box, record_mode=record_mode, flags=B.FDTD_FLAG_RECORDER_FP16)
        e16 = relerr(r16["grad"], gref)
        print(f"recorder fp32 / fp16, record={record_mode}, path={path}: gradient error {e32:.2e} / {e16:.2e}")
        assert r16["info"].recorder_bytes == r16["info"].record_floats_per_step * 2 * w.n_steps      # 2 bytes per value
        assert e16 <= TOL_GRAD, (e32, e16)


def test_pipelined_reverse_sweep_is_the_same_computation(B, monkeypatch):
    """The reverse sweep is pipelined by default: adjoint step n, inverse step n+1 and the
    injection for step n form one launch group (FDTD_REVERSE_SWEEP=grouped; =split puts them on disjoint SMs;
    =sequential is one kernel after the other).  Same arithmetic in the same order per cell, so gradient,
    cotangent and reconstructed state are bit-identical across the three; all match the oracle."""
    for n_steps, rmode in [(41, 2), (40, 1)]:
        w = wl.c3(n=120, n_steps=n_steps, source_k=38)        # source plane just below the design box (k = 42..78)
        w.loss = "final_E2"
        lo, hi = w.design_lo, w.design_hi
        box = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
        ref = run_oracle(w)
        assert np.max(np.abs(ref["grad"][box])) > 0
        monkeypatch.setenv("FDTD_REVERSE_SWEEP", "sequential")
        base = run_gpu(B, w, B.FDTD_PATH_FUSED, grad_box=(lo, hi), record_mode=rmode)
        assert base["info"].pipelined_inverse_ctas == 0
        assert relerr(base["grad"][box], ref["grad"][box]) <= TOL_GRAD and relerr(base["lam0"], ref["lam0"]) <= TOL_GRAD
        seen = []
        for mode in (None, "split"):
            if mode:
                monkeypatch.setenv("FDTD_REVERSE_SWEEP", mode)
            else:
                monkeypatch.delenv("FDTD_REVERSE_SWEEP")
            pipe = run_gpu(B, w, B.FDTD_PATH_FUSED, grad_box=(lo, hi), record_mode=rmode)
            assert pipe["info"].pipelined_inverse_ctas > 0
            seen.append(pipe["info"].pipelined_inverse_ctas)
            assert np.array_equal(pipe["grad"], base["grad"]) and np.array_equal(pipe["lam0"], base["lam0"])
            for c in range(6):
                assert np.array_equal(pipe["state0"][c][box], base["state0"][c][box])
        assert seen[0] != seen[1]                               # two different launch configurations did run
        monkeypatch.delenv("FDTD_REVERSE_SWEEP", raising=False)


def test_adjoint_sweep_only(B):
    """dL_dinv_eps = NULL (include/fdtd.h): the cotangent of state 0 alone.  It does not depend on the primal
    fields, so it needs no recorded forward, leaves `fields` untouched and is bit-identical to the cotangent the
    full backward pass returns; checked against the oracle on both kernel paths."""
    import torch
    w = wl.c3_mini(n_steps=61, kappa_max=3.0, alpha_max=0.05)
    ref = run_oracle(w)
    for path in paths(B, w):
        full = run_gpu(B, w, path)
        kw = w.grid_kwargs()
        kw.update(max_steps=w.n_steps, record=0, path=path)              # no recorder at all
        g = B.Grid(**kw)
        f = torch.zeros((6, w.nz, w.ny, w.nx), dtype=torch.float32, device="cuda")
        ie = torch.as_tensor(w.inv_eps).cuda()
        ph = g.forward(f, ie, None, w.sources, w.detectors, w.n_steps)
        keep = f.clone()
        dLp, dLf = loss_cotangents(w, f, ph)
        none, lam0 = g.backward(f, ie, None, w.sources, w.detectors, dLp, dLf, w.n_steps, want_grad=False)
        torch.cuda.synchronize()
        assert none is None and torch.equal(f, keep)
        assert np.array_equal(lam0.cpu().numpy(), full["lam0"])
        assert relerr(lam0.cpu().numpy(), ref["lam0"]) <= TOL_GRAD
        with pytest.raises(B.FdtdError):                                  # a gradient still needs the recorded forward
            g.backward(f, ie, None, w.sources, w.detectors, dLp, dLf, w.n_steps)
        g.close()


def test_c3_full_size_truncated_in_the_bench_configuration(B):
    """configs[2] at its full 200^3 size in the launch configuration bench.py times (fused kernels, tile and
    grid chosen by the library, grad box = design region, record=2 and record=1), truncated to 40 time steps
    so that the fp64 oracle finishes in seconds.  The source plane sits just below the design box (k = 66)
    and the loss is sum E^2 at the final state, so fields, gradient and cotangents are non-trivial."""
    w = wl.c3(n_steps=40, source_k=66)
    w.loss = "final_E2"
    # a seeded random initial state (amplitude 0.1, all six components, every cell): every CPML slab, edge and corner
    # cell of the 200 x 7 lock-step configuration is compared on non-zero values
    f0 = (0.1 * np.random.default_rng(40).standard_normal((6, w.nz, w.ny, w.nx))).astype(np.float32)
    ref = run_oracle(w, f0=f0)
    lo, hi = w.design_lo, w.design_hi
    box = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
    assert np.max(np.abs(ref["grad"][box])) > 0
    scale = np.max(np.abs(ref["fields"]))
    d = w.pml_cells
    regions = 0
    for rz in (slice(0, d), slice(d, w.nz - d), slice(w.nz - d, w.nz)):
        for ry in (slice(0, d), slice(d, w.ny - d), slice(w.ny - d, w.ny)):
            for rx in (slice(0, d), slice(d, w.nx - d), slice(w.nx - d, w.nx)):
                for c in range(6):         # reference fields and state-0 cotangents are non-zero in all 27 regions
                    assert np.max(np.abs(ref["fields"][c][rz, ry, rx])) > 1e-3 * scale
                    assert np.max(np.abs(ref["lam0"][c][rz, ry, rx])) > 0
                regions += 1
    assert regions == 27
    for mode in (2, 1):
        gpu = run_gpu(B, w, B.FDTD_PATH_FUSED, grad_box=(lo, hi), record_mode=mode, f0=f0)
        assert gpu["info"].path == B.FDTD_PATH_FUSED
        eE, eH = relerr(gpu["fields"][:3], ref["fields"][:3]), relerr(gpu["fields"][3:], ref["fields"][3:])
        eG, eL = relerr(gpu["grad"][box], ref["grad"][box]), relerr(gpu["lam0"], ref["lam0"])
        e0 = max(float(np.max(np.abs(gpu["state0"][c][box] - ref["state0"][c][box]))) for c in range(6)) / scale
        print("C3 full size, record", mode, "tile", gpu["info"].tile_x, gpu["info"].tile_y, eE, eH, eG, eL, e0)
        assert eE <= TOL_FIELD and eH <= TOL_FIELD and eG <= TOL_GRAD and eL <= TOL_GRAD and e0 <= 1e-4


def test_c3_full_length_self_consistency(B):
    """configs[2] exactly as bench.py runs it: 200^3, all 2000 time steps, loss = DFT phasor power on the output
    plane, record=2, fused kernels with the library's own launch configuration.  The oracle needs minutes for this,
    so the checks are properties: the directional derivative of the loss along delta = sign(dL/d inv_eps) on the
    design box by central finite differences against <dL/d inv_eps, delta>, the state reconstructed by 2000
    inverse steps on the box against its true value 0, and a gradient that vanishes outside the box."""
    import torch
    n = 2000
    w = wl.c3(n_steps=n)
    lo, hi = w.design_lo, w.design_hi
    kw = w.grid_kwargs()
    kw.update(max_steps=n, record=2, grad_lo=lo, grad_hi=hi, path=B.FDTD_PATH_FUSED)
    g = B.Grid(**kw)
    assert g.info().path == B.FDTD_PATH_FUSED and g.info().pipelined_inverse_ctas > 0
    ie = torch.as_tensor(w.inv_eps).cuda()
    box = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
    f = torch.zeros((6, w.nz, w.ny, w.nx), dtype=torch.float32, device="cuda")
    g.forward(f, ie, None, w.sources, w.detectors, 400)
    fmax = float(f.abs().max())                              # field scale while the pulse is inside the grid
    assert fmax > 0

    def run(ie_t):
        f.zero_()
        ph = g.forward(f, ie_t, None, w.sources, w.detectors, n)
        return ph, float(sum((P.double() ** 2).sum() for i, P in enumerate(ph) if i in w.loss_detectors))

    ph, L0 = run(ie)
    assert np.isfinite(L0) and L0 > 0
    dLp = [2.0 * P if i in w.loss_detectors else None for i, P in enumerate(ph)]
    grad, _ = g.backward(f, ie, None, w.sources, w.detectors, dLp, None, n)
    torch.cuda.synchronize()
    resid = max(float(f[c][box].abs().max()) for c in range(6)) / fmax
    delta = torch.zeros_like(ie)
    delta[box] = torch.sign(grad[box])
    an = float((grad.double() * delta.double()).sum())
    h = 2e-4
    fd = (run(ie + h * delta)[1] - run(ie - h * delta)[1]) / (2 * h)
    g.close()
    print("C3 full length: L", L0, "directional derivative analytic", an, "finite difference", fd, "state-0 residue", resid)
    assert an > 0 and abs(fd - an) <= 5e-3 * abs(an)         # measured 2.4e-4
    assert resid <= 1e-5                                     # measured 6.7e-7
    grad[box] = 0
    assert float(grad.abs().max()) == 0.0


def test_c3_full_length_time_reversal_equals_checkpointing(B):
    """configs[2] at its full size and length: the gradient of the time-reversed sweep (record=2, the bench configuration; also
    record=1) against the checkpointed sweep (record=3: no inverse step, nothing reconstructed), which is the
    plain reverse-mode derivative.  Two independent routes to dL/d inv_eps over 2000 steps on 864 000 voxels: they must agree
    to the rounding of the reconstruction (measured 7e-7 of the maximum; the oracle tolerance is 1e-3)."""
    import torch
    n = 2000
    w = wl.c3(n_steps=n)
    lo, hi = w.design_lo, w.design_hi
    box = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
    ie = torch.as_tensor(w.inv_eps).cuda()
    grads = {}
    for rec in (3, 2, 1):
        kw = w.grid_kwargs()
        kw.update(max_steps=n, record=rec, grad_lo=lo, grad_hi=hi, path=B.FDTD_PATH_FUSED)
        g = B.Grid(**kw)
        f = torch.zeros((6, w.nz, w.ny, w.nx), dtype=torch.float32, device="cuda")
        ph = g.forward(f, ie, None, w.sources, w.detectors, n)
        grad, _ = g.backward(f, ie, None, w.sources, w.detectors, [2.0 * P for P in ph], None, n)
        torch.cuda.synchronize()
        grads[rec] = grad[box].double().cpu().numpy()
        g.close()
    scale = np.max(np.abs(grads[3]))
    assert scale > 0
    for rec in (2, 1):
        err = float(np.max(np.abs(grads[rec] - grads[3])) / scale)
        print(f"C3 full length: time-reversed (record={rec}) vs checkpointed gradient: {err:.2e} of the maximum")
        assert err <= 1e-5


def test_c4_full_size_self_consistency(B):
    """configs[3] at its full 800 x 800 x 600 size (384 M cells; maximum size, 6 nc > 2^31 elements) in the
    bench launch configuration (fused kernels, record=2).  The oracle cannot run this size in seconds, so the
    checks are properties that hold at any size: a directional central finite difference of the loss against
    <dL/d inv_eps, delta>, and the reconstructed state 0 (true value 0) on the design box.
    Default: truncated to 24 steps with the source plane moved next to the design box and the loss on the final
    fields.  FDTD_C4_STEPS=5000 runs the config as BASELINE.json states it (source at k = 40, loss = phasor power on
    the far plane; ~4 GPU-minutes; result recorded in profiles/r2_c4_full.md)."""
    import torch
    free, _ = torch.cuda.mem_get_info()
    if free < 100e9:
        pytest.skip("needs ~100 GB of device memory")
    n = int(os.environ.get("FDTD_C4_STEPS", "24"))
    full = n > 1000
    w = wl.c4(n_steps=n)
    d, lo, hi = w.pml_cells, w.design_lo, w.design_hi
    if not full:
        s0 = w.sources[0]
        w.sources[0] = wl.Source(s0.component, (d, d, lo[2] - 4), (w.nx - d, w.ny - d, lo[2] - 3), s0.waveform, s0.profile)
    kw = w.grid_kwargs()
    kw.update(max_steps=n, record=2, grad_lo=lo, grad_hi=hi, path=B.FDTD_PATH_FUSED)
    g = B.Grid(**kw)
    assert g.info().path == B.FDTD_PATH_FUSED
    ie = torch.as_tensor(w.inv_eps).cuda()
    box = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
    f = torch.zeros((6, w.nz, w.ny, w.nx), dtype=torch.float32, device="cuda")
    fmax = 1.0
    if full:
        g.forward(f, ie, None, w.sources, w.detectors, 700)
        fmax = float(f.abs().max())                          # field scale while the pulse is inside the grid

    def loss_of(ie_t):
        f.zero_()
        ph = g.forward(f, ie_t, None, w.sources, w.detectors, n)
        if full:
            return ph, float(sum((P.double() ** 2).sum() for i, P in enumerate(ph) if i in w.loss_detectors))
        return ph, float((f[:3].double() ** 2).sum())

    ph, L0 = loss_of(ie)
    assert np.isfinite(L0) and L0 > 0
    if full:
        dLp = [2.0 * P if i in w.loss_detectors else None for i, P in enumerate(ph)]
        grad, _ = g.backward(f, ie, None, w.sources, w.detectors, dLp, None, n)
    else:
        fmax = float(f.abs().max())
        dLf = torch.zeros_like(f)
        dLf[:3] = 2.0 * f[:3]
        grad, _ = g.backward(f, ie, None, w.sources, w.detectors, None, dLf, n)
        del dLf
    torch.cuda.synchronize()
    resid = max(float(f[c][box].abs().max()) for c in range(6)) / fmax
    delta = torch.zeros_like(ie)
    if full:
        delta[box] = torch.sign(grad[box])
        h = 2e-4
    else:
        gen = torch.Generator(device="cuda").manual_seed(4)
        delta[box] = torch.randint(0, 2, delta[box].shape, generator=gen, device="cuda").float() * 2 - 1
        h = 2e-3
    an = float((grad.double() * delta.double()).sum())
    fd = (loss_of(ie + h * delta)[1] - loss_of(ie - h * delta)[1]) / (2 * h)
    info = g.info()
    g.close()
    print("C4 full size:", n, "steps, L", L0, "directional derivative analytic", an, "finite difference", fd, "state-0 residue", resid,
          "recorder bytes", info.recorder_bytes, "grid scratch bytes", info.scratch_bytes, "torch peak bytes", torch.cuda.max_memory_allocated())
    assert abs(fd - an) <= 2e-2 * abs(an)
    assert resid <= 1e-4
    grad[box] = 0
    assert float(grad.abs().max()) == 0.0


def test_error_codes_on_device(B):
    import torch
    w = wl.c3_mini(nx=24, ny=20, nz=20, d=4, n_steps=5)
    kw = w.grid_kwargs()
    kw.update(max_steps=5, record=False)
    g = B.Grid(**kw)
    f = torch.zeros((6, w.nz, w.ny, w.nx), device="cuda")
    ie = torch.as_tensor(w.inv_eps).cuda()
    with pytest.raises(B.FdtdError) as ei:
        g.forward(f, ie, None, w.sources, w.detectors, 6)            # n_steps > max_steps
    assert ei.value.code == B.FDTD_EINVAL
    bad = wl.Source(1, (0, 0, 0), (w.nx + 1, 1, 1), w.sources[0].waveform)
    with pytest.raises(B.FdtdError) as ei:
        g.forward(f, ie, None, [bad], [], 5)
    assert ei.value.code == B.FDTD_EINVAL
    g.forward(f, ie, None, w.sources, w.detectors, 5)
    with pytest.raises(B.FdtdError) as ei:
        g.backward(f, ie, None, w.sources, w.detectors, None, None, 5)   # CPML grid, nothing recorded
    assert ei.value.code == B.FDTD_ESTATE
    g.close()
    kw.update(record=True)
    g = B.Grid(**kw)
    g.forward(f, ie, None, w.sources, w.detectors, 4)
    with pytest.raises(B.FdtdError) as ei:
        g.backward(f, ie, None, w.sources, w.detectors, None, None, 5)   # different n_steps
    assert ei.value.code == B.FDTD_ESTATE
    g.close()


def test_translation_invariance_bitwise_periodic(B):
    """P12: on a periodic grid, shifting eps and the source shifts the fields bit for bit."""
    import torch
    w = wl.c1(n=16, n_steps=60)
    sx, sy, sz = 5, 3, 7
    a = run_gpu(B, w, B.FDTD_PATH_GENERIC, backward=False)["fields"]
    w2 = wl.c1(n=16, n_steps=60)
    w2.inv_eps = np.roll(w.inv_eps, (sz, sy, sx), axis=(0, 1, 2)).copy()
    s = w.sources[0]
    lo = ((s.lo[0] + sx) % 16, (s.lo[1] + sy) % 16, (s.lo[2] + sz) % 16)
    w2.sources = [wl.Source(s.component, lo, (lo[0] + 1, lo[1] + 1, lo[2] + 1), s.waveform)]
    b = run_gpu(B, w2, B.FDTD_PATH_GENERIC, backward=False)["fields"]
    assert np.array_equal(np.roll(a, (sz, sy, sx), axis=(1, 2, 3)), b)


def test_translation_invariance_bitwise_before_the_walls(B):
    """Tile-edge check for every path: in a zero-padded box, before anything reaches a wall, shifting
    the medium and the source by a vector that is not a multiple of any tile size shifts the result
    bit for bit (per-cell arithmetic does not depend on the position inside a tile)."""
    nx, ny, nz, n = 96, 80, 72, 16
    rng = np.random.default_rng(8)
    blob = (np.float32(1) / (np.float32(1) + np.float32(3) * rng.random((24, 24, 24), dtype=np.float32))).astype(np.float32)
    wav = wl.gaussian_sine(n, 6, 3, 8)

    def make(off):
        ie = np.ones((nz, ny, nx), dtype=np.float32)
        ie[off[2]:off[2] + 24, off[1]:off[1] + 24, off[0]:off[0] + 24] = blob
        c = (off[0] + 12, off[1] + 12, off[2] + 12)
        w = wl.Workload("shift", nx, ny, nz, n, ie, [wl.Source(2, c, (c[0] + 1, c[1] + 1, c[2] + 1), wav)], [])
        return w

    o1, o2 = (20, 22, 21), (20 + 29, 22 + 11, 21 + 6)
    for path in paths(B, make(o1)):
        a = run_gpu(B, make(o1), path, backward=False)["fields"]
        b = run_gpu(B, make(o2), path, backward=False)["fields"]
        assert np.max(np.abs(a)) > 0
        sh = np.roll(a, (o2[2] - o1[2], o2[1] - o1[1], o2[0] - o1[0]), axis=(1, 2, 3))
        assert np.array_equal(sh, b), path
