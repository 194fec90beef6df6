"""Domain decomposition along z (include/fdtd.h "Domain decomposition") on ONE
device: the slabs of a grid advanced in lock step with one halo exchange per step must reproduce the undivided grid
BIT FOR BIT on the planes they own -- fields, phasors, cotangent of state 0 -- on both kernel paths (the per-cell
arithmetic does not depend on where a cell sits in its grid).  The gradient agrees to the rounding of the time
reversal: next to a cut a slab's inverse step reads the RECORDED interface value (the forward run's, exact) where
the undivided grid reads its own reconstructed neighbour (equal up to the reconstruction's fp32 rounding), so
dL/d inv_eps differs by a few 1e-8 of its maximum (bound asserted: 1e-6; the oracle tolerance is 1e-3).  The
undivided grid itself is checked against the oracle in test_gpu_parity.py."""
import numpy as np
import pytest

from paper_2412_12360_b200 import sharding, workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2412_12360_b200 import binding
    return binding


def _single(B, w, path, n, dLf_fn=None):
    import torch
    kw = w.grid_kwargs()
    kw.update(max_steps=n, record=1, path=path)
    g = B.Grid(**kw)
    f = torch.zeros((6, w.nz, w.ny, w.nx), device="cuda")
    ie = torch.as_tensor(w.inv_eps).cuda()
    im = None if w.meta.get("inv_mu") is None else torch.as_tensor(w.meta["inv_mu"]).cuda()
    ph = g.forward(f, ie, im, w.sources, w.detectors, n)
    torch.cuda.synchronize()
    fields = f.cpu().numpy()
    dLp = [2.0 * P for P in ph]
    dLf = torch.zeros_like(f)
    dLf[:3] = 0.5 * f[:3]
    dLf[3:] = -0.25 * f[3:]
    grad, lam0 = g.backward(f, ie, im, w.sources, w.detectors, dLp, dLf, n, want_dL_dfields0=True)
    torch.cuda.synchronize()
    res = dict(fields=fields, phasors=[p.cpu().numpy() for p in ph], grad=grad.cpu().numpy(), lam0=lam0.cpu().numpy(),
               dLp=dLp, dLf=dLf, path=g.info().path)
    g.close()
    return res


def _slabs(B, w, path, n, cuts, ref, peer=False):
    import torch
    slabs = sharding.z_slabs(w.nz, len(cuts) + 1, w.pml_cells, cuts)
    runners = [sharding.SlabRunner(B, w, s, n, record=1, path=path) for s in slabs]
    sharding.run_slabs_lockstep(runners, n, "forward", peer=peer)
    torch.cuda.synchronize()
    fields = np.zeros_like(ref["fields"])
    phasors = [np.zeros_like(p) for p in ref["phasors"]]
    for r in runners:
        own = r.slab.owned_local()
        fields[:, r.slab.k_lo:r.slab.k_hi] = r.fields[:, own].cpu().numpy()
        for (idx, d, sl), P in zip(r.det_fwd, r.phasors):
            phasors[idx][:, :, sl] = P.cpu().numpy()
    for r in runners:
        r.set_cotangents(ref["dLp"], ref["dLf"])
    sharding.run_slabs_lockstep(runners, n, "backward", peer=peer)
    torch.cuda.synchronize()
    grad, lam0 = np.zeros_like(ref["grad"]), np.zeros_like(ref["lam0"])
    for r in runners:
        own = r.slab.owned_local()
        grad[r.slab.k_lo:r.slab.k_hi] = r.grad[own].cpu().numpy()
        lam0[:, r.slab.k_lo:r.slab.k_hi] = r.lam0[:, own].cpu().numpy()
    paths = {r.grid.info().path for r in runners}
    if peer == "flags":                                   # no wait of the device-side ordering gave up
        assert all(B.fdtd_halo_sync_error(r.grid.h) == 0 for r in runners)
    for r in runners:
        r.close()
    return dict(fields=fields, phasors=phasors, grad=grad, lam0=lam0, paths=paths)


@pytest.mark.parametrize("path_name", ["generic", "fused"])
@pytest.mark.parametrize("cuts", [(21,), (13, 33), (9, 20, 35)])
def test_z_slabs_in_lock_step_reproduce_the_single_grid_bitwise(B, path_name, cuts):
    """C3 miniature with kappa / alpha CPML, inv_mu, an extra H source; cuts through the design box, next to the
    detector plane (k = 33) and (9, 35: d = 8) next to a z CPML slab; odd step count (the fused
    ping-pong ends in its second volume)."""
    path = B.FDTD_PATH_GENERIC if path_name == "generic" else B.FDTD_PATH_FUSED
    n = 37
    w = wl.c3_mini(n_steps=n, kappa_max=3.0, alpha_max=0.05)
    rng = np.random.default_rng(3)
    w.meta["inv_mu"] = (1.0 / (1.0 + 0.5 * rng.random((w.nz, w.ny, w.nx), dtype=np.float32))).astype(np.float32)
    w.sources.append(wl.Source(3, (20, 12, 22), (60, 40, 23), (0.3 * wl.gaussian_sine(n, 12, 5, 11)).astype(np.float32)))
    w.detectors.append(wl.Detector((1 << 1) | (1 << 5), (10, 10, 18), (70, 40, 24), [wl.omega_ppw(12)]))   # a box across the cuts
    ref = _single(B, w, path, n)
    assert ref["path"] == path
    got = _slabs(B, w, path, n, list(cuts), ref)
    assert got["paths"] == {path}
    assert np.max(np.abs(ref["grad"])) > 0 and np.max(np.abs(ref["lam0"])) > 0
    assert np.array_equal(got["fields"], ref["fields"])
    for P, Pr in zip(got["phasors"], ref["phasors"]):
        assert np.max(np.abs(Pr)) > 0 and np.array_equal(P, Pr)
    assert np.array_equal(got["lam0"], ref["lam0"])
    err = float(np.max(np.abs(got["grad"].astype(np.float64) - ref["grad"])) / np.max(np.abs(ref["grad"])))
    print(f"z slabs {cuts} {path_name}: fields, phasors, lam0 bit-identical; gradient differs by {err:.1e} of its maximum")
    assert err <= 1e-6


@pytest.mark.parametrize("n", [37, 24])
@pytest.mark.parametrize("cuts", [(21,), (9, 20, 35)])
def test_peer_stores_replace_the_halo_exchange_bitwise(B, cuts, n):
    """include/fdtd.h "Peer stores": with the neighbours attached (fdtd_halo_volumes / fdtd_halo_attach) the fused step
    kernels write their boundary planes into the neighbours' ghost planes themselves and there is no fdtd_halo_export /
    _import at all; the slabs still reproduce the undivided grid bit for bit (fields, phasors, cotangent of state 0) in
    both directions, for an odd and an even step count (the seed of the reverse sweep lands in either volume of the
    ping-pong).  Same workload as the exchange test above."""
    path = B.FDTD_PATH_FUSED
    w = wl.c3_mini(n_steps=n, kappa_max=3.0, alpha_max=0.05)
    rng = np.random.default_rng(3)
    w.meta["inv_mu"] = (1.0 / (1.0 + 0.5 * rng.random((w.nz, w.ny, w.nx), dtype=np.float32))).astype(np.float32)
    w.sources.append(wl.Source(3, (20, 12, 22), (60, 40, 23), (0.3 * wl.gaussian_sine(n, 12, 5, 11)).astype(np.float32)))
    w.detectors.append(wl.Detector((1 << 1) | (1 << 5), (10, 10, 18), (70, 40, 24), [wl.omega_ppw(12)]))
    ref = _single(B, w, path, n)
    got = _slabs(B, w, path, n, list(cuts), ref, peer=True)
    assert got["paths"] == {path}
    assert np.max(np.abs(ref["grad"])) > 0 and np.max(np.abs(ref["lam0"])) > 0
    assert np.array_equal(got["fields"], ref["fields"])
    for P, Pr in zip(got["phasors"], ref["phasors"]):
        assert np.max(np.abs(Pr)) > 0 and np.array_equal(P, Pr)
    assert np.array_equal(got["lam0"], ref["lam0"])
    err = float(np.max(np.abs(got["grad"].astype(np.float64) - ref["grad"])) / np.max(np.abs(ref["grad"])))
    print(f"peer stores, z slabs {cuts}, {n} steps: fields, phasors, lam0 bit-identical; gradient differs by {err:.1e} of its maximum")
    assert err <= 1e-6


def test_device_side_ordering_of_the_slabs(B, monkeypatch):
    """include/fdtd.h "Device-side ordering": the wait / signal kernels beside every step kernel (peer = "flags").  On one
    device the slabs are issued step by step in slab order on one stream, so every wait finds its flag set by a signal
    that precedes it in the stream; the run is bit-identical to the undivided grid, no wait times out, and a slab that
    runs ahead of its neighbour gives up after the (here: 200 ms) limit and reports the state that never came."""
    import torch
    monkeypatch.setenv("FDTD_HALO_TIMEOUT_MS", "200")
    path = B.FDTD_PATH_FUSED
    n = 11
    w = wl.c3_mini(n_steps=n, kappa_max=3.0, alpha_max=0.05)
    ref = _single(B, w, path, n)
    got = _slabs(B, w, path, n, [13, 30], ref, peer="flags")
    assert np.array_equal(got["fields"], ref["fields"]) and np.array_equal(got["lam0"], ref["lam0"])
    for P, Pr in zip(got["phasors"], ref["phasors"]):
        assert np.array_equal(P, Pr)
    # flags and the bounded wait, on two fresh slabs
    slabs = sharding.z_slabs(w.nz, 2, w.pml_cells, [21])
    r0, r1 = (sharding.SlabRunner(B, w, s, n, record=1, path=path) for s in slabs)
    sharding.attach_neighbours_local([r0, r1], 0, flags=True)
    for k in range(3):
        r0.forward_steps(k, k + 1)
        r1.forward_steps(k, k + 1)
    torch.cuda.synchronize()
    assert B.fdtd_halo_sync_error(r0.grid.h) == 0 and B.fdtd_halo_sync_error(r1.grid.h) == 0
    r0.forward_steps(3, 4)                              # state 4 on slab 0 only ...
    r0.forward_steps(4, 5)                              # ... its next step waits for slab 1's state 4, which never comes
    torch.cuda.synchronize()
    assert B.fdtd_halo_sync_error(r0.grid.h) == 5       # 1 + the state index waited for
    assert B.fdtd_halo_sync_error(r0.grid.h) == 0       # read and cleared
    for r in (r0, r1):
        r.close()


def test_c3_full_size_slabs_with_peer_stores_bitwise(B):
    """C3 at its full size (200^3, d = 12: the 200 x 7 tiles and the calibrated lock-step partition of the bench, per slab) cut
    at z = 87 and z = 140 -- through the design region -- with the halo planes stored by the step kernels: fields, phasors and
    the cotangent of state 0 bit-identical to the undivided grid after 25 steps and 25 reverse steps."""
    n = 25
    w = wl.c3(n_steps=n)
    ref = _single(B, w, B.FDTD_PATH_FUSED, n)
    got = _slabs(B, w, B.FDTD_PATH_FUSED, n, [87, 140], ref, peer=True)
    assert got["paths"] == {B.FDTD_PATH_FUSED}
    assert np.max(np.abs(ref["fields"])) > 0 and np.max(np.abs(ref["lam0"])) > 0
    assert np.array_equal(got["fields"], ref["fields"])
    for P, Pr in zip(got["phasors"], ref["phasors"]):
        assert np.array_equal(P, Pr)
    assert np.array_equal(got["lam0"], ref["lam0"])
    gmax = float(np.max(np.abs(ref["grad"])))
    if gmax > 0:
        assert float(np.max(np.abs(got["grad"].astype(np.float64) - ref["grad"]))) <= 1e-6 * gmax


def _ipc_worker(rank, world, port, out):
    """One rank = one process with its own CUDA context on cuda:0: its slab, the neighbour's volumes opened from CUDA IPC
    handles, tokens over gloo with a stream synchronisation before each (no kernel waits for another process's kernel)."""
    import os
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2412_12360_b200 import binding as B
        torch.cuda.set_device(0)
        n = 9
        w = wl.c3_mini(n_steps=n, kappa_max=3.0, alpha_max=0.05)
        ref = _single(B, w, B.FDTD_PATH_FUSED, n)
        slab = sharding.z_slabs(w.nz, world, w.pml_cells, [21])[rank]
        r = sharding.SlabRunner(B, w, slab, n, record=1, path=B.FDTD_PATH_FUSED)
        sharding.run_slab_distributed(r, n, "forward", peer=True, host_sync=True)
        torch.cuda.synchronize()
        own = slab.owned_local()
        ok_f = bool(np.array_equal(r.fields[:, own].cpu().numpy(), ref["fields"][:, slab.k_lo:slab.k_hi]))
        ok_p = all(np.array_equal(P.cpu().numpy(), ref["phasors"][idx][:, :, sl]) for (idx, d, sl), P in zip(r.det_fwd, r.phasors))
        r.set_cotangents(ref["dLp"], ref["dLf"])
        sharding.run_slab_distributed(r, n, "backward", peer=True, host_sync=True)
        torch.cuda.synchronize()
        ok_l = bool(np.array_equal(r.lam0[:, own].cpu().numpy(), ref["lam0"][:, slab.k_lo:slab.k_hi]))
        eg = float(np.max(np.abs(r.grad[own].cpu().numpy().astype(np.float64) - ref["grad"][slab.k_lo:slab.k_hi])) / np.max(np.abs(ref["grad"])))
        out[rank] = (ok_f, ok_p, ok_l, eg, float(np.max(np.abs(ref["lam0"]))))
        r.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(600)
def test_peer_stores_across_two_processes_through_cuda_ipc(B):
    """The cross-process form of the peer stores (sharding.PeerLinks: fdtd_ipc_export / fdtd_ipc_open, then
    fdtd_halo_attach) with two processes on the one device there is: each rank's kernels store into memory the OTHER
    process allocated.  Bit-identical to the undivided grid again."""
    import os
    import torch.multiprocessing as mp
    world, port = 2, 35500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_ipc_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for rank in range(world):
        ok_f, ok_p, ok_l, eg, lmax = res[rank]
        assert lmax > 0 and ok_f and ok_p and ok_l, (rank, res[rank])
        assert eg <= 1e-6


def test_peer_store_argument_checks(B):
    import torch
    n = 4
    w = wl.c3_mini(n_steps=n)
    slabs = sharding.z_slabs(w.nz, 2, w.pml_cells, [21])
    r0, r1 = (sharding.SlabRunner(B, w, s, n, record=1, path=B.FDTD_PATH_FUSED) for s in slabs)
    v1 = r1.volumes(0)
    assert v1[0] == r1.fields.data_ptr() and v1[1] != 0 and v1[1] != v1[0]
    with pytest.raises(B.FdtdError) as e:          # slab 0 has no cut below
        r0.attach(0, 0, v1, r1.slab.nz)
    assert e.value.code == B.FDTD_EINVAL
    with pytest.raises(B.FdtdError) as e:          # one volume only
        B.fdtd_halo_attach(r0.grid.h, 0, 1, v1[0], None, r1.slab.nz)
    assert e.value.code == B.FDTD_EINVAL
    r0.attach(0, 1, v1, r1.slab.nz)
    with pytest.raises(B.FdtdError) as e:          # attached: one step per call
        r0.forward_steps(0, 2)
    assert e.value.code == B.FDTD_EINVAL
    r0.detach(0)
    r0.forward_steps(0, 2)                          # detached: any range again
    torch.cuda.synchronize()
    g = sharding.SlabRunner(B, w, slabs[0], n, record=1, path=B.FDTD_PATH_GENERIC)
    with pytest.raises(B.FdtdError) as e:          # the generic kernels have no peer stores
        g.volumes(0)
    assert e.value.code == B.FDTD_ESTATE
    for r in (r0, r1, g):
        r.close()


def test_subgrid_descriptor_checks(B):
    w = wl.c3_mini(n_steps=4)
    kw = w.grid_kwargs()
    for bad in (dict(nz=10, z_global=44, z_offset=0, z_ghost_lo=1, z_ghost_hi=1),      # ghost below at the global bottom
                dict(nz=10, z_global=44, z_offset=10, z_ghost_lo=1, z_ghost_hi=0),      # missing ghost above
                dict(nz=6, z_global=44, z_offset=0, z_ghost_lo=0, z_ghost_hi=1),        # owns no interior plane (d = 8)
                dict(nz=10, z_global=0, z_offset=3)):
        with pytest.raises(B.FdtdError) as e:
            B.Grid(**{**kw, **bad, "max_steps": 4})
        assert e.value.code == B.FDTD_EINVAL


@pytest.mark.parametrize("path_name", ["generic", "fused"])
def test_a_run_in_pieces_is_the_same_run(B, path_name):
    """fdtd_forward_range / fdtd_backward_range on an ordinary grid: a run cut into pieces of odd and even lengths (the
    fused ping-pong changes volume with every step) gives bit for bit what fdtd_forward / fdtd_backward give; a piece that
    does not continue the previous one is ESTATE."""
    import torch
    path = B.FDTD_PATH_GENERIC if path_name == "generic" else B.FDTD_PATH_FUSED
    n = 23
    w = wl.c3_mini(n_steps=n, kappa_max=3.0, alpha_max=0.05)
    ref = _single(B, w, path, n)
    slab = sharding.ZSlab(0, 1, w.nz, 0, w.nz)                  # the whole grid as one "slab": no ghosts, no exchange
    r = sharding.SlabRunner(B, w, slab, n, record=1, path=path)
    r.grid.close()
    kw = w.grid_kwargs()
    kw.update(max_steps=n, record=1, path=path)
    r.grid = B.Grid(**kw)                                       # an ordinary grid (z_global = 0) behind the same runner
    r.sarr, r.ns, r._k1 = r.grid.marshal_sources(r.sources)
    r.darr, r.nd, r._k2 = r.grid.marshal_detectors([d for _, d, _ in r.det_fwd], r.phasors)
    r.darr_b, r.nd_b, r._k3 = r.grid.marshal_detectors([d for _, d, _ in r.det_bwd], None)
    for a, b in [(0, 5), (5, 6), (6, 20), (20, 23)]:
        r.forward_steps(a, b)
    with pytest.raises(B.FdtdError) as e:
        r.forward_steps(7, 9)
    assert e.value.code == B.FDTD_ESTATE
    torch.cuda.synchronize()
    assert np.array_equal(r.fields.cpu().numpy(), ref["fields"])
    for P, Pr in zip(r.phasors, ref["phasors"]):
        assert np.array_equal(P.cpu().numpy(), Pr)
    # a new run may start at any time (n_begin = 0: psi reset, state taken from `fields`)
    for P in r.phasors:
        P.zero_()
    r.fields.zero_()
    for a, b in [(0, 1), (1, 8), (8, 23)]:
        r.forward_steps(a, b)
    torch.cuda.synchronize()
    for P, Pr in zip(r.phasors, ref["phasors"]):
        assert np.array_equal(P.cpu().numpy(), Pr)
    r.set_cotangents(ref["dLp"], ref["dLf"])
    for a, b in [(23, 22), (22, 15), (15, 14), (14, 0)]:
        r.backward_steps(a, b)
    torch.cuda.synchronize()
    assert np.array_equal(r.lam0.cpu().numpy(), ref["lam0"])
    assert np.array_equal(r.grad.cpu().numpy(), ref["grad"])
    r.close()
