"""fdtd_flux_static (include/fdtd.h): the Poynting flux of fdtd_flux for callers that cannot allocate device memory -- no
grid, no cudaMalloc, reduction scratch in a file-scope `static __device__` array of the library (planes of at most
FDTD_FLUX_STATIC_MAX_CELLS cells).  Checked against the existing path (fdtd_flux with a grid's scratch; itself checked
against the oracle in test_gpu_n2.py) within that test's tolerance, on calls in a row that share the array: a small plane,
a plane of several blocks with a ragged tail, the small plane again (stale partials of the larger call in the array).
Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import ctypes as C

import numpy as np
import pytest

from paper_2412_12360_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_PHASOR = 1e-4          # the flux tolerance of tests/test_gpu_n2.py::test_flux_and_its_vjp


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2412_12360_b200 import binding
    return binding


def relerr(x, ref):
    x, ref = np.asarray(x, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    return float(np.max(np.abs(x - ref)) / max(np.max(np.abs(ref)), 1e-300))


def _plane_detector(shape_xyz, axis, p, interpolate):
    nx, ny, nz = shape_xyz
    lo, hi = [0, 0, 0], [nx, ny, nz]
    lo[axis], hi[axis] = p - (1 if interpolate else 0), p + 1
    b, c = (axis + 1) % 3, (axis + 2) % 3
    mask = (1 << b) | (1 << c) | (1 << (3 + b)) | (1 << (3 + c)) | (1 << axis)      # one extra component: slots are not 0..3
    return wl.Detector(mask, tuple(lo), tuple(hi), [wl.omega_ppw(12), wl.omega_ppw(17), wl.omega_ppw(9)])


def test_flux_static_matches_fdtd_flux_on_calls_in_a_row(B):
    import torch
    nx, ny, nz = 200, 181, 6                       # z planes of 36200 cells: 17 full blocks of 2048 and a tail
    g = B.Grid(nx=nx, ny=ny, nz=nz, courant=0.5, max_steps=1, path=B.FDTD_PATH_GENERIC)
    st = g.stream()
    gen = torch.Generator(device="cuda").manual_seed(11)
    cases = [("small x plane", 0, 100, False), ("z plane, several blocks", 2, 3, True), ("small x plane again", 0, 100, False),
             ("y plane, co-located", 1, 77, True)]
    got, want, keep = [], [], []
    for name, axis, p, interp in cases:            # no synchronisation between the calls: they follow each other on one stream
        det = _plane_detector((nx, ny, nz), axis, p, interp)
        ph = torch.rand(det.phasor_shape, device="cuda", generator=gen) + 0.25
        want.append(g.flux(det, ph, axis, interp))                     # existing path: the grid's cudaMalloc'ed scratch
        darr, nd, k = g.marshal_detectors([det], None)
        out = torch.full((len(det.omega),), float("nan"), device="cuda")
        B.fdtd_flux_static(darr, ph, axis, interp, out, st)
        got.append(out)
        keep.append((darr, k, ph))
    torch.cuda.synchronize()
    g.close()
    for (name, *_), a, b in zip(cases, got, want):
        a, b = a.cpu().numpy(), b.cpu().numpy()
        assert np.all(np.isfinite(a)) and np.max(np.abs(b)) > 0, name
        assert relerr(a, b) <= TOL_PHASOR, (name, a, b)
    # the same inputs give the same bits on every call (fixed summation order; nothing left over in the array matters)
    darr, k, ph = keep[1]
    again = torch.full_like(got[1], float("nan"))
    B.fdtd_flux_static(darr, ph, 2, True, again, st)
    torch.cuda.synchronize()
    assert np.array_equal(again.cpu().numpy(), got[1].cpu().numpy())


def test_flux_static_limits_and_errors(B):
    import torch
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    dummy = torch.zeros(64, device="cuda")
    out = torch.zeros(4, device="cuda")

    def desc(lo, hi, mask, n_freq=1):
        d = (B.fdtd_detector * 1)()
        om = (C.c_float * max(n_freq, 1))(*([0.5] * max(n_freq, 1)))
        d[0].component_mask, d[0].n_freq = mask, n_freq
        d[0].lo[:], d[0].hi[:] = lo, hi
        d[0].omega = C.cast(om, C.POINTER(C.c_float))
        return d, om

    tang_z = 0b011011                                                   # Ex, Ey, Hx, Hy
    # one cell more than the static scratch covers: rejected before anything is launched (the phasor is never read)
    d, om = desc([0, 0, 5], [2048, 2049, 6], tang_z)
    assert 2048 * 2049 > B.FDTD_FLUX_STATIC_MAX_CELLS
    with pytest.raises(B.FdtdError) as e:
        B.fdtd_flux_static(d, dummy, 2, False, out, st)
    assert e.value.code == B.FDTD_EINVAL and "maximum" in str(e.value) and str(B.FDTD_FLUX_STATIC_MAX_CELLS) in str(e.value)
    for lo, hi, mask, axis, interp in (([0, 0, 5], [8, 8, 7], tang_z, 2, False),        # two planes without interpolation
                                       ([0, 0, 5], [8, 8, 6], tang_z, 2, True),         # one plane with it
                                       ([0, 0, 5], [8, 8, 6], 0b001011, 2, False),      # Hy missing
                                       ([0, 0, 5], [8, 8, 6], tang_z, 3, False),        # axis
                                       ([0, 4, 5], [8, 4, 6], tang_z, 2, False)):       # empty box
        d, om = desc(lo, hi, mask)
        with pytest.raises(B.FdtdError) as e:
            B.fdtd_flux_static(d, dummy, axis, interp, out, st)
        assert e.value.code == B.FDTD_EINVAL
    d, om = desc([0, 0, 5], [8, 8, 6], tang_z)
    with pytest.raises(B.FdtdError) as e:
        B.fdtd_flux_static(d, None, 2, False, out, st)
    assert e.value.code == B.FDTD_EINVAL
    # the largest plane the array covers runs (2048 x 2048 cells, 4 components: 134 MB of phasors)
    d, om = desc([0, 0, 5], [2048, 2048, 6], tang_z)
    ph = torch.ones((1, 4, 1, 2048, 2048, 2), device="cuda")
    res = torch.full((1,), float("nan"), device="cuda")
    B.fdtd_flux_static(d, ph, 2, False, res, st)
    torch.cuda.synchronize()
    assert float(res[0]) == 0.0                                         # E = H = 1 + i everywhere: the two pairs cancel in every cell
    ph[0, 0] *= 3.0                                                     # E_x = 3 + 3i: 1/2 Re(E_x conj H_y - E_y conj H_x) = 1/2 (6 - 2) = 2 per cell
    B.fdtd_flux_static(d, ph, 2, False, res, st)
    torch.cuda.synchronize()
    assert float(res[0]) == 2.0 * 2048 * 2048
