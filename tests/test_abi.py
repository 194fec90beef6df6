"""CPU-side checks of the C ABI: the library loads without a GPU, exports every symbol the header
declares, and rejects bad descriptors before touching the device (no compute calls here)."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def _lib():
    from paper_2412_12360_b200 import build
    build.build()
    from paper_2412_12360_b200 import binding
    return binding


def test_library_exports_every_declared_symbol():
    b = _lib()
    header = (ROOT / "include" / "fdtd.h").read_text()
    declared = re.findall(r"FDTD_API\s+[\w\s\*]+?\b(fdtd_\w+)\s*\(", header)
    assert len(declared) >= 9
    lib = C.CDLL(str(b.LIB_PATH))
    for name in declared:
        assert hasattr(lib, name), name
    assert set(declared) == set(b.EXPORTS)
    assert b.fdtd_version().startswith("fdtd-b200")
    assert b.fdtd_last_error() == "" or isinstance(b.fdtd_last_error(), str)


def test_struct_layouts_match_the_header():
    b = _lib()
    # 12 int32/float + 2*3 int32 + 1 + 7 = 26 four-byte fields
    assert C.sizeof(b.fdtd_grid_desc) == 4 * (14 + 6 + 1 + 7)
    assert C.sizeof(b.fdtd_source) == 4 * 7 + 4 + 16          # 7 ints, pad, 2 pointers
    assert C.sizeof(b.fdtd_detector) == 4 * 8 + 16
    assert C.sizeof(b.fdtd_grid_info) == 16 + 8 * 8


@pytest.mark.parametrize("kw,frag", [
    (dict(nx=0, ny=8, nz=8, courant=0.5), "dims"),
    (dict(nx=8, ny=8, nz=8, courant=0.6), "courant"),
    (dict(nx=8, ny=8, nz=8, courant=0.0), "courant"),
    (dict(nx=8, ny=8, nz=8, courant=0.5, periodic=True, pml_cells=2), "periodic"),
    (dict(nx=8, ny=8, nz=8, courant=0.5, pml_cells=4), "pml_cells"),
    (dict(nx=8, ny=8, nz=8, courant=0.5, pml_cells=-1), "pml_cells"),
    (dict(nx=8, ny=8, nz=8, courant=0.5, max_steps=-1), "max_steps"),
    (dict(nx=8, ny=8, nz=8, courant=0.5, pml_kappa_max=0.5), "kappa"),
    (dict(nx=8, ny=8, nz=8, courant=0.5, path=7), "path"),
])
def test_create_grid_rejects_bad_descriptors_without_a_device(kw, frag):
    b = _lib()
    with pytest.raises(b.FdtdError) as ei:
        b.fdtd_create_grid(b.make_desc(**kw))
    assert ei.value.code == b.FDTD_EINVAL
    assert frag in str(ei.value)


def test_null_arguments_are_einval():
    b = _lib()
    assert b._L.fdtd_create_grid(None, None) == b.FDTD_EINVAL
    assert b._L.fdtd_forward(None, None, None, None, None, 0, None, 0, 0, None) == b.FDTD_EINVAL
    assert b._L.fdtd_get_info(None, None) == b.FDTD_EINVAL
    assert b._L.fdtd_destroy(None) == b.FDTD_OK
    assert b._L.fdtd_halo_attach(None, 0, 0, None, None, 0) == b.FDTD_EINVAL
    assert b._L.fdtd_halo_volumes(None, None, 0, None, None) == b.FDTD_EINVAL
    assert b._L.fdtd_ipc_export(None, None, None) == b.FDTD_EINVAL
    assert b._L.fdtd_ipc_open(None, 0, None) == b.FDTD_EINVAL
    assert b._L.fdtd_ipc_close(None, 0) == b.FDTD_OK
    assert "NULL" in b.fdtd_last_error() or b.fdtd_last_error()
