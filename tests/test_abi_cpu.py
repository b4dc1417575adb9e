"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol include/tslb.h
declares, and the pure-host validation paths return the documented status codes."""
import ctypes as C
import os
import re

import pytest

from paper_2401_17074_b200 import binding as B
from paper_2401_17074_b200 import build as BLD

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    BLD.build_lib()
    return B.load_library()


def test_header_symbols_all_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "tslb.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(tslb_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(B.SYMBOLS), declared ^ set(B.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_version_and_no_torch_types_in_signatures(lib):
    assert lib.tslb_version().decode().startswith("tslb-b200")
    hdr = open(os.path.join(ROOT, "include", "tslb.h")).read()
    assert "torch" not in hdr and "at::" not in hdr


@pytest.mark.parametrize("args", [(2, 8, 8, 0.8, 0), (8, 8, 8, 0.5, 0), (8, 8, 8, float("nan"), 1), (8, 8, 8, 0.8, 7),
                                  (2048, 2048, 2048, 0.8, 0)])
def test_create_rejects_bad_arguments(lib, args):
    h = C.c_void_p()
    assert lib.tslb_create(*args, C.byref(h)) == B.TSLB_EINVAL
    assert not h.value
    assert len(lib.tslb_last_error(None)) > 0


def test_host_only_state_machine(lib):
    s = B.TSLB(8, 6, 5, 0.8, "f64", bind=False)
    assert s.workspace_bytes() >= 2 * 10 * 8 * 6 * 5 * 8
    assert s.step_count == -1 and s.launch_count == 0
    with pytest.raises(B.TSLBError) as e:
        s.step(1, stream=0)
    assert e.value.code == B.TSLB_ESTATE
    # boundary validation is host-only
    with pytest.raises(B.TSLBError) as e:
        s._chk(s._lib.tslb_set_boundary(s._h, 9, B.BC_BOUNCE_BACK, None), "tslb_set_boundary")
    assert e.value.code == B.TSLB_EINVAL
    with pytest.raises(B.TSLBError):
        s._chk(s._lib.tslb_set_boundary(s._h, 0, 17, None), "tslb_set_boundary")
    with pytest.raises(B.TSLBError):
        s._chk(s._lib.tslb_set_boundary(s._h, 0, B.BC_VELOCITY_INLET, None), "tslb_set_boundary")
    with pytest.raises(B.TSLBError):
        s.set_body_force((float("inf"), 0, 0))
    s.set_body_force((1e-6, 0, 0))
    s.set_boundary(B.FACE_YLO, B.BC_BOUNCE_BACK)
    # slab ghost planes exist on the z faces only; face export / import need a state
    with pytest.raises(B.TSLBError) as e:
        s.set_boundary(B.FACE_XLO, B.BC_EXCHANGE)
    assert e.value.code == B.TSLB_EINVAL
    s.set_boundary(B.FACE_ZHI, B.BC_EXCHANGE)
    assert s.face_bytes() == 10 * 6 * 8 * 8
    assert s._lib.tslb_export_face(s._h, B.FACE_ZHI, C.c_void_p(0x1000), None) == B.TSLB_ESTATE
    assert s._lib.tslb_import_face(s._h, B.FACE_ZHI, C.c_void_p(0x1000), None) == B.TSLB_ESTATE
    with pytest.raises(B.TSLBError):
        s.set_kernel(5)
    # misaligned / undersized workspace
    assert s._lib.tslb_bind_workspace(s._h, C.c_void_p(0), 1 << 30) == B.TSLB_EINVAL
    assert s._lib.tslb_bind_workspace(s._h, C.c_void_p(0x1001), 1 << 30) == B.TSLB_EINVAL
    assert s._lib.tslb_bind_workspace(s._h, C.c_void_p(0x1000), 16) == B.TSLB_EINVAL
    s.close()


def test_missing_library_fails_loudly(tmp_path):
    with pytest.raises(FileNotFoundError):
        B.load_library(str(tmp_path / "nope.so"))


def test_product_never_imports_oracle():
    """The CUDA path and its binding must not reach into oracle/ (no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2401_17074_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "tslb_oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "tslb_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "csrc" not in osrc.replace("paper_2401_17074_b200/csrc", "") and "import paper_2401_17074_b200" not in osrc
