"""CPU-side checks of the C-ABI boundary: the CUDA library builds for sm_100a, loads without a
GPU, exports every symbol include/tslb.h declares, sizes its workspace as DESIGN.md §5 says, and
FAILS LOUDLY (no CPU fallback) when no CUDA device is present.  No compute calls here."""
import ctypes
import os
import re

import pytest

from paper_2403_15773_b200 import build, tslb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return tslb.lib()


def test_exports_match_header(lib):
    hdr = open(os.path.join(ROOT, "include", "tslb.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(tslb_[a-z_]+)\s*\(", hdr))
    assert declared == set(tslb.EXPORTS), declared ^ set(tslb.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_params_struct_matches_header():
    hdr = open(os.path.join(ROOT, "include", "tslb.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} tslb_params;", hdr, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        parts = decl.replace("*", " ").split(",")
        names.append(parts[0].split()[-1])
        names += [p.strip() for p in parts[1:]]
    assert names == [f[0] for f in tslb.Params._fields_]


def test_workspace_bytes(lib):
    def ws(**kw):
        return tslb.workspace_bytes(**kw)

    # padded layout: (nx + 16) x (ny + 4) x nz elements per field, rounded to 256 B; 2 buffers
    def field_bytes(nx, ny, nz, es):
        el = (nx + 16) * (ny + 4) * nz
        el = (el + 63) // 64 * 64
        return (el * es + 255) // 256 * 256

    assert ws(nx=512, ny=512, nz=1536, omega=1.0, two_component=True) == 22 * field_bytes(512, 512, 1536, 4)
    assert ws(nx=64, ny=64, nz=64, omega=1.0, precision=tslb.F64, two_component=True) == 22 * field_bytes(64, 64, 64, 8)
    assert ws(nx=32, ny=32, nz=32, omega=1.8, precision=tslb.F64) == 20 * field_bytes(32, 32, 32, 8)
    # generic two-component path carries 3 scratch arrays (n)
    assert ws(nx=20, ny=12, nz=10, omega=1.0, two_component=True) == 25 * field_bytes(20, 12, 10, 4)
    # TSLB_FORCING_GUO: generic path + 3 more scratch arrays (F); no tiled kernel, needs two_component
    assert ws(nx=64, ny=64, nz=64, omega=1.0, two_component=True, forcing=tslb.FORCING_GUO) == 28 * field_bytes(64, 64, 64, 4)
    assert ws(nx=64, ny=64, nz=64, omega=1.0, two_component=True, forcing=tslb.FORCING_GUO, kernel=tslb.KERNEL_TILED) == 0
    assert ws(nx=64, ny=64, nz=64, omega=1.0, forcing=tslb.FORCING_GUO) == 0
    assert ws(nx=64, ny=64, nz=64, omega=1.0, two_component=True, forcing=2) == 0
    # invalid parameters -> 0
    assert ws(nx=0, ny=4, nz=4, omega=1.0) == 0
    assert ws(nx=4, ny=4, nz=4, omega=2.0) == 0
    assert ws(nx=4, ny=4, nz=4, omega=1.0, hermite_order=4) == 0
    assert ws(nx=4, ny=4, nz=3, omega=1.0, jet=True) == 0
    assert ws(nx=4, ny=4, nz=4, omega=1.0, two_component=True, interface_width=0.0) == 0
    assert ws(nx=20, ny=12, nz=10, omega=1.0, kernel=tslb.KERNEL_TILED) == 0


def test_create_fails_loudly_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    p = tslb.make_params(32, 32, 32, 1.0)
    h = ctypes.c_void_p()
    rc = lib.tslb_create(ctypes.byref(p), ctypes.byref(h))
    assert rc == tslb.ECUDA and not h.value
    assert b"no CPU fallback" in lib.tslb_last_error(None)
    with pytest.raises(tslb.TslbError):
        tslb.Tslb(32, 32, 32, 1.0)
    # invalid parameters are reported before any device is touched
    p = tslb.make_params(32, 32, 32, 2.5)
    assert lib.tslb_create(ctypes.byref(p), ctypes.byref(h)) == tslb.EINVAL
    assert b"omega" in lib.tslb_last_error(None)


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2403_15773_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", "") or f == "inputs.py", f
