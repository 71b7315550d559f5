"""CPU-only checks of the boundary: the C-ABI library builds, loads, exports every symbol that
include/inpc_raster.h declares, and its host-side logic (argument validation, workspace sizing,
error strings) behaves as the header says.  No compute call is made here (there is no GPU)."""
import ctypes as C
import os
import re

import pytest

import __graft_entry__ as entry
from paper_2403_16862_b200 import raster

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    entry.build()
    return raster.load()


def _declared_symbols():
    names = set()
    inc = os.path.join(ROOT, "include")
    for fn in os.listdir(inc):
        if fn.endswith(".h"):
            src = open(os.path.join(inc, fn)).read()
            src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
            names |= set(re.findall(r"\b(inpc_(?:raster|sample)_\w+)\s*\(", src))
    return names


def test_every_declared_symbol_is_exported(lib):
    declared = _declared_symbols()
    assert {"inpc_raster_forward", "inpc_raster_backward"} <= declared
    for name in declared:
        assert hasattr(lib, name), f"{name} is declared in include/ but not exported"
    assert declared == set(raster.EXPORTS), "binding and header disagree on the entry points"


def test_camera_struct_layout_matches_header(lib):
    # 4 + 9 + 3 + 2 floats + 2 int32 = 80 bytes, no padding
    assert C.sizeof(raster.InpcCamera) == 80
    assert C.sizeof(raster.InpcStats) == 56       # 7 x uint64


def test_workspace_bytes_host_logic(lib):
    ws = raster.inpc_raster_workspace_bytes
    assert ws(0, 4, 64, 64) > 0
    a, b = ws(1 << 20, 4, 1297, 840), ws(1 << 23, 4, 1297, 840)
    assert 0 < a < b
    assert ws(1 << 20, 8, 1297, 840) > a                       # wider records
    assert ws(1 << 20, 4, 1297, 840, raster.SAVE_FOR_BACKWARD | raster.SAVE_SORTED) > a
    # 8M training config: the workspace stays well under 180 GB of HBM (it is a few GB)
    assert b < 8 << 30
    for bad in [(-1, 4, 64, 64), (10, 3, 64, 64), (10, 4, 0, 64), (10, 4, 64, -1), (1 << 30, 4, 64, 64), (10, 4, 5000, 64)]:
        assert ws(*bad) == 0


def test_argument_validation_returns_codes_not_crashes(lib):
    cam = raster.InpcCamera()
    cam.fx = cam.fy = 64.0; cam.cx = cam.cy = 32.0
    cam.near_z, cam.far_z, cam.width, cam.height = 0.01, 100.0, 64, 64
    for i, v in enumerate([1, 0, 0, 0, 1, 0, 0, 0, 1]):
        cam.R[i] = float(v)
    fake = C.c_void_p(0x1000)                                   # never dereferenced: validation fails first
    f = lib.inpc_raster_forward
    assert f(fake, fake, fake, 16, 4, None, fake, fake, fake, 1 << 20, 0, None) == -1          # NULL camera
    assert f(fake, fake, fake, -5, 4, C.byref(cam), fake, fake, fake, 1 << 20, 0, None) == -1   # N < 0
    assert f(fake, fake, fake, 16, 5, C.byref(cam), fake, fake, fake, 1 << 20, 0, None) == -5   # D unsupported
    assert f(fake, fake, fake, 16, 4, C.byref(cam), None, fake, fake, 1 << 20, 0, None) == -1   # NULL output
    assert f(C.c_void_p(0x1004), fake, fake, 16, 4, C.byref(cam), fake, fake, fake, 1 << 20, 0, None) == -1  # misaligned
    assert f(fake, fake, fake, 16, 4, C.byref(cam), fake, fake, fake, 64, 0, None) == -2        # workspace too small
    cam.near_z = 200.0
    assert f(fake, fake, fake, 16, 4, C.byref(cam), fake, fake, fake, 1 << 20, 0, None) == -1   # near >= far
    cam.near_z = 0.01
    b = lib.inpc_raster_backward
    assert b(fake, fake, fake, 16, 4, C.byref(cam), fake, None, fake, fake, fake, fake, 64, None) == -2     # workspace too small
    assert b(fake, fake, fake, 16, 4, C.byref(cam), None, None, fake, fake, fake, fake, 1 << 20, None) == -1  # NULL grad_out
    assert b(fake, fake, fake, 16, 4, C.byref(cam), fake, None, fake, fake, fake, C.c_void_p(0x1010), 1 << 20, None) == -1  # workspace not 256-aligned
    assert lib.inpc_raster_get_counts(None, 64, 64, fake, None) == -1
    assert lib.inpc_raster_get_blended_counts(fake, 0, 64, fake, None) == -1
    st = raster.InpcStats()
    assert lib.inpc_raster_get_stats(None, C.byref(st), None) == -1
    assert lib.inpc_raster_get_status(None, None) == -1
    import torch
    if not torch.cuda.is_available():
        # no device: every compute / read-back call reports INPC_ERR_CUDA (there is no CPU fallback)
        assert f(fake, fake, fake, 16, 4, C.byref(cam), fake, fake, fake, 1 << 20, 0, None) == -3
        assert lib.inpc_raster_get_status(fake, None) == -3
        assert lib.inpc_raster_last_cuda_error().decode() != ""


def test_strerror_and_launch_counter(lib):
    msgs = {lib.inpc_raster_strerror(c).decode() for c in (0, -1, -2, -3, -4, -5)}
    assert len(msgs) == 6 and "ok" in msgs
    assert lib.inpc_raster_strerror(-99).decode() == "unknown status"
    assert raster.inpc_raster_launch_count() >= 0
    assert isinstance(raster.inpc_raster_launched_kernels(), set)


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(raster, "_lib", None)
    monkeypatch.setattr(raster, "LIB_PATH", "/nonexistent/libinpc_raster.so")
    with pytest.raises(ImportError):
        raster.load()


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2403_16862_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), fn
                assert "liboracle" not in src and "oracle.cpp" not in src, fn


def test_static_scratch_sampler_limit_is_checked_on_the_host(lib):
    """inpc_sample_view_static (the sampler for callers that cannot allocate device memory) refuses more leaves than its
    built-in array holds before it touches the device, with a status and a message of its own."""
    cam = raster.InpcCamera()
    cam.fx = cam.fy = 64.0; cam.cx = cam.cy = 32.0
    cam.near_z, cam.far_z, cam.width, cam.height = 0.01, 100.0, 64, 64
    fake = C.c_void_p(0x1000)
    mx = lib.inpc_sample_static_max_leaves()
    assert mx == 1 << 18
    assert lib.inpc_sample_workspace_bytes(mx) == 4458240          # the size the header states for the array
    rc = lib.inpc_sample_view_static(fake, fake, fake, mx + 1, 8.0, C.byref(cam), 1, 16, fake, fake, None)
    assert rc == -6 and b"inpc_sample_static_max_leaves" in lib.inpc_raster_strerror(rc)


def test_backward_accepts_null_gradient_outputs_on_the_host(lib):
    """SURVEY.md:321-322: grad_feat / grad_opacity / grad_uv "or NULL".  With all three NULL the host-side validation
    still passes (the next failure is the workspace size, checked after the pointers)."""
    cam = raster.InpcCamera()
    cam.fx = cam.fy = 64.0; cam.cx = cam.cy = 32.0
    cam.near_z, cam.far_z, cam.width, cam.height = 0.01, 100.0, 64, 64
    fake = C.c_void_p(0x1000)
    assert lib.inpc_raster_backward(fake, fake, fake, 16, 4, C.byref(cam), fake, None, None, None, None, fake, 64, None) == -2
    assert lib.inpc_raster_backward(fake, fake, fake, 16, 4, C.byref(cam), None, None, None, None, None, fake, 64, None) == -1


def test_staging_kernels_use_bulk_copies_and_nothing_spills(lib):
    """The built library's SASS, per kernel (python -m paper_2403_16862_b200.sass_summary, the table of
    profiles/r03_sass.md): the tile kernels stage with cp.async.bulk on an mbarrier (UBLKCP + SYNCS), the saving forward
    also stores the order lists with one, and no hot kernel spills registers to local memory."""
    import contextlib
    import io
    from paper_2403_16862_b200 import sass_summary
    buf = io.StringIO()
    with contextlib.redirect_stdout(buf):
        assert sass_summary.main() == 0
    rows = {}
    for line in buf.getvalue().splitlines():
        if line.startswith("| `"):
            c = [x.strip() for x in line.strip("|").split("|")]
            rows[c[0].strip("`")] = c
    head = [x.strip() for x in next(l for l in buf.getvalue().splitlines() if l.startswith("| kernel")).strip("|").split("|")]
    col = {n: i for i, n in enumerate(head)}
    for k in ("k_blend<4, 1, 0>", "k_blend<4, 0, 0>", "k_blend<8, 0, 0>", "k_back<4>", "k_back<8>"):
        assert int(rows[k][col["UBLKCP"]]) >= 3 and int(rows[k][col["SYNCS"]]) >= 3, k
    assert int(rows["k_blend<4, 1, 0>"][col["UBLKCP"]]) > int(rows["k_blend<4, 0, 0>"][col["UBLKCP"]])   # + the bulk store
    for k in ("k_blend<4, 1, 0>", "k_blend<4, 0, 0>", "k_back<4>", "k_combine<4>", "k_cellsort<4>", "k_scatter<0>", "k_project_count"):
        assert rows[k][col["spill st/ld B"]].startswith("0 "), f"{k} spills"
    assert int(rows["k_project_count"][col["RED"]]) >= 1                   # fire-and-forget reductions in the count pass
