"""The C-ABI library loads on a machine without a GPU and exports every symbol that
include/gsplat_b200.h declares; host-side argument validation works without a device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cuda_lib():
    from paper_2606_11390_b200 import build
    build.build()
    from paper_2606_11390_b200 import binding
    return binding


def _declared():
    src = open(os.path.join(ROOT, "include", "gsplat_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gs_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_five_north_star_entry_points():
    names = _declared()
    for n in ("gs_project_fwd", "gs_project_bwd", "gs_bin_tiles", "gs_raster_fwd", "gs_raster_bwd"):
        assert n in names


def test_library_exports_every_declared_symbol(cuda_lib):
    lib = cuda_lib.lib()
    names = _declared()
    assert len(names) >= 9
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(cuda_lib.EXPORTS) == names


def test_struct_layouts_match_header(cuda_lib):
    assert C.sizeof(cuda_lib.gs_camera) == 2 * 4 + 4 * 4 + 12 * 4 + 2 * 4
    assert C.sizeof(cuda_lib.gs_config) == 7 * 4


def test_default_config_and_status_strings(cuda_lib):
    cfg = cuda_lib.default_config()
    assert abs(cfg.dilation - 0.3) < 1e-7 and abs(cfg.alpha_min - 1 / 255) < 1e-9
    assert abs(cfg.alpha_max - 0.99) < 1e-7 and abs(cfg.t_min - 1e-4) < 1e-10
    assert cfg.extent == 3.0 and cfg.tile == 16 and cfg.sh_degree == 3
    assert cuda_lib.status_string(0) == "ok"
    assert "capacity" in cuda_lib.status_string(cuda_lib.GS_ERR_CAPACITY)


def test_host_side_validation_needs_no_gpu(cuda_lib):
    from paper_2606_11390_b200 import scenes
    lib = cuda_lib.lib()
    cams = cuda_lib.make_cameras([scenes.make_camera(64, 64, 64.0, 64.0, (0, 0, -3), (0, 0, 0), (0, -1, 0))])
    cfg = cuda_lib.default_config()
    # null pointers with N > 0
    rc = lib.gs_project_fwd(C.byref(cfg), C.c_int64(10), None, None, None, None, None, C.c_int32(1), cams,
                            None, None, None, None, None, None, None, None, None, None)
    assert rc == cuda_lib.GS_ERR_INVALID_ARGUMENT
    # bad SH degree, bad tile
    bad = cuda_lib.default_config(sh_degree=4)
    assert lib.gs_project_fwd(C.byref(bad), C.c_int64(0), None, None, None, None, None, C.c_int32(1), cams,
                              None, None, None, None, None, None, None, None, None, None) == cuda_lib.GS_ERR_INVALID_ARGUMENT
    bad = cuda_lib.default_config(tile=8)
    assert lib.gs_project_fwd(C.byref(bad), C.c_int64(0), None, None, None, None, None, C.c_int32(1), cams,
                              None, None, None, None, None, None, None, None, None, None) == cuda_lib.GS_ERR_UNSUPPORTED
    # N < 0, C out of range
    assert lib.gs_project_fwd(C.byref(cfg), C.c_int64(-1), None, None, None, None, None, C.c_int32(1), cams,
                              None, None, None, None, None, None, None, None, None, None) == cuda_lib.GS_ERR_INVALID_ARGUMENT
    assert lib.gs_project_fwd(C.byref(cfg), C.c_int64(0), None, None, None, None, None, C.c_int32(0), cams,
                              None, None, None, None, None, None, None, None, None, None) == cuda_lib.GS_ERR_INVALID_ARGUMENT
    # N == 0 is a no-op
    assert lib.gs_project_fwd(C.byref(cfg), C.c_int64(0), None, None, None, None, None, C.c_int32(1), cams,
                              None, None, None, None, None, None, None, None, None, None) == cuda_lib.GS_OK
    # workspace size query grows with capacity and is 256-byte granular
    a = cuda_lib.gs_bin_tiles_workspace_bytes(cfg, 1000, cams, 10_000)
    b = cuda_lib.gs_bin_tiles_workspace_bytes(cfg, 1000, cams, 1_000_000)
    assert b > a > 10_000 * 12 and a % 256 == 0
    # capacity beyond the 2^30 record limit
    n = C.c_size_t(0)
    assert lib.gs_bin_tiles(C.byref(cfg), C.c_int64(10), C.c_int32(1), cams, None, None, None, None, None, C.byref(n),
                            C.c_int64(1 << 30), None, None, None, None, None, C.c_int32(0), None) == cuda_lib.GS_ERR_UNSUPPORTED


def test_binding_refuses_cpu_tensors(cuda_lib):
    import torch
    with pytest.raises(TypeError):
        cuda_lib._ptr(torch.zeros(4))


def test_missing_library_fails_loudly(cuda_lib, monkeypatch):
    monkeypatch.setattr(cuda_lib, "_lib", None)
    monkeypatch.setattr(cuda_lib, "LIB_PATH", "/nonexistent/libgsplat_b200.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        cuda_lib.lib()
