"""CPU-side checks of the C-ABI boundary: libgs.so builds for sm_100a, loads without a GPU, and exports every symbol
that include/gs.h declares (no compute calls are made here)."""
import ctypes
import os
import re

from paper_2606_16566_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "gs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gs_[a-z_0-9]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    names = _declared()
    assert "gs_render" in names and "gs_workspace_bytes" in names and len(names) >= 10
    for n in names:
        assert hasattr(lib, n), "include/gs.h declares %s but libgs.so does not export it" % n
    assert set(binding.EXPORTS) == set(names), "binding.EXPORTS out of sync with include/gs.h"


def test_workspace_bytes_and_error_strings_host_only():
    # host-only entry points: layout arithmetic and strings
    a = binding.gs_workspace_bytes(1000, 128, 128, 10_000)
    b = binding.gs_workspace_bytes(1000, 128, 128, 20_000)
    c = binding.gs_workspace_bytes(2000, 128, 128, 10_000)
    assert 0 < a < b and a < c and a % 256 == 0
    # small frames fuse the duplication into the first tile pass: 8 (entries) + 4 (ids) bytes per duplicate;
    # large frames keep a second 8-byte entry buffer for the stand-alone duplication (the sorted super-tile ids of the
    # two-level binning share the first one)
    small = binding.gs_workspace_bytes(0, 800, 800, 1 << 20) - binding.gs_workspace_bytes(0, 800, 800, 0)
    large = binding.gs_workspace_bytes(0, 800, 800, 8 << 20) - binding.gs_workspace_bytes(0, 800, 800, 0)
    assert (1 << 20) * 12 <= small < (1 << 20) * 16
    assert (8 << 20) * 20 <= large < (8 << 20) * 23
    L = binding.lib()
    assert L.gs_workspace_bytes(-1, 10, 10, 0) == 0 and L.gs_workspace_bytes(1, 0, 10, 0) == 0
    assert L.gs_workspace_bytes(1, 10, 10, 1 << 32) == 0
    assert binding.gs_error_string(0) == "ok"
    for code in (-1, -2, -3, -4):
        assert binding.gs_error_string(code) not in ("ok", "unknown error")
    assert L.gs_set_render_variant(9) == binding.GS_ERR_BAD_ARG
    assert L.gs_set_render_variant(4) == 0 and binding.gs_get_render_variant() == 4
    assert L.gs_set_render_variant(5) == binding.GS_ERR_BAD_ARG          # the removed warp-specialised experiment
    # host-only argument checks of the round-2 entry points
    assert L.gs_set_rank_mode(2) == binding.GS_ERR_BAD_ARG and L.gs_set_rank_mode(-1) == 0
    assert L.gs_set_tile_cull(7) == binding.GS_ERR_BAD_ARG and L.gs_set_tile_cull(0) == 0
    fake = ctypes.c_void_p(0x1000)
    assert L.gs_set_workspace_option(fake, 9, 0) == binding.GS_ERR_BAD_ARG
    assert L.gs_set_workspace_option(fake, binding.GS_OPT_RENDER_VARIANT, 5) == binding.GS_ERR_BAD_ARG
    assert L.gs_set_workspace_option(fake, binding.GS_OPT_TILE_CULL, 3) == binding.GS_ERR_BAD_ARG
    assert L.gs_set_workspace_option(fake, binding.GS_OPT_TILE_CULL, 2) == 0 and L.gs_set_workspace_option(fake, binding.GS_OPT_TILE_CULL, -1) == 0
    assert L.gs_set_workspace_option(None, 0, 0) == binding.GS_ERR_BAD_ARG
    assert L.gs_set_workspace_option(fake, binding.GS_OPT_STATS, 1) == 0 and L.gs_release(fake) == 0   # nothing CUDA was created
    assert L.gs_release(fake) == 0 and L.gs_release(None) == binding.GS_ERR_BAD_ARG


def test_product_does_not_import_oracle():
    """The product path must never route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2606_16566_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "gs_oracle" not in txt, f
