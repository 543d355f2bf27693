"""Host-side checks of the C ABI that need no GPU: the library loads, exports every symbol that
include/opx.h declares, validates its arguments, and refuses to compute without a device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2309_12496_b200 as pkg
import workloads as wl
from paper_2309_12496_b200 import opx
from workloads.scenes import MAT_ABSORBER, MAT_DETECTOR, MAT_MIRROR, N_LAMBDA, Scene

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2309_12496_b200 import build
    build.build()
    return pkg.load_library()


def test_every_declared_symbol_is_exported(lib):
    header = open(os.path.join(ROOT, "include", "opx.h")).read()
    declared = set(re.findall(r"\b(opx_[a-z0-9_]+)\s*\(", header))
    assert declared == set(pkg.EXPORTS)
    # the debugging / measurement exports live in their own header, outside the product boundary
    debug = set(re.findall(r"\b(opx_[a-z0-9_]+)\s*\(", open(os.path.join(ROOT, "include", "opx_debug.h")).read()))
    assert debug == set(pkg.DEBUG_EXPORTS) and not (debug & declared)
    for name in declared | debug:
        assert hasattr(lib, name), name
    assert lib.opx_version().decode().startswith("opx")
    assert lib.opx_last_error() is not None


def test_struct_sizes_match_header(lib):
    assert C.sizeof(opx.SceneParams) == 20 and C.sizeof(opx.PixelFrame) == 56
    assert C.sizeof(opx.Mesh) == 48 and C.sizeof(opx.Hits) == 48 and C.sizeof(opx.SceneLayout) == 112 and C.sizeof(opx.Detected) == 32


def test_scene_create_and_info(lib):
    sc = wl.toy_rich_scene()
    s = pkg.Scene(sc)
    assert (s.n_triangles, s.n_nodes, s.n_pixels, s.n_surfaces) == (20014, 20013, 208 * 208, 3)
    scene_b, tmp_b = s.workspace_bytes()
    lay = s.layout()
    assert lay["total_bytes"] == scene_b and scene_b >= 20013 * 64 + 20014 * 64 and tmp_b > 20014 * 36
    offs = [lay[k] for k in ("nodes", "triangles", "normals", "surfaces", "mat_kinds", "tables", "frames",
                             "sorted_keys", "parents", "wide_nodes")]
    assert offs == sorted(offs) and all(o % 256 == 0 for o in offs)
    empty = pkg.Scene(Scene())
    assert (empty.n_triangles, empty.n_pixels) == (0, 0)


def _bad(mutate):
    sc = wl.toy_rich_scene(cells=4)
    mutate(sc)
    with pytest.raises(pkg.OpxError) as e:
        pkg.Scene(sc)
    assert e.value.status == opx.OPX_ERR_INVALID_ARG
    return str(e.value)


def test_scene_create_rejects_bad_arguments(lib):
    assert "n_lambda" in _bad(lambda s: setattr(s, "n_lambda", 1))
    assert "lambda_max" in _bad(lambda s: setattr(s, "lambda_max", 100.0))
    assert "max_bounces" in _bad(lambda s: setattr(s, "max_bounces", 0))
    assert "max_bounces" in _bad(lambda s: setattr(s, "max_bounces", 256))
    assert "t_min" in _bad(lambda s: setattr(s, "t_min", -1.0))
    assert "material" in _bad(lambda s: s.meshes[0].__setitem__("material", 9))
    assert "frame" in _bad(lambda s: s.meshes[1].__setitem__("frame", -1))
    assert "frame" in _bad(lambda s: s.meshes[1].__setitem__("frame", 5))
    assert "vertex index" in _bad(lambda s: s.meshes[0]["indices"].__setitem__((0, 0), 10 ** 6))
    assert "pitch" in _bad(lambda s: s.frames[0].__setitem__("pitch_u", 0.0))
    assert "grid" in _bad(lambda s: s.frames[0].__setitem__("nu", 0))
    assert "table" in _bad(lambda s: s.materials[1]["table"].__setitem__(3, 1.5))
    assert "table" in _bad(lambda s: s.materials[2]["table"].__setitem__(3, np.nan))
    assert "kind" in _bad(lambda s: s.materials[0].__setitem__("kind", 7))
    # NULL handles
    assert lib.opx_scene_create(None, None, 0, None, 0, None, 0, None) == opx.OPX_ERR_INVALID_ARG
    assert lib.opx_scene_info(None, None, None, None, None) == opx.OPX_ERR_INVALID_ARG
    assert b"NULL" in lib.opx_last_error()


def test_no_device_means_an_error_not_a_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    s = pkg.Scene(wl.toy_rich_scene(cells=4))
    buf = (C.c_char * 4096)()
    addr = (C.addressof(buf) + 255) // 256 * 256
    st = lib.opx_bvh_build(s._h, C.c_void_p(addr), 1 << 30, C.c_void_p(addr), 1 << 30, None)
    assert st in (opx.OPX_ERR_CUDA, opx.OPX_ERR_UNSUPPORTED_DEVICE)
    h = opx.Hits()
    st = lib.opx_propagate(s._h, 1, 0, C.c_void_p(addr), C.c_void_p(addr), C.c_void_p(addr), 0, C.byref(h), None, None, None)
    assert st == opx.OPX_ERR_BAD_STATE and b"before opx_bvh_build" in lib.opx_last_error()


def test_missing_library_fails_loudly(tmp_path):
    with pytest.raises(pkg.OpxError):
        old, opx._lib = opx._lib, None
        try:
            opx.load_library(str(tmp_path / "libopx.so"))
        finally:
            opx._lib = old


def test_product_path_does_not_touch_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2309_12496_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", src, re.M), f
                assert "liboracle" not in src and "opx_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2309_12496_b200", src, re.M), f
            assert "libopx" not in src and "opx.h" not in src
    for f in os.listdir(os.path.join(ROOT, "workloads")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "workloads", f)).read()
            assert not re.search(r"^\s*(import|from)\s+(oracle|paper_2309_12496_b200)", src, re.M), f


def test_bench_reference_arm_prints_one_json_line():
    """`bench.py --impl reference` (the oracle timed on the host cores) needs no GPU and prints the contract's line."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                          "--reference-sample", "1500"], capture_output=True, text=True, timeout=600, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "photons/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["gpu_launches"] == 0


def test_prefilter_noalloc_checks_its_arguments_before_touching_a_device(lib):
    """opx_prefilter_noalloc (the filter for callers that cannot allocate device memory) validates like opx_prefilter:
    a NULL scene and a scene that was never built are refused on the host, with no CUDA call made."""
    args = (0, 0, None, None, None, 0, None, 0, None, None, None, None, 0, None, None)
    assert lib.opx_prefilter_noalloc(None, *args) == opx.OPX_ERR_INVALID_ARG and b"scene is NULL" in lib.opx_last_error()
    s = pkg.Scene(wl.toy_rich_scene(cells=4))
    assert lib.opx_prefilter_noalloc(s._h, *args) == opx.OPX_ERR_BAD_STATE
    assert b"opx_prefilter_noalloc before opx_bvh_build" in lib.opx_last_error()
    header = open(os.path.join(ROOT, "include", "opx.h")).read()
    assert f"#define OPX_PREFILTER_NOALLOC_MAX_PHOTONS {opx.PREFILTER_NOALLOC_MAX_PHOTONS}ull" in header
