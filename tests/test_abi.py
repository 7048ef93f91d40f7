"""CPU-side checks of the boundary: libmg.so builds, loads and exports every symbol include/mg.h declares;
argument validation that needs no GPU; the product never routes through the oracle."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2412_20522_b200 import build, binding

    build.build()
    return binding.lib()


def declared_symbols(testing=False):
    """Functions include/mg.h declares: the shipped ABI, or (testing=True) only what -DMG_TESTING adds to it."""
    text = open(os.path.join(ROOT, "include", "mg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    guarded = re.findall(r"#ifdef MG_TESTING\n(.*?)#endif", text, flags=re.S)
    text = "\n".join(guarded) if testing else re.sub(r"#ifdef MG_TESTING\n.*?#endif", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mg_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_five_calls():
    syms = declared_symbols()
    for s in ("mg_preprocess", "mg_bin_sort", "mg_render_fwd", "mg_render_bwd", "mg_preprocess_bwd"):
        assert s in syms


def test_library_exports_every_declared_symbol(lib):
    from paper_2412_20522_b200 import binding

    for s in declared_symbols():
        assert hasattr(lib, s), f"libmg.so does not export {s}"
    assert sorted(binding.EXPORTS) == declared_symbols()
    assert lib.mg_version() >= 100


def test_test_hooks_are_only_in_the_test_build(lib):
    """mg_debug_set_lookback_spin_limit is process-wide state that can make every sort fail: it is compiled only with
    -DMG_TESTING, into libmg_testing.so, and the shipped libmg.so must not export it."""
    from paper_2412_20522_b200 import build

    hooks = declared_symbols(testing=True)
    assert hooks == ["mg_debug_set_lookback_spin_limit"]
    testing = C.CDLL(build.LIB_TESTING)
    for s in hooks:
        assert not hasattr(lib, s), f"libmg.so exports the test hook {s}"
        assert hasattr(testing, s), f"libmg_testing.so lacks {s}"
    for s in declared_symbols():
        assert hasattr(testing, s)


def test_workspace_bytes_host_logic(lib):
    from paper_2412_20522_b200 import binding

    assert binding.mg_workspace_bytes(-1, 64, 64, 10) == 0
    assert binding.mg_workspace_bytes(10, 0, 64, 10) == 0
    assert binding.mg_workspace_bytes(10, 64, 64, 1 << 32) == 0
    small = binding.mg_workspace_bytes(1000, 128, 128, 3000)
    big = binding.mg_workspace_bytes(1000, 128, 128, 3_000_000)
    assert 0 < small < big
    # layout of bin_sort v2: 8 B of row records per key of capacity, 24 B per Gaussian (depth keys, ids, packed
    # rects), plus the look-back status words and count tables (a few % of that)
    keys_only = binding.mg_workspace_bytes(0, 512, 512, 1_000_000)
    assert 8e6 <= keys_only < 9.5e6
    both = binding.mg_workspace_bytes(1_000_000, 512, 512, 1_000_000)
    assert 24e6 <= both - keys_only < 28e6


def test_invalid_arguments_are_rejected_without_a_gpu(lib):
    from paper_2412_20522_b200 import binding

    cam = binding.mg_camera()
    cam.width, cam.height, cam.fx, cam.fy, cam.sh_degree = 64, 64, 50.0, 50.0, 7
    rc = lib.mg_render_fwd(C.byref(cam), *[C.c_void_p(0)] * 11)
    assert rc == binding.MG_ERR_INVALID_ARG and b"sh_degree" in lib.mg_last_error_string()
    cam.sh_degree = 0
    rc = lib.mg_render_fwd(C.byref(cam), *[C.c_void_p(0)] * 11)
    assert rc == binding.MG_ERR_INVALID_ARG and b"null" in lib.mg_last_error_string()
    rc = lib.mg_bin_sort(C.byref(cam), C.c_int64(-5), *[C.c_void_p(0)] * 3, C.c_uint64(0), C.c_void_p(0), C.c_size_t(0),
                         *[C.c_void_p(0)] * 5)
    assert rc == binding.MG_ERR_INVALID_ARG
    rc = lib.mg_preprocess(None, C.c_int64(1), *[C.c_void_p(0)] * 16)
    assert rc == binding.MG_ERR_INVALID_ARG


def test_product_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2412_20522_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M), f
                assert "mg_oracle" not in src and "libmg_oracle" not in src, f
    orc_src = open(os.path.join(ROOT, "oracle", "mg_oracle.cpp")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_2412_20522_b200" not in orc_src.replace("paper_2412_20522_b200/csrc (the", "").replace("paper_2412_20522_b200 never", "")
    assert '#include "mg' not in orc_src


def test_constants_agree_between_header_and_oracle():
    """The oracle keeps its own copy of the readings (no shared header); the values must coincide."""
    h = open(os.path.join(ROOT, "include", "mg.h")).read()
    o = open(os.path.join(ROOT, "oracle", "mg_oracle.cpp")).read()

    def hv(name):
        return re.search(rf"#define {name} (.*?)\s*/\*", h).group(1).strip()

    def ov(name):
        return re.search(rf"const (?:double|int) {name} = ([^;]+);", o).group(1).strip()

    ev = lambda s: eval(s.replace("f", ""))
    for a, b in (("MG_TILE", "TILE"), ("MG_ALPHA_MIN", "ALPHA_MIN"), ("MG_ALPHA_MAX", "ALPHA_MAX"), ("MG_T_MIN", "T_MIN"),
                 ("MG_DILATION", "DILATION"), ("MG_ZNEAR", "ZNEAR"), ("MG_JCLAMP", "JCLAMP"), ("MG_EIG_FLOOR", "EIG_FLOOR")):
        assert abs(ev(hv(a)) - ev(ov(b))) < 1e-12, (a, hv(a), ov(b))


def test_invalid_arguments_of_the_next_rows_are_rejected_without_a_gpu(lib):
    """Mask head, compaction and render loss: argument checks happen before any CUDA call."""
    from paper_2412_20522_b200 import binding

    null = C.c_void_p(0)
    rc = lib.mg_mask_sample(C.c_int64(10), null, null, C.c_float(0.0), null, null, null)
    assert rc == binding.MG_ERR_INVALID_ARG and b"tau" in lib.mg_last_error_string()
    rc = lib.mg_mask_sample(C.c_int64(10), null, null, C.c_float(1.0), null, null, null)
    assert rc == binding.MG_ERR_INVALID_ARG and b"null" in lib.mg_last_error_string()
    assert lib.mg_mask_sample(C.c_int64(0), null, null, C.c_float(1.0), null, null, null) == binding.MG_OK
    rc = lib.mg_mask_sample_bwd(C.c_int64(-1), null, null, C.c_float(1.0), null, null)
    assert rc == binding.MG_ERR_INVALID_ARG
    rc = lib.mg_mask_loss(C.c_int64(0), null, C.c_float(0.1), null, null, null)
    assert rc == binding.MG_ERR_INVALID_ARG  # the mean over zero Gaussians is undefined
    rc = lib.mg_mask_prune_keep(C.c_int64(5), C.c_int32(-1), null, null, null, null)
    assert rc == binding.MG_ERR_INVALID_ARG
    assert binding.mg_compact_workspace_bytes(-1) == 0 and binding.mg_compact_workspace_bytes(1000) >= 4000
    rc = lib.mg_compact(C.c_int64(10), null, C.c_int32(17), null, null, null, null, C.c_size_t(0), null, null)
    assert rc == binding.MG_ERR_INVALID_ARG and b"n_arrays" in lib.mg_last_error_string()
    assert binding.mg_render_loss_workspace_bytes(0, 5) == 0
    assert binding.mg_render_loss_workspace_bytes(10, 5) == 9 * 4 * 50
    rc = lib.mg_render_loss(C.c_int32(10), C.c_int32(5), null, null, C.c_float(0.2), null, null, null, C.c_size_t(0), null)
    assert rc == binding.MG_ERR_INVALID_ARG


def test_invalid_arguments_of_f4_are_rejected_without_a_gpu(lib):
    """Density statistics and the optimiser step: argument checks happen before any CUDA call."""
    from paper_2412_20522_b200 import binding

    null = C.c_void_p(0)
    rc = lib.mg_density_stats(C.c_int64(10), null, null, C.c_float(1.0), C.c_float(1.0), null, null, null, null)
    assert rc == binding.MG_ERR_INVALID_ARG and b"null" in lib.mg_last_error_string()
    assert lib.mg_density_stats(C.c_int64(0), null, null, C.c_float(1.0), C.c_float(1.0), null, null, null, null) == 0
    grp = (binding.mg_adam_group * 1)()
    grp[0].n_rows, grp[0].row_floats, grp[0].lr = 10, 3, 0.1
    f = lambda *a: lib.mg_adam_step(*a)
    assert f(C.c_int32(1), grp, C.c_float(0.9), C.c_float(0.999), C.c_float(1e-15), C.c_int64(1), null, null) == binding.MG_ERR_INVALID_ARG
    assert b"null" in lib.mg_last_error_string()
    assert f(C.c_int32(1), grp, C.c_float(0.9), C.c_float(0.999), C.c_float(1e-15), C.c_int64(0), null, null) == binding.MG_ERR_INVALID_ARG
    assert f(C.c_int32(1), grp, C.c_float(1.0), C.c_float(0.999), C.c_float(1e-15), C.c_int64(1), null, null) == binding.MG_ERR_INVALID_ARG
    assert f(C.c_int32(9), grp, C.c_float(0.9), C.c_float(0.999), C.c_float(1e-15), C.c_int64(1), null, null) == binding.MG_ERR_INVALID_ARG
    assert f(C.c_int32(0), null, C.c_float(0.9), C.c_float(0.999), C.c_float(1e-15), C.c_int64(1), null, null) == 0
