"""CPU-side checks of the C-ABI library (no GPU, no compute calls): libgpfc.so builds, loads,
exports every function include/gpfc.h declares, the Python binding names the same set, and the
host-side argument validation / sizing logic behaves as the header says."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2312_02063_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def declared_functions():
    src = open(os.path.join(ROOT, "include", "gpfc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gpfc_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert {"gpfc_make_period_grid", "gpfc_fold", "gpfc_normalize", "gpfc_fold_batch"} <= set(names)
    for n in names:
        assert getattr(lib, n) is not None, n


def test_binding_names_match_header():
    from paper_2312_02063_b200 import binding
    assert sorted(binding.EXPORTS) == declared_functions()
    for n in binding.EXPORTS:
        assert hasattr(binding, n), "binding lacks %s" % n


def test_binding_does_not_import_the_oracle():
    import paper_2312_02063_b200.binding as b
    import paper_2312_02063_b200.workloads as w
    for mod in (b, w):
        text = open(mod.__file__).read()
        assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M)
    for fn in os.listdir(os.path.join(ROOT, "paper_2312_02063_b200", "csrc")):
        text = open(os.path.join(ROOT, "paper_2312_02063_b200", "csrc", fn)).read()
        assert "gpfc_ref" not in text and "oracle/" not in text.replace("under oracle/", "")


def test_host_side_validation_without_gpu(lib):
    lib.gpfc_n_sample.restype = ctypes.c_double
    lib.gpfc_n_sample.argtypes = [ctypes.c_double] * 3
    assert int(lib.gpfc_n_sample(2.0, 4 * 365.0, 0.03)) == 97333
    lib.gpfc_last_error.restype = ctypes.c_char_p
    lib.gpfc_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.gpfc_version()
    f64, i64, i32, vp = ctypes.c_double, ctypes.c_int64, ctypes.c_int, ctypes.c_void_p
    lib.gpfc_make_period_grid.argtypes = [f64, f64, i64, i32, vp]
    assert lib.gpfc_make_period_grid(-1.0, 1.0, 10, 0, None) == 1          # INVALID_ARG
    assert lib.gpfc_make_period_grid(0.5, 0.2, 10, 0, None) == 1
    assert lib.gpfc_make_period_grid(0.2, 1.0, -1, 0, None) == 1
    assert lib.gpfc_make_period_grid(0.2, 1.0, 0, 0, None) == 0            # valid no-op
    assert lib.gpfc_make_period_grid(0.2, 1.0, 5, 0, None) == 1            # NULL output
    assert lib.gpfc_last_error() != b""
    lib.gpfc_fold.argtypes = [vp, vp, i64, vp, i64, i32, f64, vp, vp]
    assert lib.gpfc_fold(None, None, -1, None, 0, 16, 0.0, None, None) == 1
    assert lib.gpfc_fold(None, None, 0, None, 3, 0, 0.0, None, None) == 2  # UNSUPPORTED nbins
    assert lib.gpfc_fold(None, None, 0, None, 3, 5000, 0.0, None, None) == 2
    assert lib.gpfc_fold(None, None, 0, None, 0, 16, 0.0, None, None) == 0  # nperiods = 0
    assert lib.gpfc_fold(None, None, 0, None, 3, 16, 0.0, None, None) == 1  # periods NULL
    lib.gpfc_normalize.argtypes = [vp, vp, i64, i32, vp]
    assert lib.gpfc_normalize(None, None, 0, 64, None) == 0
    assert lib.gpfc_normalize(None, None, 4, 64, None) == 1
    assert lib.gpfc_normalize(None, None, 4, 0, None) == 2
    fb = [vp, vp, vp, i64, i64, vp, i64, i32, vp, vp, vp, vp]
    lib.gpfc_fold_batch.argtypes = fb
    assert lib.gpfc_fold_batch(None, None, None, 2, 10, None, 4, 64, None, None, None, None) == 1
    assert lib.gpfc_fold_batch(None, None, None, 0, 0, None, 4, 64, None, None, None, None) == 0
    lib.gpfc_fold_batch_host.argtypes = fb
    assert lib.gpfc_fold_batch_host(None, None, None, 2, 10, None, 4, 64, None, None, None, None) == 1
    # gpfc_fold_noalloc refuses sizes beyond its static scratch before it touches the device
    lib.gpfc_fold_noalloc.argtypes = [vp, vp, i64, vp, i64, i32, f64, vp, vp, vp]
    assert lib.gpfc_fold_noalloc(None, None, 131073, None, 8, 64, 0.0, None, None, None) == 2
    assert b"GPFC_NOALLOC_MAX_SAMPLES" in lib.gpfc_last_error()
    assert lib.gpfc_fold_noalloc(None, None, 100, None, 262145, 64, 0.0, None, None, None) == 2
    assert b"GPFC_NOALLOC_MAX_PERIODS" in lib.gpfc_last_error()
    assert lib.gpfc_fold_noalloc(None, None, -1, None, 8, 64, 0.0, None, None, None) == 1
    assert lib.gpfc_fold_noalloc(None, None, 100, None, 8, 0, 0.0, None, None, None) == 2
    lib.gpfc_set_workspace.argtypes = [vp, ctypes.c_size_t]
    assert lib.gpfc_set_workspace(None, 16) == 1
    assert lib.gpfc_set_workspace(None, 0) == 0


def test_workspace_bytes_covers_the_scratch_layout(lib):
    lib.gpfc_workspace_bytes.restype = ctypes.c_size_t
    lib.gpfc_workspace_bytes.argtypes = [ctypes.c_int64] * 3 + [ctypes.c_int]
    assert lib.gpfc_workspace_bytes(-1, 0, 0, 64) == 0
    for nc, n, npd in [(1, 4000, 2000), (1024, 1024 * 65000, 20000), (7, 5194, 50)]:
        b = lib.gpfc_workspace_bytes(nc, n, npd, 256)
        # u (8) + q (4) + records (8) per sample, tile table, per-curve and per-period tables
        assert b >= n * 20 + (n // 128 + nc) * 16 + nc * 64 + npd * 8
        assert b <= n * 20 + (n // 128 + nc) * 16 + nc * 128 + npd * 8 + 16 * 4096
    # monotone in every size
    assert lib.gpfc_workspace_bytes(2, 1000, 10, 64) <= lib.gpfc_workspace_bytes(3, 2000, 20, 64)
