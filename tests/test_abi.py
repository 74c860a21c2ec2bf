"""CPU-side checks of the C ABI: libscmd.so loads and exports every symbol include/scmd.h
declares; argument validation that needs no GPU.  No compute calls here."""
import ctypes

import pytest

import paper_1210_3559_b200 as pkg
from paper_1210_3559_b200 import build as pkg_build


@pytest.fixture(scope="module")
def lib():
    pkg_build.build()
    return pkg.load_library()


def test_header_symbols_are_all_exported(lib):
    names = pkg.exported_symbols()
    must = {"sc_create", "sc_destroy", "sc_density", "sc_forces", "sc_energy", "sc_step", "sc_kinetic",
            "sc_set_state", "sc_get_state", "sc_workspace_bytes", "sc_stats", "sc_eval_host", "sc_step_host",
            "sc_last_error", "sc_set_option", "sc_get_option", "sc_launch_count", "sc_rdf", "sc_msd",
            "sc_workspace_bytes_ex", "sc_create_ex"}
    assert must <= set(names)
    for name in names:
        assert hasattr(lib, name), f"{name} declared in include/scmd.h but not exported by libscmd.so"
    assert not any(n.startswith("sc_probe") for n in names)             # diagnostics live in their own library


def test_probe_library_exports_its_header():
    """libscmd_probe.so (include/scmd_probe.h): bench / test diagnostics, kept out of the product ABI."""
    from paper_1210_3559_b200 import binding
    probe = pkg.load_probe_library()
    names = [n for n in pkg.exported_symbols(binding._PROBE_HEADER) if n.startswith("sc_probe")]
    assert sorted(names) == ["sc_probe_reciprocal", "sc_probe_throughput"]
    for name in names:
        assert hasattr(probe, name)


def test_create_options_validation(lib):
    P = pkg.ScParams(9, 6, 1.5707e-2, 39.432, 3.52, 58.69, 10.0)
    base = lib.sc_workspace_bytes(ctypes.byref(P), 5000, pkg.SC_PREC_FP64, 1.0)
    same = lib.sc_workspace_bytes_ex(ctypes.byref(P), 5000, pkg.SC_PREC_FP64, 1.0, None)
    big = lib.sc_workspace_bytes_ex(ctypes.byref(P), 5000, pkg.SC_PREC_FP64, 1.0, ctypes.byref(pkg.ScCreateOptions(2048, 0)))
    assert base == same and big > base + 4 * 1000 * 5000                 # ~(2048 - 672) more entries per atom
    bad = pkg.ScCreateOptions(-1, 0)
    assert lib.sc_workspace_bytes_ex(ctypes.byref(P), 5000, pkg.SC_PREC_FP64, 1.0, ctypes.byref(bad)) == 0
    bad = pkg.ScCreateOptions(0, 1)
    assert lib.sc_workspace_bytes_ex(ctypes.byref(P), 5000, pkg.SC_PREC_FP64, 1.0, ctypes.byref(bad)) == 0
    Q = pkg.ScParams(9, 6, 1.5707e-2, 39.432, 3.52, 58.69, 0.0)
    with_n3 = lib.sc_workspace_bytes(ctypes.byref(Q), 65536, pkg.SC_PREC_FP64, 0.0)
    without = lib.sc_workspace_bytes_ex(ctypes.byref(Q), 65536, pkg.SC_PREC_FP64, 0.0, ctypes.byref(pkg.ScCreateOptions(0, 2)))
    assert without < 64 * 1024 * 1024 < with_n3                          # O(N) without the Newton's-third-law partials


def test_version_string(lib):
    assert b"libscmd" in lib.sc_version()


def test_workspace_bytes_validation(lib):
    P = pkg.ScParams(9, 6, 1.5707e-2, 39.432, 3.52, 58.69, 0.0)
    n1 = lib.sc_workspace_bytes(ctypes.byref(P), 1415, pkg.SC_PREC_FP64, 0.0)
    n2 = lib.sc_workspace_bytes(ctypes.byref(P), 65536, pkg.SC_PREC_FP64, 0.0)
    assert 0 < n1 < 64 * 1024 * 1024 and n1 < n2 < 1024 * 1024 * 1024    # N = 65536 carves 0.54 GB of Newton's-third-law partials
    n3 = lib.sc_workspace_bytes(ctypes.byref(P), 300000, pkg.SC_PREC_FP64, 0.0)  # beyond their range: O(N) again
    assert n3 < 256 * 1024 * 1024
    assert lib.sc_workspace_bytes(ctypes.byref(P), 0, pkg.SC_PREC_FP64, 0.0) == 0          # N < 1
    assert lib.sc_workspace_bytes(ctypes.byref(P), 100, 7, 0.0) == 0                       # precision
    assert lib.sc_workspace_bytes(ctypes.byref(P), 100, pkg.SC_PREC_FP64, -1.0) == 0       # skin < 0
    bad = pkg.ScParams(6, 9, 1.5707e-2, 39.432, 3.52, 58.69, 0.0)                          # n <= m
    assert lib.sc_workspace_bytes(ctypes.byref(bad), 100, pkg.SC_PREC_FP64, 0.0) == 0
    bad = pkg.ScParams(9, 6, -1.0, 39.432, 3.52, 58.69, 0.0)                               # eps <= 0
    assert lib.sc_workspace_bytes(ctypes.byref(bad), 100, pkg.SC_PREC_FP64, 0.0) == 0


def test_create_rejects_bad_arguments_without_a_device(lib):
    P = pkg.ScParams(9, 6, 1.5707e-2, 39.432, 3.52, 58.69, 0.0)
    ctx = ctypes.c_void_p()
    assert lib.sc_create(ctypes.byref(P), 100, 0, 0.0, None, 1 << 20, None, ctypes.byref(ctx)) == pkg.binding.SC_ERR_INVALID
    assert lib.sc_create(ctypes.byref(P), 100, 0, 0.0, 4096 + 8, 1 << 20, None, ctypes.byref(ctx)) == pkg.binding.SC_ERR_INVALID
    assert lib.sc_create(ctypes.byref(P), 100, 0, 0.0, 4096, 16, None, ctypes.byref(ctx)) == pkg.binding.SC_ERR_NOMEM
    assert not ctx.value


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(pkg.ScError):
        pkg.SuttonChen(147)
