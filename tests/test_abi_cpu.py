"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol that
include/qmll.h declares; host-side argument checks and workspace arithmetic work without a GPU (no compute)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2206_01580_b200 import build as qbuild
    qbuild.build()
    import paper_2206_01580_b200 as pkg
    return pkg, pkg.load_library()


def declared_symbols():
    names = set()
    inc = os.path.join(ROOT, "include")
    for h in sorted(os.listdir(inc)):
        if h.endswith(".h"):
            text = open(os.path.join(inc, h)).read()
            text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
            names |= set(re.findall(r"\b(qmll_[a-z_0-9]+)\s*\(", text))
    return sorted(names)


def test_header_symbols_are_exported(lib):
    pkg, l = lib
    names = declared_symbols()
    assert {"qmll_sorf_forward", "qmll_sorf_backward_forces", "qmll_normal_equations", "qmll_predict"} <= set(names)
    for n in names:
        assert hasattr(l, n), n
    assert set(pkg.EXPORTS) <= set(names)


def test_status_strings(lib):
    pkg, l = lib
    assert l.qmll_status_string(0) == b"QMLL_OK"
    for code in (-1, -2, -3, -4):
        assert l.qmll_status_string(code).startswith(b"QMLL_ERR")


def test_workspace_arithmetic(lib):
    pkg, l = lib
    p = pkg._CParams(128, 8192, 3, 5, 8.0, None, None)
    fwd = l.qmll_workspace_bytes(pkg.CALL_FORWARD, ctypes.byref(p), 21000, 1000, 0)
    fwdg = l.qmll_workspace_bytes(pkg.CALL_FORWARD_GRAD, ctypes.byref(p), 21000, 1000, 0)
    pred = l.qmll_workspace_bytes(pkg.CALL_PREDICT, ctypes.byref(p), 21000, 1000, 0)
    assert fwd >= 5 * 8192 * 4 + 5 * 64 * 3 * 128 // 8          # permuted bias + packed sign bits
    assert fwdg - fwd >= 21000 * 8192 * 4                        # per-atom sin table for the force rows
    assert pred >= fwd + 8192 * 4 + 1000 * 8                     # + alpha table + fp64 energy accumulators (g stays on-chip)
    ne = l.qmll_workspace_bytes(pkg.CALL_NORMAL_EQUATIONS, ctypes.byref(p), 0, 0, 64000)
    assert ne >= 2 * 8192 * 64000 * 2                            # fp16 hi + lo copies of A^T
    assert 0 < l.qmll_normal_equations_min_workspace(8192) <= ne
    assert l.qmll_normal_equations_workspace(64000, 8192, pkg.NE_SPLIT_TF32) >= 2 * 8192 * 64000 * 4
    assert l.qmll_normal_equations_workspace(64000, 8192, 7) == 0
    bad = pkg._CParams(100, 8192, 3, 5, 8.0, None, None)          # d not a power of two
    assert l.qmll_workspace_bytes(pkg.CALL_FORWARD, ctypes.byref(bad), 10, 1, 0) == 0


def test_host_side_argument_checks_need_no_gpu(lib):
    pkg, l = lib
    # null parameter struct / invalid sizes are rejected before any CUDA call
    assert l.qmll_sorf_forward(None, None, None, None, 0, 0, None, None, None, None, 0, None) == -1
    assert l.qmll_normal_equations(None, None, -1, 256, 0, None, None, None, 0, None) == -1
    assert l.qmll_normal_equations_mode(None, None, 4, 256, 0, None, None, None, 0, 9, None) == -1
    assert l.qmll_predict(None, None, None, None, 0, 0, None, None, None, None, None, 0, None) == -1
    assert l.qmll_sorf_backward_forces(None, None, None, None, 0, 0, None, None, None, None, 0, None) == -1
    assert l.qmll_energies(None, None, 4, 16, None, None) == -1 and l.qmll_energies(None, None, -1, 16, None, None) == -1
    # the static-scratch prediction: null / invalid parameters and problems beyond the array are rejected on the host
    assert l.qmll_predict_static(None, None, None, None, 0, 0, None, None, None, None, None) == -1
    assert int(l.qmll_predict_static_max_bytes()) == 4 << 20
    bad = pkg._CParams(48, 96, 3, 2, 1.0, None, None)                      # d not a power of two
    assert l.qmll_predict_static(ctypes.byref(bad), None, None, None, 0, 0, None, None, None, None, None) == -1
    big = pkg._CParams(256, 65536, 3, 16, 1.0, None, None)                 # 4.9 MB of tables
    assert l.qmll_workspace_bytes(pkg.CALL_PREDICT, ctypes.byref(big), 0, 1000, 0) > 4 << 20
    assert l.qmll_predict_static(ctypes.byref(big), None, None, None, 0, 1000, None, None, None, None, None) == -3


def test_next_row_entry_points_check_arguments_on_the_host(lib):
    """FCHL19, projections, tensor-core feature map: parameter checks and size arithmetic need no GPU."""
    pkg, l = lib
    fp = pkg.Fchl19Params().c()
    assert l.qmll_fchl19_rep_size(ctypes.byref(fp)) == 5 * 24 + 5 * 6 * 20 == 720          # Table I (E + F), 5 elements
    e = pkg.Fchl19Params(n2=23, n3=22).c()
    assert l.qmll_fchl19_rep_size(ctypes.byref(e)) == 5 * 23 + 30 * 22
    assert l.qmll_fchl19_rep_size(ctypes.byref(pkg.Fchl19Params(n3=40).c())) == -1          # beyond 32 grid points
    assert l.qmll_fchl19_rep_size(ctypes.byref(pkg.Fchl19Params(r_cut=0.0).c())) == -1
    assert l.qmll_fchl19(None, None, None, 0, None, None, 0, None, None, None, None, None) == -1
    bad = pkg.Fchl19Params(n_elem=17).c()
    assert l.qmll_fchl19(ctypes.byref(bad), None, None, 0, None, None, 0, None, None, None, None, None) == -2
    assert l.qmll_fchl19(ctypes.byref(fp), None, None, 5, None, None, 4, None, None, None, None, None) == -1   # no info
    assert l.qmll_fchl19_backward(ctypes.byref(fp), None, None, 5, None, None, 4, None, None, None, None) == -1
    assert l.qmll_project_neighbor(None, None, None, 3, 2, 0, 16, 2, None, None, None) == -1
    assert l.qmll_project_back(None, None, 3, 10, 18, 2, None, None, None) == -1              # d % 4 != 0
    assert l.qmll_rff_forward(None, None, 128, 512, 2, None, None, None, 0, 0, None, None, 0, None) == -1
    assert l.qmll_sorf_forward_mma(None, None, None, None, 0, 0, None, None, 0, None) == -1
    assert l.qmll_sorf_backward_g(None, None, None, None, 0, 0, None, None, None, None, 0, None) == -1
    ws_s = l.qmll_featmap_workspace_bytes(128, 16384, 5, 1_600_000, 0)
    ws_r = l.qmll_featmap_workspace_bytes(128, 16384, 5, 1_600_000, 1)
    assert ws_s >= 5 * 16384 * 128 * 2 + 2 * 1_600_000 * 128 * 2        # fp16 W table + hi / lo copies of x
    assert ws_r - ws_s >= 5 * 16384 * 128 * 2 - (1 << 22)               # RFF: W as hi + lo
    assert l.qmll_featmap_workspace_bytes(0, 16384, 5, 10, 0) == 0


def test_launch_counter(lib):
    pkg, l = lib
    pkg.reset_launch_count()
    assert pkg.launch_count() == 0


def test_product_never_imports_oracle():
    pkgdir = os.path.join(ROOT, "paper_2206_01580_b200")
    for dirpath, _, files in os.walk(pkgdir):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "sorf_oracle" not in text \
                    and "fchl19_oracle" not in text, f
    otext = "".join(open(os.path.join(ROOT, "oracle", f)).read() for f in ("__init__.py", "sorf_oracle.c", "fchl19_oracle.c"))
    assert "import paper_2206_01580_b200" not in otext and "qmll.h" not in otext
