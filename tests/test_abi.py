"""CPU checks of the boundary: libqp.so builds with nvcc (no GPU needed), loads, exports every symbol that
include/qp.h declares, and its host-only entry points behave. No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1512_07437_b200 import build as qp_build
from paper_1512_07437_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    return qp_build.build()


def test_exports_every_declared_symbol(lib_path):
    hdr = open(os.path.join(ROOT, "include", "qp.h")).read()
    declared = set(re.findall(r"\b(qp_[a-z_]+)\s*\(", hdr))
    assert {"qp_posteriors", "qp_workspace_bytes", "qp_status_string", "qp_version", "qp_last_launch_count"} <= declared
    lib = C.CDLL(lib_path)
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in qp.h but not exported"


def test_binding_names_match_header(lib_path):
    from paper_1512_07437_b200 import qp
    for name in qp.EXPORTS:
        assert hasattr(qp._lib, name)
    assert qp.status_string(0) == "ok" and "nnz" in qp.status_string(qp.ERR["NNZ_CAPACITY"])
    assert "sm_100a" in qp.version()


def test_workspace_query_is_host_only_and_validates(lib_path, default_params):
    from paper_1512_07437_b200 import qp
    fam = inputs.config_family(0)
    pairs = inputs.all_pairs(fam.k)
    cp = qp.CParams(default_params)
    full = qp.workspace_bytes(fam.offsets, fam.k, pairs, cp, nnz_capacity=10000)
    assert full > 0
    capped = qp.workspace_bytes(fam.offsets, fam.k, pairs, cp, nnz_capacity=10000, budget=full // 2)
    assert capped <= full // 2 or capped == full
    with pytest.raises(qp.QpError) as ei:
        qp.workspace_bytes(fam.offsets, fam.k, pairs, cp, nnz_capacity=10000, budget=4096)
    assert ei.value.code == qp.ERR["WORKSPACE_TOO_SMALL"]
    with pytest.raises(qp.QpError) as ei:
        qp.workspace_bytes(fam.offsets, fam.k, np.array([[0, 0]], np.int32), cp, nnz_capacity=1)
    assert ei.value.code == qp.ERR["BAD_PAIR"]
    with pytest.raises(qp.QpError) as ei:
        qp.workspace_bytes(fam.offsets, fam.k, np.array([[0, 99]], np.int32), cp, nnz_capacity=1)
    assert ei.value.code == qp.ERR["BAD_PAIR"]
    bad = inputs.default_params()
    bad.threshold = 0.0
    with pytest.raises(qp.QpError) as ei:
        qp.workspace_bytes(fam.offsets, fam.k, pairs, qp.CParams(bad), nnz_capacity=1)
    assert ei.value.code == qp.ERR["INVALID_ARG"]
    # fp64 needs more scratch than fp32 for the same pairs
    assert qp.workspace_bytes(fam.offsets, fam.k, pairs, qp.CParams(default_params, precision="fp64"), 10000) > 0


def test_kernels_are_sm100a_sass(lib_path):
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", lib_path], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_header_is_plain_c(tmp_path):
    """include/qp.h is a C header: it compiles with a C99 compiler, no C++ and no CUDA types in the signatures."""
    import subprocess
    src = tmp_path / "t.c"
    src.write_text('#include "qp.h"\nint main(void) { qp_params p; qp_output o; qp_host_output h; qp_csr c; qp_csr_out co;\n'
                   'qp_consistency_params cp; qp_peaks pk; (void)p; (void)o; (void)h; (void)c; (void)co; (void)cp; (void)pk;\n'
                   'return QP_OK; }\n')
    r = subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I" + os.path.join(ROOT, "include"), "-c",
                        str(src), "-o", str(tmp_path / "t.o")], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
