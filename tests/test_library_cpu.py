"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/bta.h declares; argument errors are reported without a GPU; no product module imports oracle/."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as ge
    ge.build()
    import paper_2605_06392_b200 as pkg
    return pkg.lib()


def declared_symbols():
    names = set()
    for hdr in ("bta.h", "bta_diag.h"):
        src = open(os.path.join(ROOT, "include", hdr)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b((?:bta|inla)_[a-z0-9_]+)\s*\(", src))
    return sorted(names)


def test_every_declared_symbol_is_exported(lib):
    names = declared_symbols()
    assert {"bta_create", "bta_destroy", "bta_assemble", "bta_factor_logdet", "bta_solve", "bta_selinv",
            "inla_value_and_grad", "bta_workspace_bytes", "bta_last_error"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    out = subprocess.run(["nm", "-D", "--defined-only", os.path.join(ROOT, "paper_2605_06392_b200", "libbta_b200.so")],
                         capture_output=True, text=True).stdout
    for n in names:
        assert re.search(rf"\bT {n}\b", out), n
    # built with -fvisibility=hidden: nothing but the declared entry points is exported
    exported = set(re.findall(r"\b[TDB] (\w+)", out))
    assert exported == set(names), exported ^ set(names)


def test_library_holds_sm100a_dmma_code():
    so = os.path.join(ROOT, "paper_2605_06392_b200", "libbta_b200.so")
    out = subprocess.run(["cuobjdump", "-lelf", so], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_argument_errors_without_gpu(lib):
    h = ctypes.c_void_p()
    assert lib.bta_create(ctypes.byref(h), None, None, 0) == 1            # BTA_ERR_ARG
    assert b"null" in lib.bta_last_error()
    assert lib.bta_workspace_bytes(None) == 0
    assert lib.bta_destroy(None) == 0


def test_create_fails_loudly_without_a_b200(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2605_06392_b200 import BtaError, BtaModel
    from workloads import make_w0
    model, obs, th = make_w0()
    with pytest.raises(BtaError) as ei:
        BtaModel.from_workload(model, obs)
    assert ei.value.code == 3                                              # BTA_ERR_NODEVICE: no CPU fallback


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2605_06392_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower().replace("no oracle", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2605_06392_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "`paper_2605_06392_b200/`", "")


def test_gemm_flop_count_matches_brute_force(lib):
    """Host logic behind bench.py's in-step TFLOP/s: the element-exact flop count of a GEMM launch with a restricted
    k-range (KLO_*/KHI_* of csrc/common.cuh) and a lower-only output, against a triple loop."""
    import itertools
    from paper_2605_06392_b200.binding import gemm_alg_flop
    for (M, N, K) in [(7, 7, 7), (5, 9, 6), (9, 5, 12), (1, 1, 1), (13, 13, 4)]:
        for klo, khi, out in itertools.product((0, 1, 2), (0, 1, 2), (0, 1, 2)):
            want = 0
            for m in range(M):
                for n in range(N):
                    if out != 0 and n > m:
                        continue
                    lo = {0: 0, 1: n, 2: m}[klo]
                    hi = {0: K, 1: min(K, n + 1), 2: min(K, m + 1)}[khi]
                    want += 2 * max(0, hi - lo)
            assert gemm_alg_flop(M, N, K, klo, khi, out) == want, (M, N, K, klo, khi, out)


def test_noalloc_entry_point_rejects_oversize_without_gpu(lib):
    """bta_rows_times_block_noalloc checks its sizes against the built-in scratch before any CUDA call."""
    rc = lib.bta_rows_times_block_noalloc(9, 4224, 4096, ctypes.c_void_p(8), 4224, ctypes.c_void_p(8), 4096, 0,
                                          ctypes.c_double(1.0), ctypes.c_double(0.0), None, 0, ctypes.c_void_p(8), 4096,
                                          None)
    assert rc == 1 and b"BTA_NOALLOC_MAX_PART" in lib.bta_last_error()
