"""The C-ABI library builds, loads and exports every symbol include/pce.h declares (no compute: no GPU here)."""
import ctypes
import os
import re

import pytest

import paper_2401_04865_b200 as pce

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    pce.build()
    return pce.load()


def test_exports_match_header(lib):
    hdr = open(os.path.join(ROOT, "include", "pce.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pce_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(pce.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_suggest_params_follows_eqs_23_28_31_32(lib):
    import math
    p = pce.suggest_params([10.0] * 3, [32] * 3, 0.137952, 1e-10)
    s = math.sqrt(-math.log(1e-10))
    kc = math.pi * 31 / 10.0
    assert p.xi == pytest.approx(kc / (2 * s), rel=1e-14)          # eq. 28 with N_g = 1 + L k_c/pi
    assert p.rc == pytest.approx(s / p.xi + 2 * 0.137952, rel=1e-14)  # eq. 23 (+2a for shells)
    assert p.P == 20 and p.P % 2 == 0
    assert math.exp(-math.pi * p.P / 2) < 1e-10                    # eq. 32
    p2 = pce.suggest_params([10.0] * 3, [32] * 3, 0.1, 1e-12, P=24)
    assert p2.P == 24


def test_bench_restates_the_parameter_rule_of_the_library(lib):
    """bench.py's reference arm describes its configuration without loading libpce.so; its restatement of eqs. 23, 28, 32 must
    give what pce_suggest_params gives, on cubic and rectangular boxes, with and without a fixed P."""
    import bench
    for L, Ng, a, tol, P in (([10.0] * 3, [32] * 3, 0.137952, 1e-10, 0), ([20.0, 24.0, 31.0], [64, 80, 96], 0.05, 1e-6, 0),
                             ([40.0] * 3, [128] * 3, 0.0346, 1e-3, 0), ([108.0] * 3, [512] * 3, 0.0789, 1e-10, 18),
                             ([5.0] * 3, [16, 12, 16], 0.1, 1e-12, 0)):
        p = pce.suggest_params(L, Ng, a, tol, P)
        xi, rc, Pp = bench.ewald_params(L, Ng, a, tol, P)
        assert xi == pytest.approx(p.xi, rel=1e-15) and rc == pytest.approx(p.rc, rel=1e-15) and Pp == p.P == p.P_matvec


def test_reference_arm_of_the_bench_does_not_load_the_product_library():
    """`bench.py --impl reference` times the oracle; the product must not even be mapped into that process."""
    import subprocess
    import sys
    code = ("import sys, types; sys.argv=['bench.py','--impl','reference','--config','1'];"
            "import bench; a=bench.parse(); bench.config_dict(bench.make_workload(1), a);"
            "assert not any(m.startswith('paper_2401_04865_b200') for m in sys.modules), 'product imported';"
            "assert 'libpce' not in open('/proc/self/maps').read(), 'libpce.so mapped'")
    subprocess.check_call([sys.executable, "-c", code], cwd=ROOT)


def test_bad_arguments_are_rejected_without_a_gpu(lib):
    bad = pce.PceParams()
    h = ctypes.c_void_p()
    assert lib.pce_create(ctypes.byref(bad), None, ctypes.byref(h)) == -1  # PCE_EINVAL
    assert b"invalid" in lib.pce_last_error(None)
    with pytest.raises(pce.PceError):
        pce.suggest_params([10.0] * 3, [32] * 3, -1.0, 1e-10)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    p = pce.suggest_params([10.0] * 3, [32] * 3, 0.1, 1e-10)
    with pytest.raises(pce.PceError):
        pce.Context(p)
