"""The C-ABI library loads and exports every symbol include/*.h declares (no compute without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1206_1779_b200 import build, binding
    build.build()
    return binding.load_library()


def test_header_symbols_exported(lib):
    names = set()
    for h in ("dse.h", "dse_diag.h"):
        hdr = open(os.path.join(ROOT, "include", h)).read()
        hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
        names |= set(re.findall(r"\b(dse_[a-z0-9_]+)\s*\(", hdr))
    assert {"dse_create", "dse_create_with_tables", "dse_destroy", "dse_residual", "dse_jacobian", "dse_newton_step"} <= names
    for n in names:
        assert hasattr(lib, n), n
    from paper_1206_1779_b200.binding import EXPORTS
    assert set(EXPORTS) == names


def test_struct_layout_matches_header():
    from paper_1206_1779_b200.binding import DseParams
    # 4 int32 + 10 double + 2 int32
    assert ctypes.sizeof(DseParams) == 16 + 80 + 8
    assert DseParams.eps2.offset == 16 and DseParams.flags.offset == 96


def test_error_paths_without_gpu(lib):
    from paper_1206_1779_b200.binding import DseParams
    from workloads import CONFIGS
    from paper_1206_1779_b200 import params_from_workload
    h = ctypes.c_void_p()
    assert lib.dse_strerror(0) == b"ok" and lib.dse_strerror(-1) == b"invalid argument"
    assert lib.dse_create(None, ctypes.byref(h)) == -1
    bad = params_from_workload(CONFIGS[0])
    bad.n_cheb = 1
    assert lib.dse_create(ctypes.byref(bad), ctypes.byref(h)) == -1
    bad = params_from_workload(CONFIGS[0])
    bad.eps2 = 2e10
    assert lib.dse_create(ctypes.byref(bad), ctypes.byref(h)) == -1
    bad = params_from_workload(CONFIGS[0])
    bad.x_G = -1.0
    assert lib.dse_create(ctypes.byref(bad), ctypes.byref(h)) == -1
    bad = params_from_workload(CONFIGS[0])
    bad.n_r_ir = -3
    assert lib.dse_create(ctypes.byref(bad), ctypes.byref(h)) == -1
    # caller-supplied tables: the flag and the entry point go together
    ok = params_from_workload(CONFIGS[0])
    ok.flags = 8
    assert lib.dse_create(ctypes.byref(ok), ctypes.byref(h)) == -1
    assert lib.dse_create_with_tables(ctypes.byref(ok), None, ctypes.byref(h)) == -1
    ok.flags = 1 << 12                                                     # unknown flag bit
    assert lib.dse_create(ctypes.byref(ok), ctypes.byref(h)) == -1
    assert lib.dse_strerror(-4) == b"constant-bank coefficient slot is held by another handle"
    assert lib.dse_destroy(None) == 0
    assert lib.dse_jacobian(None, None, None, None, None, None) == -1
    import torch
    if not torch.cuda.is_available():
        ok = params_from_workload(CONFIGS[0])
        assert lib.dse_create(ctypes.byref(ok), ctypes.byref(h)) == -3      # no CPU fallback
        from paper_1206_1779_b200 import Dse, DseError
        with pytest.raises(DseError):
            Dse(ok)


def test_no_environment_switches_in_the_library():
    """one POD struct, no env vars -- nothing under csrc/ reads the environment."""
    src = os.path.join(ROOT, "paper_1206_1779_b200", "csrc")
    for f in os.listdir(src):
        if f.endswith((".cu", ".cuh", ".cpp", ".h")):
            assert "getenv" not in open(os.path.join(src, f)).read(), f


def test_phase_stamps_need_an_instrumented_build(lib):
    """include/dse_diag.h: the phase stamps exist only in a library built with -DDSE_PHASE_TIMING; the library the repository
    builds by default (and ships to the GPU box) is the plain one, and says so."""
    import numpy as np
    out = np.zeros(16, dtype=np.int64)
    lib.dse_diag_phase_stamps.argtypes = [ctypes.c_int32, ctypes.c_void_p, ctypes.c_int32]
    assert lib.dse_diag_phase_stamps(0, ctypes.c_void_p(out.ctypes.data), 16) == -1
    assert b"DSE_PHASE_TIMING" in lib.dse_last_error()
    assert lib.dse_diag_phase_stamps(2, ctypes.c_void_p(out.ctypes.data), 16) == -1          # unknown selector
