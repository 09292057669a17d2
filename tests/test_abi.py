"""The C-ABI library builds, loads and exports every symbol include/phi4smc.h declares; host-side
argument checks; the binding refuses to run without a CUDA device (no CPU fallback) -- CPU only."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2511_15196_b200 import build, binding
    build.build()
    return binding.load()


def header_functions():
    src = open(os.path.join(ROOT, "include", "phi4smc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^\s*(?:const\s+char\s*\*|size_t|int|double|uint64_t)\s+(\w+)\s*\(", src, flags=re.M)
    return sorted(set(names))


def test_header_symbols_are_exported_and_bound(lib):
    from paper_2511_15196_b200 import binding
    names = header_functions()
    assert len(names) >= 24 and "smc_step" in names and "ns_step" in names and "log_Z" in names
    for n in names:
        assert hasattr(lib, n), n
        assert n in binding.SIGNATURES, n
    assert sorted(binding.SIGNATURES) == names


def test_struct_sizes_match_header(lib):
    from paper_2511_15196_b200 import binding as B
    assert C.sizeof(B.smc_params) == 32
    assert C.sizeof(B.smc_step_info) == 6 * 8 + 4 * 4
    assert C.sizeof(B.ns_step_info) == 56   # 5 doubles + 3 ints, padded to 8
    assert C.sizeof(B.phi4_observables) == (5 + 80) * 8
    assert C.sizeof(B.phi4_run_state) == 6 * 8 + 2 * 4 + 8


def test_workspace_sizes(lib):
    from paper_2511_15196_b200 import binding as B
    assert B.smc_workspace_bytes(0, 100) == 0 and B.smc_workspace_bytes(4, 1) == 0
    a, b = B.smc_workspace_bytes(4, 1024), B.smc_workspace_bytes(10, 16384)
    assert 0 < a < b
    # C4: 2 GB of state, double-buffered, plus proposal scratch and two buffers of split normals
    # (4.3 GB each): < 16 GB of 180 GB
    assert 8.5e9 < B.smc_workspace_bytes(64, 131072) < 16e9
    assert B.ns_workspace_bytes(10, 4096, 4096, 10) == 0
    assert B.ns_workspace_bytes(10, 4096, 512, 2048) > 0


def test_strerror_and_null_handles(lib):
    assert lib.phi4_strerror(0) == b"ok"
    assert b"positive definite" in lib.phi4_strerror(-3)
    assert lib.smc_step(None, None) == -1
    assert lib.ns_step(None, None) == -1
    assert lib.smc_destroy(None) == 0
    assert lib.observables(None, None) == -1
    import math
    assert math.isnan(lib.log_Z(None))


def test_init_argument_checks_and_no_cpu_fallback(lib):
    import torch
    from paper_2511_15196_b200 import binding as B
    ptr = C.c_void_p()
    need = B.smc_workspace_bytes(4, 1024)
    fake = C.c_void_p(1 << 20)                      # aligned, never dereferenced on the host
    assert lib.smc_init(C.byref(ptr), 4, -4.0, 1.0, 1024, 0, fake, need - 1, None) == -1
    assert lib.smc_init(C.byref(ptr), 4, -4.0, 1.0, 1024, 0, C.c_void_p((1 << 20) + 4), need, None) == -1
    assert lib.smc_init(C.byref(ptr), 4, -4.0, 1.0, 1024, 0, None, need, None) == -1
    assert lib.ns_init(C.byref(ptr), 4, -4.0, 1.0, (1 << 20) + 1, 10, 5, 0, 1e-3, 10, fake, 1 << 40, None) == -1
    if not torch.cuda.is_available():
        assert lib.smc_init(C.byref(ptr), 4, -4.0, 1.0, 1024, 0, fake, need, None) == -5   # PHI4_ECUDA
        with pytest.raises(RuntimeError, match="no CPU fallback"):
            B.smc_init(4, -4.0, 1.0, 1024, 0)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2511_15196_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("a CPU\noracle", "").replace("CPU oracle", ""), f
