"""CPU-only checks of the boundary: libdr.so builds, loads and exports every symbol include/dr.h declares;
without a CUDA device compute calls fail loudly (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libdr():
    from paper_2410_20441_b200 import build, binding
    build.build()
    return binding.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "dr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dr_[a-zA-Z_0-9]+)\s*\(", src)))


def test_header_symbols_are_all_exported(libdr):
    from paper_2410_20441_b200 import binding
    names = declared_symbols()
    assert len(names) >= 13
    for n in names:
        assert hasattr(libdr, n), n
    assert sorted(binding.EXPORTS) == names


def test_workspace_bytes_host_logic(libdr):
    from paper_2410_20441_b200 import binding
    assert binding.workspace_bytes(1, 8, 8) == 0 and binding.workspace_bytes(8, 8, 0) == 0
    b32 = binding.workspace_bytes(32, 32, 32)
    # 22 padded boxes of PX x 35 x 35 doubles (+ small scratch); PX = 17 + 34 rounded up to 64, +16 off the 512 B pitch
    # + tile-blocked uint8 phase ids: 2 x 3 tiles x 35 layers x 512 B
    # + stencil codes of the two-iteration kernel: 2 x 3 tiles (28 x 12 owned nodes of 32 x 16) x 37 layers x 512 x 8 B
    ids = 2 * 3 * 35 * 512 + 2 * 3 * 37 * 512 * 8
    assert 22 * 80 * 35 * 35 * 8 + ids <= b32 <= 22 * 80 * 35 * 35 * 8 + ids + 22 * 256 + 131072
    assert binding.workspace_bytes(703, 703, 703) < 72e9          # config 5 fits one B200 (180 GB)


def test_no_cpu_fallback(libdr):
    import torch
    from paper_2410_20441_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = C.c_void_p()
    buf = (C.c_double * 64)()
    st = libdr.dr_create(2, 2, 2, 1.0, C.cast(buf, C.c_void_p), C.cast(buf, C.c_void_p), None, 0, None, C.byref(h))
    assert st == binding.ERR_WORKSPACE and not h
    big = C.create_string_buffer(binding.workspace_bytes(2, 2, 2) + 512)
    addr = (C.addressof(big) + 255) & ~255
    st = libdr.dr_create(2, 2, 2, 1.0, C.cast(buf, C.c_void_p), C.cast(buf, C.c_void_p), C.c_void_p(addr),
                         binding.workspace_bytes(2, 2, 2), None, C.byref(h))
    assert st == binding.ERR_CUDA and not h
    with pytest.raises(RuntimeError):
        binding.Solver(torch.zeros(2, 2, 2, dtype=torch.float64), torch.zeros(2, 2, 2, dtype=torch.float64))


def test_null_handle_calls_return_err_arg(libdr):
    from paper_2410_20441_b200 import binding
    assert libdr.dr_set_param(None, 0, 0.5) == binding.ERR_ARG
    assert libdr.dr_solve(None, 0, 1e-4, 1e-8, 10) == binding.ERR_ARG
    assert libdr.dr_effective_C(None, None) == binding.ERR_ARG
    assert libdr.dr_last_error(None) == b"null handle"
    assert libdr.dr_launch_count(None) == 0
    libdr.dr_destroy(None)
