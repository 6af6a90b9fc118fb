"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every
symbol include/qmcd.h declares, and its host-only calls validate arguments.  No compute calls."""
import ctypes
import os
import re

import pytest

from paper_1708_00744_b200 import binding, buildlib

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    buildlib.build()
    return binding.load()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "qmcd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(qmcd_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_all_exported_and_bound(lib):
    names = _declared_symbols()
    assert "qmcd_create" in names and "qmcd_flush" in names and "qmcd_ratio" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in qmcd.h but not exported"
        assert n in binding.SYMBOLS, f"{n} has no binding"
    assert sorted(binding.SYMBOLS) == names


def test_invert_scratch_bytes_validation(lib):
    assert lib.qmcd_invert_scratch_bytes(512, 16) >= 16 * 512 * 4
    assert lib.qmcd_invert_scratch_bytes(0, 1) == 0
    assert lib.qmcd_invert_scratch_bytes(8, 0) == 0
    assert lib.qmcd_invert_scratch_bytes(20000, 1) == 0     # two rows + the gather no longer fit in shared memory


def test_invert_static_host_side(lib):
    assert lib.qmcd_invert_static_max_bytes() == 1 << 20
    assert lib.qmcd_invert_static(None, None, None, None) == binding.EINVAL
    assert b"limit" in lib.qmcd_strerror(binding.ELIMIT)
    # every BASELINE.json shape fits the static array
    for N, batch in [(64, 1), (512, 16), (1024, 64), (2048, 32), (4096, 8)]:
        assert 0 < lib.qmcd_invert_scratch_bytes(N, batch) <= lib.qmcd_invert_static_max_bytes()


def test_workspace_bytes_validation(lib):
    assert lib.qmcd_workspace_bytes(64, 4, 1) > 2 * 4 * 64 * 8
    assert lib.qmcd_workspace_bytes(0, 1, 1) == 0
    assert lib.qmcd_workspace_bytes(8, 0, 1) == 0
    assert lib.qmcd_workspace_bytes(8, 9, 1) == 0          # K > N (reading G16)
    assert lib.qmcd_workspace_bytes(8, 8, 0) == 0
    assert lib.qmcd_workspace_bytes(8192, 4096, 1) == 0    # K <= 4095: the job descriptor holds m in 12 bits
    # K x N buffers per walker dominate: C, W and Y = M W (one per walker)
    big = lib.qmcd_workspace_bytes(4096, 256, 8)
    assert 3 * 8 * 256 * 4096 * 8 <= big < 3 * 8 * 256 * 4096 * 8 + (8 << 20)


def test_strerror_and_version(lib):
    assert lib.qmcd_strerror(0) == b"ok"
    assert b"state" in lib.qmcd_strerror(binding.ESTATE)
    assert b"invalid" in lib.qmcd_strerror(binding.EINVAL)
    assert b"sm_100a" in lib.qmcd_version()


def test_create_rejects_bad_arguments_without_touching_a_device(lib):
    h = ctypes.c_void_p()
    assert lib.qmcd_create(ctypes.byref(h), 8, 9, 1, 256, 1 << 20, None) == binding.EINVAL
    assert lib.qmcd_create(ctypes.byref(h), 8, 2, 1, None, 1 << 20, None) == binding.EINVAL
    assert lib.qmcd_create(ctypes.byref(h), 8, 2, 1, 256, 16, None) == binding.EINVAL      # too small
    assert lib.qmcd_create(ctypes.byref(h), 8, 2, 1, 264, 1 << 20, None) == binding.EINVAL  # misaligned
    assert lib.qmcd_create(None, 8, 2, 1, 256, 1 << 20, None) == binding.EINVAL
    assert not h.value


def test_null_handle_calls_are_errors(lib):
    assert lib.qmcd_destroy(None) == 0
    assert lib.qmcd_flush(None) == binding.EINVAL
    assert lib.qmcd_reject(None) == binding.EINVAL
    assert lib.qmcd_accept(None, None) == binding.EINVAL
    assert lib.qmcd_sweep_host_min_staging(0, 1) == 0
    assert lib.qmcd_sweep_host_min_staging(512, 16) >= 2 * 16 * 512 * 8


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        binding.Qmcd(8, 2, 1)


def test_product_path_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1708_00744_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "qmcd_oracle" not in txt, f
