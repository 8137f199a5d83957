"""CPU-side checks of the boundary: libsw_b200.so builds, loads and exports every symbol that
include/sw.h declares; argument validation that needs no device."""
import ctypes as C
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "sw.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sw_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_four_calls():
    syms = declared_symbols()
    for name in ("sw_create", "sw_step", "sw_observables", "sw_destroy"):
        assert name in syms


def test_library_exports_every_declared_symbol():
    from paper_1403_7560_b200 import binding
    lib = binding.lib()
    for name in declared_symbols():
        assert hasattr(lib, name), f"libsw_b200.so does not export {name}"


def test_workspace_bytes_and_validation_without_device():
    from paper_1403_7560_b200 import binding
    lib = binding.lib()
    # 3D L=512 Ising: spins N + bonds N + labels 4N + pair list 10N/4 + tile origins, accumulators
    n = 512 ** 3
    b = lib.sw_workspace_bytes(3, 512, binding.ISING, 0)
    assert 8 * n + n // 2 <= b <= 8 * n + n // 2 + n // 64
    assert lib.sw_workspace_bytes(3, 256, binding.XY, 0) >= 9 * 256 ** 3
    assert lib.sw_workspace_bytes(2, 48, binding.ISING, 0) == 0      # not a multiple of 32
    assert lib.sw_workspace_bytes(4, 64, binding.ISING, 0) == 0      # dim
    assert lib.sw_workspace_bytes(2, 64, binding.POTTS, 1) == 0      # q
    assert lib.sw_workspace_bytes(3, 2048, binding.ISING, 0) == 0    # N > 2^31
    assert lib.sw_workspace_bytes(3, 1024, binding.POTTS, 3) > 0     # 2^30 sites x 2 state bits
    assert lib.sw_workspace_bytes(3, 1024, binding.POTTS, 5) == 0    # 2^30 sites x 3 state bits > 2^32
    h = C.c_void_p()
    rc = lib.sw_create(C.byref(h), 2, 48, binding.ISING, 0, 0.4, 1)
    assert rc == binding.SW_EINVAL and not h
    assert b"invalid" in lib.sw_last_error()
    rc = lib.sw_create(C.byref(h), 2, 64, binding.ISING, 0, float("nan"), 1)
    assert rc == binding.SW_EINVAL and not h
    assert lib.sw_destroy(None) == binding.SW_OK
    assert lib.sw_step(None, 1) == binding.SW_EINVAL


def test_no_cpu_fallback_without_device():
    import torch
    from paper_1403_7560_b200 import binding
    if torch.cuda.is_available():
        return
    h = C.c_void_p()
    rc = binding.lib().sw_create(C.byref(h), 2, 64, binding.ISING, 0, 0.4, 1)
    assert rc == binding.SW_ECUDA and not h
    try:
        binding.SwendsenWang(2, 64, binding.ISING, 0, 0.4, 1)
    except binding.SwError as e:
        assert e.code == binding.SW_ECUDA
    else:
        raise AssertionError("a context was created without a CUDA device")
