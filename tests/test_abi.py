"""C-ABI boundary checks that need no GPU (`-m "not gpu"`): the shared library loads, exports
every symbol include/*.h declares, and its host-only entry points behave."""
import ctypes
import os
import re

import pytest

from paper_1807_10750_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    names = set()
    for header in sorted(os.listdir(os.path.join(ROOT, "include"))):
        if not header.endswith(".h"):
            continue
        src = open(os.path.join(ROOT, "include", header)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(ising_[a-z_]+)\s*\(", src))
    return sorted(names)


def test_library_builds_and_exports_every_declared_symbol():
    L = binding.lib()
    names = declared_symbols()
    assert {"ising_load_csr", "ising_anneal", "ising_energy_cut", "ising_best_state", "ising_free",
            "ising_workspace_bytes", "ising_status_string"} <= set(names)
    for name in names:
        assert hasattr(L, name), name
    assert os.path.exists(build.LIB)


def test_status_strings():
    L = binding.lib()
    seen = set()
    for code in range(0, 15):
        s = L.ising_status_string(code)
        assert s and s not in seen
        seen.add(s)
    assert L.ising_status_string(999) == b"unknown status"
    assert set(binding.STATUS_NAMES) == set(range(15))


def test_workspace_bytes_host_only():
    assert binding.ising_workspace_bytes(800, 38000, 4, 1, 19) > 800 * 32 * 3
    a = binding.ising_workspace_bytes(1000, 10000, 1, 32, 4)
    b = binding.ising_workspace_bytes(1000, 10000, 1, 64, 4)
    assert b > a
    with pytest.raises(binding.IsingError) as e:
        binding.ising_workspace_bytes(0, 0, 1, 1, 0)
    assert e.value.status == 2
    with pytest.raises(binding.IsingError) as e:
        binding.ising_workspace_bytes(10, 0, 1, 0, 0)
    assert e.value.status == 8
    with pytest.raises(binding.IsingError) as e:
        binding.ising_workspace_bytes(10, 0, 3, 1, 0)
    assert e.value.status == 2


def test_null_arguments_are_rejected_without_a_device():
    L = binding.lib()
    assert L.ising_workspace_bytes(10, 10, 1, 1, 0, None) == 1
    assert L.ising_anneal(None, 0, 0, 1, 0, 0, None, 0, 0, 0, None, None, None) == 1
    assert L.ising_energy_cut(None, None, 1, None, None, None) == 1
    assert L.ising_best_state(None, 0, None, None, None, None, None) == 1
    assert L.ising_free(None) == 0


def test_no_cpu_fallback_without_gpu():
    """On a machine without a B200 the product path must fail loudly, not fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import numpy as np
    rp = np.array([0, 1, 2], dtype=np.int64)
    col = np.array([1, 0], dtype=np.int32)
    w = np.array([1, 1], dtype=np.int8)
    with pytest.raises(RuntimeError):
        binding.ising_load_csr(rp, col, w)
    h = ctypes.c_void_p(0)
    buf = ctypes.create_string_buffer(1 << 16)
    st = binding.lib().ising_load_csr(2, 2, rp.ctypes.data, col.ctypes.data, w.ctypes.data, 1, None, 0, 1,
                                      ctypes.addressof(buf), 1 << 16, 0, None, ctypes.byref(h))
    assert st == 11   # ISING_ERR_UNSUPPORTED_DEVICE


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1807_10750_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".c")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
