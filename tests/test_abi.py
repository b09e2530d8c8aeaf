"""The C-ABI boundary (CPU only): libsw.so builds, loads, and exports every symbol include/sw.h declares.

No compute call is made here; on a box without a GPU, creating a context must fail loudly
(SW_ERR_CUDA), never fall back to a CPU path.
"""
import ctypes as C
import os
import re

import pytest

from paper_1208_2080_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libsw():
    build.build()
    return binding.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "sw.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sw_[a-z_]+)\s*\(", text)))


def test_header_and_binding_agree():
    assert declared_symbols() == sorted(binding.SYMBOLS)


def test_library_exports_every_declared_symbol(libsw):
    raw = C.CDLL(binding.LIB_PATH)
    for name in declared_symbols():
        assert hasattr(raw, name), name
    assert b"sm_100a" in libsw.sw_version()


def test_library_is_built_for_sm_100a():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump not available")
    assert "sm_100a" in out.stdout


def test_workspace_plan_no_device_needed(libsw):
    assert binding.workspace_bytes(1, 2) == 0 and binding.workspace_bytes(64, 1) == 0
    assert binding.workspace_bytes(70000, 2) == 0
    for L, q in ((2, 2), (3, 3), (64, 2), (256, 10), (4096, 2)):
        n = binding.workspace_bytes(L, q)
        N = L * L
        assert n >= N + N // 4 + 4 * N                       # spins + bond bits + labels
        # + tile-root bitmap, border / edge records, border table of the cluster-size count (0.25 B/site), draw bits, cluster
        # counts, and the context-owned scratch: the row ring of sw_sweep_measure (<= 256 KiB), the staging buffer of
        # sw_get_bonds (min(N, 32 MiB)), pass counters
        assert n <= 7.25 * N + 8192 + (256 << 10)
        assert binding.workspace_bytes(L, q, binding.FLAG_WS_CLUSTER_SIZES) >= n + 4 * N      # the optional cluster-size scratch
    # headline size: 2^32 sites must fit one B200 with room to spare (180 GB)
    n = binding.workspace_bytes(65536, 2)
    assert 21 * 2 ** 30 <= n <= 25 * 2 ** 30


def test_null_and_invalid_arguments_do_not_crash(libsw):
    assert libsw.sw_create(None, 4, 2, 0.5, 1) == binding.ERR_INVALID_ARG
    h = C.c_void_p()
    for L, q, K in ((1, 2, 0.5), (4, 1, 0.5), (4, 256, 0.5), (4, 2, -1.0), (4, 2, float("nan")), (65537, 2, 0.5)):
        assert libsw.sw_create(C.byref(h), L, q, K, 1) == binding.ERR_INVALID_ARG
        assert not h
    assert libsw.sw_sweep(None, 1) == binding.ERR_INVALID_ARG
    assert libsw.sw_init(None, 0) == binding.ERR_INVALID_ARG
    libsw.sw_destroy(None)


def test_no_cpu_fallback_without_a_gpu(libsw):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    assert libsw.sw_create(C.byref(h), 64, 2, 0.5, 1) in (binding.ERR_CUDA, binding.ERR_OOM)
    assert not h
    with pytest.raises(binding.SwError):
        binding.SwendsenWang(64, 2, 0.5, 1)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1208_2080_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "sw_oracle" not in text and "from oracle" not in text and "import oracle" not in text, f
