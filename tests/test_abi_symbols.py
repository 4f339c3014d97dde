"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol include/gpusparse.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2606_26441_b200 import build
    return build.build_cuda()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "gpusparse.h")).read()
    return re.findall(r"^GS_API\s+[\w\s\*]+?\b(gs_\w+)\s*\(", src, flags=re.M)


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for must in ("gs_index_build", "gs_search", "gs_search_host", "gs_index_free", "gs_topk_dense", "gs_score_dense"):
        assert must in names
    assert len(names) == len(set(names)) >= 15


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    for name in declared_symbols():
        assert hasattr(L, name), f"{name} declared in gpusparse.h but not exported"
    from paper_2606_26441_b200 import binding
    assert sorted(binding.EXPORTS) == sorted(declared_symbols())
    binding.lib()
    assert "sm_100a" in binding.version()
    L.gs_abi_version.restype = ctypes.c_int32
    assert L.gs_abi_version() == 5


def test_host_checked_arguments_without_gpu(libpath):
    """No compute: only host-side argument checks (these return before any CUDA call)."""
    from paper_2606_26441_b200 import binding as B
    L = B.lib()
    h = ctypes.c_void_p()
    assert L.gs_index_build(None, 0, None, None, None, ctypes.byref(h)) == 1          # vocab <= 0
    assert L.gs_index_build(None, 8, None, None, None, None) == 1                     # out == NULL
    need = ctypes.c_size_t()
    assert L.gs_topk_workspace_bytes(4, 100, 0, ctypes.byref(need)) == 2               # k < 1
    assert L.gs_topk_workspace_bytes(4, 100, B.GS_MAX_K + 1, ctypes.byref(need)) == 2  # k too large
    assert L.gs_topk_workspace_bytes(4, 100, 10, ctypes.byref(need)) == 0 and need.value > 0
    assert L.gs_strerror(7).decode().startswith("unsupported device")


def test_only_sm100a_code_in_the_library(libpath):
    import subprocess
    out = subprocess.run(["cuobjdump", "--list-elf", libpath], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs
