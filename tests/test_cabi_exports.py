"""The C-ABI boundary (`-m "not gpu"`): the library builds for sm_100a without a GPU, loads, and exports every
symbol include/crownb200.h declares; the Python binding binds exactly those names; struct layouts agree with the
header; the product path fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "crownb200.h")


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^\s*(?:const\s+char\s*\*|int)\s+(\w+)\s*\(", src, flags=re.M)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_09377_b200 import build
    build.build()                                    # nvcc cross-compiles; no GPU needed
    from paper_2606_09377_b200 import binding
    return binding.load_library()


def test_header_declares_the_four_calls_of_the_boundary():
    names = _declared_functions()
    for n in ("crown_init", "ibp_forward", "crown_backward", "concretize", "crown_run", "crown_run_host",
              "crown_workspace_bytes", "crown_destroy", "crown_last_error"):
        assert n in names


def test_library_exports_every_declared_symbol(lib):
    for n in _declared_functions():
        assert hasattr(lib, n), f"{n} is declared in crownb200.h but not exported"


def test_binding_binds_exactly_the_declared_symbols():
    from paper_2606_09377_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_functions()


def test_struct_layouts_match_the_header():
    from paper_2606_09377_b200 import binding
    # crown_node: 13 int32 + 3 pointers; crown_opts: u64, 4 x i32, u64, u64, 4 x i32
    assert ctypes.sizeof(binding.CrownNode) == 13 * 4 + 4 + 3 * 8
    assert ctypes.sizeof(binding.CrownOpts) == 8 + 4 * 4 + 8 + 8 + 4 * 4      # ..., disable_epi_fusion, disable_conc_fusion, disable_graph, reserved
    assert binding.CrownOpts.stream_min_elems.offset == 24 and binding.CrownOpts.disable_epi_fusion.offset == 40


def test_version_and_error_paths_without_compute(lib):
    assert b"sm_100a" in lib.crown_version()
    assert lib.crown_destroy(None) != 0                       # CROWN_EINVAL, no crash
    assert lib.crown_last_error(None) == b"null context"
    out = ctypes.c_size_t(0)
    assert lib.crown_workspace_bytes(None, 0, 1, 1, 1, 1, 1, None, ctypes.byref(out)) != 0


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import workloads as W
    from paper_2606_09377_b200 import CrownContext, CrownError
    with pytest.raises(CrownError):
        CrownContext(W.small_mlp([4, 4, 2], 0).net, 1, 1)
