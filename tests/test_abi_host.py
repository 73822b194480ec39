"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol that
include/sap_dpsr.h declares, and validates arguments before touching CUDA."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def lib():
    from paper_2106_03452_b200 import build, binding
    build.build()
    return binding.lib()


def declared_symbols():
    text = (ROOT / "include" / "sap_dpsr.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sap_dpsr_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    from paper_2106_03452_b200 import binding
    names = declared_symbols()
    assert len(names) >= 10
    for n in names:
        assert hasattr(lib, n), f"{n} declared in sap_dpsr.h but not exported"
    assert sorted(binding.EXPORTS) == names


def test_mesh_header_symbols_are_exported_and_table_matches_the_oracle(lib):
    from paper_2106_03452_b200 import mesh
    text = (ROOT / "include" / "sap_mesh.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = sorted(set(re.findall(r"\b(sap_(?:mesh|mc|chamfer|points)[a-z_]*)\s*\(", text)))
    assert len(names) >= 8 and sorted(mesh.EXPORTS) == names
    L = mesh.lib()
    for n in names:
        assert hasattr(L, n), f"{n} declared in sap_mesh.h but not exported"
    assert L.sap_mesh_create(16, 10, 10, 10, None) == 1
    assert L.sap_mesh_create(0, 10, 10, 10, ctypes.byref(ctypes.c_void_p())) == 1
    assert L.sap_mesh_create(24, 10, 10, 10, ctypes.byref(ctypes.c_void_p())) == 2      # not a power of two
    assert L.sap_mc_extract(None, None, None, None, None, None, None) == 1
    assert L.sap_chamfer(None, None, 0, None, None, 0, None, None, None, None, None) == 1
    # the cube triangulation is built by the same RULE (reading M3) in two independent implementations: the library's
    # (host C++, csrc/sap_mesh.cu) and the oracle's (C, oracle/mesh_oracle.c); no table is shared or copied
    import numpy as np
    from oracle import mesh_oracle as mo
    a, b = mesh.mc_table(), mo.mc_table()
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_create_validates_arguments_before_cuda(lib):
    h = ctypes.c_void_p()
    out = ctypes.byref(h)
    assert lib.sap_dpsr_create(128, 2.0, 1, 100, None) == 1           # null out
    assert lib.sap_dpsr_create(0, 2.0, 1, 100, out) == 1
    assert lib.sap_dpsr_create(128, 2.0, 0, 100, out) == 1
    assert lib.sap_dpsr_create(128, 2.0, 1, 0, out) == 1
    assert lib.sap_dpsr_create(128, -1.0, 1, 100, out) == 1
    assert lib.sap_dpsr_create(128, float("nan"), 1, 100, out) == 1
    assert lib.sap_dpsr_create(128, float("inf"), 1, 100, out) == 1
    assert lib.sap_dpsr_create(100, 2.0, 1, 100, out) == 2            # not a supported resolution
    assert lib.sap_dpsr_create(1024, 2.0, 1, 100, out) == 2
    assert lib.sap_dpsr_create(16, 2.0, 1, 100, out) == 2
    assert not h.value
    assert b"N must be one of" in lib.sap_dpsr_last_error(None)


def test_null_handle_is_rejected(lib):
    assert lib.sap_dpsr_forward(None, None, None, 1, None, None) == 1
    assert lib.sap_dpsr_backward(None, None, None, 1, None, None, None, None, None) == 1
    assert lib.sap_dpsr_forward_mse(None, None, None, 1, None, None, None, None) == 1
    assert lib.sap_dpsr_backward_mse(None, None, None, 1, None, None, None, None) == 1
    assert lib.sap_dpsr_forward_host(None, None, None, 1, None, None) == 1
    assert lib.sap_dpsr_backward_host(None, None, None, None, None) == 1
    assert lib.sap_dpsr_get_stats(None, None, None) == 1
    assert lib.sap_dpsr_set_profiling(None, 1) == 1
    assert lib.sap_dpsr_workspace_bytes(None) == 0
    assert lib.sap_dpsr_last_launch_count(None) == 0
    lib.sap_dpsr_destroy(None)


def test_no_gpu_is_an_error_not_a_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = ctypes.c_void_p()
    st = lib.sap_dpsr_create(32, 2.0, 1, 100, ctypes.byref(h))
    assert st in (2, 4) and not h.value
    from paper_2106_03452_b200.binding import Dpsr, SapError
    with pytest.raises(SapError):
        Dpsr(32, 2.0, 1, 100)


def test_product_does_not_import_the_oracle():
    pat = re.compile(r"import\s+oracle|from\s+oracle|dpsr_oracle|libdpsr_oracle")
    pat = re.compile(r"import\s+oracle|from\s+oracle|dpsr_oracle|mesh_oracle|libdpsr_oracle|libmesh_oracle")
    for p in list((ROOT / "paper_2106_03452_b200").rglob("*")) + list((ROOT / "include").rglob("*")):
        if p.suffix in (".py", ".cu", ".cuh", ".h"):
            text = p.read_text()
            if p.name == "sap_mesh.h":      # the header names the oracle file in its documentation of the readings
                text = text.replace("oracle/mesh_oracle.c", "")
            assert not pat.search(text), p
