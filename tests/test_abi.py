"""C-ABI library: loads, exports every symbol include/darwinopt.h declares, fails loudly without a GPU.
No compute calls here (-m "not gpu")."""
import ctypes as C
import re
from pathlib import Path

import pytest

from paper_2203_14354_b200 import binding

ROOT = Path(__file__).resolve().parent.parent


def declared_symbols():
    text = (ROOT / "include" / "darwinopt.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dw_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported():
    L = binding.load()
    syms = declared_symbols()
    assert set(syms) == set(binding.EXPORTS), (syms, binding.EXPORTS)
    for s in syms:
        assert hasattr(L, s), s
    assert L.dw_version() >= 100


def test_struct_layouts_match_header_sizes():
    # sizes implied by the header's field lists (LP64)
    assert C.sizeof(binding.Photons) == 8 + 8 + 11 * 8
    assert C.sizeof(binding.Results) == 14 * 8
    assert C.sizeof(binding.Hists) == 8 + 8 + 8 + 4 + 4 + 8 + 8 + 8
    assert C.sizeof(binding.PropagateParams) == 32
    assert C.sizeof(binding.BuildParams) == 32
    assert C.sizeof(binding.RefitStats) == 4 + 3 * 4 + 6 * 4 + 4
    assert C.sizeof(binding.BuildStats) == 4 * 8 + 2 * 4 + 6 * 4 + 4 + 6 * 4 + 4  # build_ms, ploc_rounds, binary_depth, grid_res, grid_free_cells, n_refs, split_div + tail padding to 8


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    L = binding.load()
    h = C.c_void_p()
    rc = L.dw_create(0, C.byref(h))
    assert rc == binding.DW_E_CUDA and not h.value
    assert b"no CPU fallback" in L.dw_last_error(None)
    with pytest.raises(binding.DwError):
        binding.Context(0)


def test_null_context_is_an_argument_error():
    L = binding.load()
    assert L.dw_set_materials(None, 1, 1, 175.0, 1.0, None, None, None) == binding.DW_E_ARG
    assert L.dw_propagate(None, None, 0, 0, None, None, None, None) == binding.DW_E_ARG
    assert L.dw_destroy(None) == binding.DW_OK


def test_product_path_does_not_import_the_oracle():
    for p in (ROOT / "paper_2203_14354_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h"):
            src = p.read_text()
            assert "import oracle" not in src and "from oracle" not in src and "liboracle" not in src, p


def test_no_indirect_branches_in_device_code():
    """profiles/r01_pool_hang.md: an indirect branch (jump table) inside the traversal loop left a warp split for good on
    sm_100a, and the schedulers take warp-wide decisions from votes.  The built library must contain none."""
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    lib = binding._LIB_PATH
    binding.load()
    sass = subprocess.run([cuobjdump, "-sass", str(lib)], capture_output=True, text=True, check=True).stdout
    assert "Function :" in sass, "no device code found in the library"
    bad = [ln.strip() for ln in sass.splitlines() if " BRX" in ln or " JMX" in ln or " BRXU" in ln or " JMXU" in ln]
    assert not bad, f"{len(bad)} indirect branches in device code, e.g. {bad[0]}"
