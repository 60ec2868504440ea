"""CPU-side checks of the C-ABI boundary: the library builds and loads, exports every symbol
include/pca.h declares, and fails loudly (no CPU fallback) when there is no CUDA device.
No compute call is made here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "pca.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(pca_[a-z_0-9]+)\s*\(", src)
    return sorted(set(names))


def test_header_declares_the_north_star_entry_points():
    names = _declared_functions()
    for required in ("pca_create", "pca_center", "pca_run", "pca_destroy"):
        assert required in names


def test_library_exports_every_declared_symbol():
    from paper_0811_1081_b200 import binding
    lib = binding.load_library()
    names = _declared_functions()
    assert sorted(binding.EXPORTED_SYMBOLS) == names
    for n in names:
        assert getattr(lib, n) is not None


def test_header_compiles_as_plain_c(tmp_path):
    """include/pca.h is a C header: no C++ and no CUDA/torch types in the signatures."""
    import subprocess
    c = tmp_path / "t.c"
    c.write_text('#include "pca.h"\nint main(void){ pca_ctx* c = 0; (void)c; return PCA_OK; }\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
                    "-c", str(c), "-o", str(tmp_path / "t.o")], check=True)


def test_strerror_and_null_handling_need_no_device():
    from paper_0811_1081_b200 import binding
    lib = binding.load_library()
    for code in range(6):
        assert binding.pca_strerror(code)
    assert binding.pca_strerror(12345) == "unknown error"
    assert lib.pca_workspace_bytes(None) == 0
    assert lib.pca_last_cuda_error(None) == 0
    lib.pca_destroy(None)
    out = ctypes.c_void_p()
    assert lib.pca_create(ctypes.byref(out), 0, 0, 0, 0.0, 0, 0) == binding.PCA_EINVAL


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_0811_1081_b200 import binding
    with pytest.raises(binding.PcaError) as e:
        binding.PcaContext(64, 16, 2)
    assert e.value.code == binding.PCA_ECUDA


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_0811_1081_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "pca_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_0811_1081_b200\b", text, flags=re.M), f
            assert "cuda_runtime" not in text and "csrc" not in text.replace("paper_0811_1081_b200/csrc", ""), f
