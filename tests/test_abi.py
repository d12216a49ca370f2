"""CPU-only checks of the C-ABI boundary: the library builds/loads without a GPU and exports
every function include/woden_b200.h declares; the Python binding names the same entry points;
argument errors are reported as status codes before any CUDA work."""
import ctypes as C
import os
import re

import pytest

from paper_2005_09316_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "woden_b200.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(woden_[a-z_0-9]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    assert os.path.exists(path)
    lib = C.CDLL(path)
    names = _declared()
    assert {"woden_create", "woden_destroy", "woden_predict_points", "woden_predict_gaussians",
            "woden_predict_shapelets", "woden_simulate_host", "woden_strerror"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in woden_b200.h but not exported"
    assert sorted(binding.EXPORTS) == names


def test_status_strings_and_constants_match_header():
    L = binding.load()
    src = open(HEADER).read()
    pipes = {}
    for name, val in re.findall(r"#define\s+(WODEN_[A-Z_0-9]+)\s+(-?\d+)", src):
        if name == "WODEN_PIPE_COUNT":
            assert len(binding.PIPES) == int(val)
        elif name.startswith("WODEN_PIPE_"):
            pipes[name[len("WODEN_PIPE_"):]] = int(val)
        else:
            assert getattr(binding, name) == int(val), name
    assert pipes == binding.PIPES          # every pattern bench.py uses is a documented id
    for code in (0, -1, -2, -3, -4, -5, -6, -7):
        assert L.woden_strerror(code).decode() not in ("", "unknown status")
    assert L.woden_strerror(-99).decode() == "unknown status"


def test_null_arguments_are_rejected_without_cuda():
    L = binding.load()
    assert L.woden_create(None, 0) == binding.WODEN_ERR_NULL
    assert L.woden_destroy(None) == binding.WODEN_ERR_NULL
    assert L.woden_check(None) == binding.WODEN_ERR_NULL
    assert L.woden_set_path(None, 0) == binding.WODEN_ERR_NULL
    assert L.woden_predict_points(None, None, 0, None, None, None, None, 1.0, None, 0, None) == binding.WODEN_ERR_NULL


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(binding.WodenError) as e:
        binding.Woden(0)
    assert e.value.status == binding.WODEN_ERR_CUDA


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2005_09316_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "woden_oracle" not in text, f
