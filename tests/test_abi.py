"""The C-ABI boundary (include/gene_nl.h): the library builds, loads and exports every declared symbol.
No compute calls here (no GPU on the CPU box)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions(header="gene_nl.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gene_nlx?_\w+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for n in ("gene_nl_create", "gene_nl_compute", "gene_nl_destroy",
              "gene_nlx_create", "gene_nlx_compute", "gene_nlx_destroy"):   # x-global variant
        assert n in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1310_1485_b200 import binding
    lib = binding.load_library()
    assert os.path.dirname(binding.library_path()) == os.path.join(ROOT, "paper_1310_1485_b200")
    names = declared_functions()
    assert sorted(binding.EXPORTED_SYMBOLS) == names
    bench_names = declared_functions("gene_nl_bench.h")          # benchmark-only helpers, in a header of their own
    assert sorted(binding.BENCH_SYMBOLS) == bench_names and not set(bench_names) & set(names)
    names = names + bench_names
    for n in names:
        assert hasattr(lib, n), n
    raw = ctypes.CDLL(binding.library_path())
    for n in names:
        getattr(raw, n)


def test_binding_exposes_the_same_names():
    import paper_1310_1485_b200 as pkg
    for n in declared_functions():
        assert callable(getattr(pkg, n))


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1310_1485_b200 import GeneNLError, gene_nl_create
    with pytest.raises(GeneNLError):
        gene_nl_create(16, 8, 1, 1, 1, 1, 0.1, 0.1, 0)
    from paper_1310_1485_b200 import gene_nlx_create
    with pytest.raises(GeneNLError):
        gene_nlx_create(64, 16, 1)


def test_no_environment_knobs_in_the_product_path():
    """SURVEY.md sect. 5: configuration comes through gene_nl_create arguments only (no env flags)."""
    pkg = os.path.join(ROOT, "paper_1310_1485_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "getenv" not in text, f
                if f != "build.py":   # build.py may honour NVCC (the compiler's location), nothing else
                    assert "os.environ" not in text, f


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1310_1485_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "oracle/" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1310_1485_b200" not in text and "from paper_1310_1485_b200" not in text, f
