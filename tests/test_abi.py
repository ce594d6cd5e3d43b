"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol include/ris.h declares,
and the binding fails loudly (no CPU fallback) when no CUDA device is present."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    names = set()
    for header in ("ris.h", "ris_bench.h"):      # the product boundary + the measurement / diagnostic entry points
        text = open(os.path.join(ROOT, "include", header)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names |= set(re.findall(r"\b(ris_[a-zA-Z0-9_]+)\s*\(", text))
    return sorted(names)


@pytest.fixture(scope="module")
def lib():
    from paper_2511_18233_b200 import build, ris
    build.build()
    return ris.load_library()


def test_library_exports_every_declared_symbol(lib):
    names = _declared_symbols()
    assert {"ris_setup", "ris_grad_J", "ris_grad_K", "ris_grad_PQ", "ris_destroy", "ris_strerror"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_binding_lists_the_same_symbols():
    from paper_2511_18233_b200 import ris
    assert sorted(ris.EXPORTS) == _declared_symbols()


def test_strerror_without_gpu(lib):
    assert lib.ris_strerror(0) == b"success"
    assert lib.ris_strerror(-1) == b"invalid argument"


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2511_18233_b200 import RisError, ris_setup, synth
    with pytest.raises(RisError):
        ris_setup(synth.make_molecule(1)[0])


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2511_18233_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|ris_oracle|libris_oracle", text, flags=re.M), \
                    os.path.join(dirpath, f)
