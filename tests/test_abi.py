"""CPU-only checks of the boundary: libtacg.so builds/loads, exports every symbol that
include/tacg.h declares, and fails loudly (no CPU fallback) without an sm_100 device."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tacg():
    from paper_2606_01007_b200 import build
    build.build()
    import paper_2606_01007_b200 as t
    return t


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "tacg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b((?:tacg|gesr)_[a-z_]+)\s*\(", src)
    return sorted(set(names))


def test_header_symbols_are_exported(tacg):
    lib = tacg.lib()
    declared = _declared_symbols()
    assert "tacg_coact_accumulate" in declared and "gesr_select" in declared
    assert "tacg_affinity_swapgain" in declared and "tacg_eval_placement" in declared
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in tacg.h but not exported"
    assert sorted(tacg.EXPORTS) == declared


def test_strerror_and_version(tacg):
    lib = tacg.lib()
    assert lib.tacg_strerror(0) == b"ok"
    for code in range(-6, 0):
        assert len(lib.tacg_strerror(code)) > 3
    assert re.match(r"^\d+\.\d+$", tacg.version())


def test_no_cpu_fallback(tacg):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(tacg.TacgError) as ei:
        tacg.Context(0)
    assert ei.value.code == -6          # TACG_ERR_ARCH: no device, and nothing else to run on
    with pytest.raises(ValueError):
        tacg.binding._ptr(torch.zeros(4, dtype=torch.int16), torch.int16, "indices")   # CPU tensors are refused


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_01007_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in text and "from oracle" not in text, fn
                assert "tacg_oracle" not in text, fn
