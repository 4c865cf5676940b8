"""CPU-side checks of the C-ABI boundary: libvoila builds for sm_100a, loads, and exports every
symbol include/voila.h declares; without a GPU the product path fails loudly (no CPU fallback)."""
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "voila.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(voila_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_all_exported():
    import paper_2606_19729_b200 as vl
    lib = vl.load_library()
    declared = _declared_symbols()
    assert len(declared) >= 15
    assert sorted(vl.EXPORTS) == declared
    for name in declared:
        assert hasattr(lib, name), name
    assert lib.voila_version() >= 100
    assert lib.voila_status_string(0) == b"ok"


def test_library_is_sm100a_native_code():
    """The shared object carries sm_100a SASS (and nothing older)."""
    import paper_2606_19729_b200 as vl
    vl.load_library()
    out = subprocess.run(["cuobjdump", "-lelf", vl.lib_path()], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    archs = set(re.findall(r"sm_(\d+a?)", out.stdout))
    assert archs == {"100a"}, archs


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2606_19729_b200 as vl
    from paper_2606_19729_b200 import synth
    with pytest.raises(vl.VoilaError):
        vl.Voila(synth.make_model(synth.CONFIGS[1]))


def test_product_does_not_import_oracle():
    """The product package never references oracle/ (and the oracle never the product)."""
    pkg = os.path.join(ROOT, "paper_2606_19729_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "voila_oracle" not in src and "import oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2606_19729_b200 import" not in src and "libvoila.so" not in src, f
