"""No-GPU checks of the boundary: the C-ABI library builds, loads and exports every symbol include/b200md.h declares;
the product path fails loudly (no CPU fallback) when there is no CUDA device."""
import os
import re

import pytest

from paper_1412_3387_b200 import binding as B
from paper_1412_3387_b200.csrc import build as csrc_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    txt = open(os.path.join(ROOT, "include", "b200md.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(md_[a-z_0-9]+)\s*\(", txt)))


def test_library_builds_and_exports_every_declared_symbol():
    csrc_build.build()
    L = B.load()
    names = _declared()
    assert "md_create" in names and "md_step" in names and len(names) >= 20
    for n in names:
        assert hasattr(L, n), f"{n} declared in b200md.h but not exported"
    assert sorted(B.EXPORTS) == names            # the binding mirrors the header 1:1


def test_struct_layouts_match_header():
    import ctypes as C
    L = B.load()                                      # (load() itself refuses a library whose struct sizes differ)
    for k, st in enumerate((B.md_step_desc, B.md_stats, B.md_thermo_t, B.md_pressure_t)):
        assert L.md_struct_size(k) == C.sizeof(st), st.__name__
    assert C.sizeof(B.md_step_desc) == 192 and C.sizeof(B.md_pressure_t) == 72 and L.md_struct_size(9) == -1


def test_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(B.MDError, match="no CUDA device"):
        B.MD([10.0, 10.0, 10.0], 100, 2.5, 0.4)


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1412_3387_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in s and "from oracle" not in s and "md_oracle" not in s, f
