"""CPU-only checks of the boundary: libgs.so loads and exports every symbol include/gs.h declares; the binding lists
the same names; the product path raises (no fallback) when no CUDA device is present."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "gs.h")).read()
    return sorted(set(re.findall(r"GS_API\s+(?:const\s+)?\w+\*?\s+(gs_\w+)\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_2605_10760_b200 import build, binding
    lib_path = build.build()
    lib = ctypes.CDLL(lib_path)
    names = _declared()
    assert len(names) >= 15 and {"gs_preprocess", "gs_bin_tiles", "gs_rasterize_fwd", "gs_rasterize_bwd",
                                 "gs_pose_grad"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names


def test_binding_has_the_five_calls_and_no_cpu_fallback():
    import torch
    from paper_2605_10760_b200 import binding
    for n in ("gs_preprocess", "gs_bin_tiles", "gs_rasterize_fwd", "gs_rasterize_bwd", "gs_pose_grad"):
        assert callable(getattr(binding.Context, n))
    if not torch.cuda.is_available():
        with pytest.raises(RuntimeError, match="no CPU fallback"):
            binding.Context(0)


def test_product_code_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2605_10760_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "gso" not in txt and "libgs_oracle" not in txt, f
                for line in txt.splitlines():
                    if line.lstrip().startswith(("import ", "from ", "#include")):
                        assert "oracle" not in line, (f, line)
