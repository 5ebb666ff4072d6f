"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/mlp.h
declares; compute entry points fail loudly without a GPU (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    txt = open(os.path.join(ROOT, "include", "mlp.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(mlp_[a-z_]+)\s*\(", txt)))


def test_library_builds_and_exports_every_declared_symbol():
    import paper_2506_04055_b200 as P
    lib = P.load_library()
    names = _declared()
    assert set(names) == set(P.EXPORTED_SYMBOLS), (names, P.EXPORTED_SYMBOLS)
    raw = ctypes.CDLL(P.lib_path())
    for n in names:
        assert hasattr(raw, n), n
    assert b"sm_100a" in lib.mlp_version()


def test_no_cpu_fallback():
    import torch
    import gen
    import paper_2506_04055_b200 as P
    if torch.cuda.is_available():
        pytest.skip("GPU present: covered by the -m gpu tests")
    blob = gen.make_weights(2, 32, 16, 2, 5.0, seed=1)
    with pytest.raises(P.MLPError) as ei:
        P.Model(blob, 2, 5.0, 100)
    assert ei.value.code == 6        # MLP_ERR_CUDA


def test_product_path_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2506_04055_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert "oracle" not in src.replace("no oracle", ""), os.path.join(dp, f)
