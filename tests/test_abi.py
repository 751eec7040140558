"""CPU-side checks of the boundary: the shared library loads, exports every symbol that
include/mlip.h declares, refuses to run without a GPU (no CPU fallback), and the header size
formula matches the input generator."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "mlip.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mlip_[a-z_]+)\s*\(", text)))


def _lib():
    import paper_2509_21694_b200 as mlip
    from paper_2509_21694_b200 import build
    build.build()
    return mlip, mlip.load_library()


def test_library_exports_every_declared_symbol():
    mlip, lib = _lib()
    syms = _declared_symbols()
    assert len(syms) >= 18
    for name in syms:
        assert hasattr(lib, name), name


def test_weight_count_matches_generator():
    mlip, lib = _lib()
    from paper_2509_21694_b200.binding import make_header
    from synth_inputs import ModelSpec
    import ctypes as C
    for d, k, L, S in [(64, 8, 2, 4), (256, 16, 15, 4), (128, 16, 4, 2)]:
        spec = ModelSpec(S, d, k, L, 5.0, 0.1)
        h = make_header(S, d, k, L, 5.0, 0.1)
        assert lib.mlip_model_num_weights(C.byref(h)) == spec.n_weights()


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    mlip, lib = _lib()
    with pytest.raises(mlip.MlipError):
        mlip.Context(0)
    import ctypes as C
    h = C.c_void_p()
    assert lib.mlip_ctx_create(0, None, C.byref(h)) == -6 and not h.value


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2509_21694_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert "oracle" not in open(os.path.join(dirpath, f)).read().lower().replace("no oracle", ""), f
