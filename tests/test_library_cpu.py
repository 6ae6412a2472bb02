"""CPU-side checks of the CUDA library: it loads, exports every symbol include/vd.h declares, and
fails loudly (no CPU fallback) when no device is present.  No compute calls here."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "vd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(vd_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_2509_07175_b200 import binding, build
    build.build()
    lib = ctypes.CDLL(build.lib_path())
    names = _declared_symbols()
    assert "vd_create" in names and "vd_compute" in names and "vd_destroy" in names and "vd_set_domain" in names
    for name in names:
        assert hasattr(lib, name), f"libvd.so does not export {name}"
    assert sorted(binding.EXPORTS) == names


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2509_07175_b200 import binding
    with pytest.raises(binding.VdError) as e:
        binding.Context(np.random.default_rng(0).random((10, 2)))
    assert e.value.status == 5  # VD_E_CUDA


def test_argument_errors_need_no_device():
    from paper_2509_07175_b200 import binding
    lib = binding.load()
    h = ctypes.c_void_p()
    s = np.zeros((4, 2))
    assert lib.vd_create(None, 4, 2, ctypes.byref(h)) == 1          # VD_E_ARG
    assert lib.vd_create(s.ctypes.data, 0, 2, ctypes.byref(h)) == 1
    assert lib.vd_create(s.ctypes.data, 4, 5, ctypes.byref(h)) == 2  # VD_E_DIM
    assert lib.vd_compute(None, None) == 1
    assert lib.vd_version().startswith(b"vd-b200")


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2509_07175_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "vd_oracle" not in txt, f
    txt = open(os.path.join(ROOT, "oracle", "vd_oracle.cpp")).read() + open(os.path.join(ROOT, "oracle", "oracle.py")).read()
    assert "paper_2509_07175_b200" not in txt.replace("(paper_2509_07175_b200/csrc)", "") and "vd.h\"" not in txt


def test_input_recipes_are_seeded_and_shaped():
    from paper_2509_07175_b200 import inputs
    w = inputs.config(1)
    assert w.n == 2000 and w.m == 2 and w.kind == 0
    assert np.array_equal(w.sites, inputs.config(1).sites)
    w = inputs.config(2, "small")
    assert w.m == 4 ** 3 * 6 and w.n == 2000 and abs(w.measure - 1.0) < 1e-12
    w = inputs.config(4, "small")
    assert w.m == 1024 and w.kind == 1
    v, t = inputs.cube_kuhn_mesh(3)
    # conforming: every interior face is shared by exactly two tets
    faces = {}
    for a, tet in enumerate(t):
        for k in range(4):
            key = tuple(sorted(np.delete(tet, k).tolist()))
            faces.setdefault(key, []).append(a)
    assert max(len(v) for v in faces.values()) == 2
