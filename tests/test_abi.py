"""The C-ABI boundary without a GPU: the library builds, loads, exports every function include/fe_cheb.h declares, the
Python binding lists the same names, and a call without a CUDA device fails loudly instead of falling back."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "fe_cheb.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"^\s*(?:const\s+char\s*\*|int64_t|int)\s+(\w+)\s*\(", text, flags=re.M)))


def test_header_declares_the_four_named_calls():
    names = _declared()
    for required in ("fe_mesh_create", "fe_set_potential", "fe_apply_H", "cheb_filter"):  # BASELINE.json north_star
        assert required in names
    assert len(names) >= 20


def test_library_exports_every_declared_symbol():
    import paper_2510_10529_b200 as fe
    from paper_2510_10529_b200 import binding, build
    build.build()
    lib = ctypes.CDLL(fe.library_path())
    for name in _declared():
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == _declared()
    for name in binding.EXPORTS:  # the binding exposes the same names
        assert hasattr(fe, name), name


def test_no_cpu_fallback():
    """Without a CUDA device every entry point that needs one returns an error code with a message; nothing computes."""
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2510_10529_b200 as fe
    e = np.array([0.0, 1.0, 2.0])
    with pytest.raises(fe.FEError) as ei:
        fe.FEMesh(e, e, e, 2)
    assert ei.value.code < 0 and str(ei.value)


def test_argument_errors_need_no_device():
    import paper_2510_10529_b200 as fe
    lib = fe.load_library()
    out = ctypes.c_void_p()
    e = (ctypes.c_double * 3)(0.0, 1.0, 2.0)
    assert lib.fe_mesh_create(e, 2, e, 2, e, 2, 9, 0, ctypes.byref(out)) == -1       # order outside 1..8
    assert b"order" in lib.fe_last_error()
    bad = (ctypes.c_double * 3)(0.0, 1.0, 1.0)
    assert lib.fe_mesh_create(bad, 2, e, 2, e, 2, 2, 0, ctypes.byref(out)) == -1     # edges not increasing
    assert lib.fe_mesh_create(None, 2, e, 2, e, 2, 2, 0, ctypes.byref(out)) == -1    # NULL edges
    assert lib.fe_num_nodes(None) < 0 and lib.fe_mesh_destroy(None) == 0
