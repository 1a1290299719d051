"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol that
include/das.h declares, and rejects bad arguments before touching CUDA.  No compute calls."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "das.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(das_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared_functions()
    for need in ("das_plan_create", "das_convert", "das_execute"):
        assert need in names


def test_library_exports_every_declared_symbol(das_lib):
    lib = ctypes.CDLL(das_lib.library_path())
    names = _declared_functions()
    assert sorted(das_lib.EXPORTS) == names
    for n in names:
        assert hasattr(lib, n), n


def test_no_torch_types_in_signatures():
    src = open(os.path.join(ROOT, "include", "das.h")).read()
    assert "torch" not in src.lower() and "at::" not in src and "#include <cuda" not in src


def _good_kwargs():
    return dict(elem_pos=np.zeros((4, 3), np.float32), tx_type=[0], tx_v=[[0, 0, 1]], tx_t0=[0.0],
                xs=[0.0], ys=[0.0], zs=[1e-3], c=1540.0, fc=7.8e6, fs=15.6e6, n_samples=64)


@pytest.mark.parametrize("patch,status", [
    (dict(n_samples=1), "INVALID_ARG"),
    (dict(c=0.0), "INVALID_ARG"),
    (dict(c=float("nan")), "INVALID_ARG"),
    (dict(fs=-1.0), "INVALID_ARG"),
    (dict(fc=-1.0), "INVALID_ARG"),
    (dict(data_kind=1, fc=7.8e6), "INVALID_ARG"),          # RF with fc != 0
    (dict(tx_v=[[0, 0, 0.5]]), "INVALID_ARG"),             # non-unit plane direction
    (dict(tx_type=[7]), "UNSUPPORTED"),
    (dict(storage=3), "UNSUPPORTED"),
    (dict(data_kind=2), "UNSUPPORTED"),
    (dict(algo=9), "UNSUPPORTED"),
    (dict(n_frames=-1), "INVALID_ARG"),
    (dict(n_frames=4, algo=3, storage=1), "UNSUPPORTED"),      # tensor-core batch needs a multiple of 8
    (dict(n_frames=8, algo=3, storage=0), "UNSUPPORTED"),      # ... and fp16 storage
    (dict(xs=[float("inf")]), "INVALID_ARG"),
    (dict(elem_dir=np.tile([0, 0, 2.0], (4, 1))), "INVALID_ARG"),
])
def test_plan_create_rejects_bad_arguments(das_lib, patch, status):
    kw = _good_kwargs()
    kw.update(patch)
    args = [kw.pop(k) for k in ("elem_pos", "tx_type", "tx_v", "tx_t0", "xs", "ys", "zs")]
    with pytest.raises(das_lib.DasError) as ei:
        das_lib.Plan(*args, **kw)
    assert das_lib.status_string(ei.value.status) == "DAS_ERR_" + status
    assert das_lib.last_error() != ""


def test_null_arguments(das_lib):
    lib = das_lib.load()
    h = ctypes.c_void_p()
    assert lib.das_plan_create(None, ctypes.byref(h)) == das_lib.ERR_INVALID_ARG
    assert lib.das_plan_create(None, None) == das_lib.ERR_INVALID_ARG
    assert lib.das_plan_destroy(None) == das_lib.OK
    assert lib.das_convert(None, None, None, 1.0, None) == das_lib.ERR_INVALID_ARG
    assert lib.das_execute(None, None, None, None) == das_lib.ERR_INVALID_ARG
    assert lib.das_beamform_host(None, None, None, None) == das_lib.ERR_INVALID_ARG
    assert lib.das_plan_count_work(None, None, None) == das_lib.ERR_INVALID_ARG
    assert lib.das_converted_bytes(None) == 0
    assert das_lib.status_string(0) == "DAS_OK"


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2606_13259_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "das_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2606_13259_b200\b", txt, flags=re.M), f
