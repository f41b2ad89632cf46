"""CPU-side checks of the C-ABI boundary: libobem.so builds, loads, and exports every symbol include/obem.h
declares; the Python binding declares the same set.  No compute calls (no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "obem.h")


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(obem_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2110_09214_b200 import build
    return build.build_lib()


def test_header_declares_the_path_calls():
    names = declared_symbols()
    for must in ["obem_create", "obem_destroy", "obem_set_softening", "obem_set_panels", "obem_set_sigma",
                 "obem_set_charges", "obem_eval_at_charges", "obem_eval_at_points", "obem_status_string"]:
        assert must in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in declared_symbols():
        assert hasattr(lib, name), "libobem.so does not export %s" % name


def test_binding_covers_every_declared_symbol(lib_path):
    from paper_2110_09214_b200 import api
    assert sorted(api.SIGNATURES) == declared_symbols()


def test_no_torch_types_in_the_abi():
    src = open(HEADER).read()
    assert "torch" not in re.sub(r"/\*.*?\*/", "", src, flags=re.S).lower()
    assert "at::" not in src and "Tensor" not in re.sub(r"/\*.*?\*/", "", src, flags=re.S)


def test_status_strings_and_null_handling(lib_path):
    from paper_2110_09214_b200 import api
    assert api.status_string(0) == "OBEM_OK"
    for s in (-1, -2, -3, -4):
        assert api.status_string(s).startswith("OBEM_E")
    lib = api.load_library()
    assert lib.obem_create(None, 0) == -1                   # OBEM_EINVAL, no device touched
    assert lib.obem_destroy(None) == 0
    assert lib.obem_n_charges(None) == -1
    assert lib.obem_set_softening(None, 0.0, 0.0) == -1


def test_create_fails_loudly_without_a_device(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2110_09214_b200 import api
    with pytest.raises(api.ObemError) as e:
        api.Context(0)
    assert e.value.status == -3                             # OBEM_ECUDA: there is no CPU fallback


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2110_09214_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "obem_ref" not in txt, f
    txt = open(os.path.join(ROOT, "oracle", "ref.py")).read()
    assert not re.search(r"^\s*(from|import)\s+paper_2110_09214_b200\b", txt, flags=re.M)
