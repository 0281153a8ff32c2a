"""CPU-only: libsgw.so loads and exports every symbol include/sgw.h declares; no compute calls."""
import ctypes as C
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "sgw.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sgw_[a-z_A-Z]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_2601_21005_b200 import build
    lib = C.CDLL(build.build())
    names = _declared()
    assert {"sgw_init_grid", "sgw_random_vectors", "sgw_apply_H", "sgw_cheb_filter", "sgw_td_propagate",
            "sgw_hartree"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_binding_names_match_header_and_fail_without_gpu():
    import torch
    from paper_2601_21005_b200 import api
    assert set(api.EXPORTS) == set(_declared())
    for n in api.EXPORTS:
        if n not in ("sgw_init_grid", "sgw_destroy", "sgw_last_error"):
            assert hasattr(api.Context, n), n
    if not torch.cuda.is_available():          # no CPU fallback: init must fail loudly
        lib = api.load()
        h = C.c_void_p()
        assert lib.sgw_init_grid(C.byref(h), 32, 32, 32, 0.5, 0.5, 0.5, 1, None) == -4
        assert b"no CPU fallback" in lib.sgw_last_error()
        assert lib.sgw_init_grid(C.byref(h), 30, 32, 32, 0.5, 0.5, 0.5, 1, None) == -2
        assert lib.sgw_init_grid(C.byref(h), 32, 32, 32, -0.5, 0.5, 0.5, 1, None) == -1


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2601_21005_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "sgw_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            assert "paper_2601_21005_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "paper_2601_21005_b200/csrc", "")
