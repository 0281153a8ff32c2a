"""CPU-only: libsgw.so loads and exports every symbol include/sgw.h declares; no compute calls."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "sgw.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sgw_[a-z_A-Z0-9]+)\s*\(", src)))


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


_CTYPE = {"int": C.c_int, "double": C.c_double, "uint64_t": C.c_uint64, "int64_t": C.c_int64}


def _prototypes():
    """{name: (restype token, [arg type strings])} parsed from include/sgw.h."""
    src = open(os.path.join(ROOT, "include", "sgw.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    protos = {}
    for m in re.finditer(r"([A-Za-z_0-9 ]+?[ *]+)(sgw_[A-Za-z_0-9]+)\s*\(([^)]*)\)\s*;", src):
        args = [a.strip() for a in m.group(3).split(",")] if m.group(3).strip() != "void" else []
        protos[m.group(2)] = (m.group(1).strip(), args)
    return protos


def _expected_ctype(arg):
    """ctypes type the binding must use for one C parameter declaration."""
    if "*" in arg:
        base = arg.replace("const", "").split("*")[0].strip()
        if arg.count("*") == 1 and base == "double" and re.search(r"\bh_", arg):
            return C.POINTER(C.c_double)              # host double arrays / out-parameters
        if arg.count("*") == 1 and base == "int64_t" and "count" in arg:
            return C.POINTER(C.c_int64)
        if arg.count("*") == 1 and base == "double" and "total_ms" in arg:
            return C.POINTER(C.c_double)
        if arg.count("*") == 2:
            return C.POINTER(C.c_void_p)
        return C.c_void_p                             # device pointers and the opaque context
    return _CTYPE[arg.split()[0]]


def test_ctypes_argtypes_match_the_header_prototypes():
    """A signature drift between include/sgw.h and the hand-written ctypes argtypes in api.py fails here."""
    from paper_2601_21005_b200 import api
    lib = api.load()
    protos = _prototypes()
    assert set(protos) == set(api.EXPORTS)
    for name, (ret, args) in protos.items():
        fn = getattr(lib, name)
        if name == "sgw_last_error":
            assert fn.restype is C.c_char_p and not args
            continue
        assert fn.argtypes is not None, name
        want = [_expected_ctype(a) for a in args]
        assert len(fn.argtypes) == len(want), (name, fn.argtypes, args)
        for got, w_, a in zip(fn.argtypes, want, args):
            assert got is w_ or (C.sizeof(got) == C.sizeof(w_) and got in (C.c_void_p,) and w_ in (C.c_void_p,)), (name, a, got, w_)
        assert (fn.restype is C.c_int64) == (ret == "int64_t"), name


def _build_consumer(tmp_path):
    from paper_2601_21005_b200 import build
    lib = build.build()
    exe = str(tmp_path / "c_abi_consumer")
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    cmd = ["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-I", os.path.join(cuda, "include"),
           os.path.join(ROOT, "tests", "c_abi_consumer.c"), lib, "-L", os.path.join(cuda, "lib64"), "-lcudart", "-lm",
           "-Wl,-rpath," + os.path.dirname(lib), "-Wl,-rpath," + os.path.join(cuda, "lib64"), "-o", exe]
    subprocess.check_call(cmd)
    return exe


def test_c_consumer_compiles_links_and_reports_errors_without_gpu(tmp_path):
    """include/sgw.h compiles as C99, every entry point links, and error paths behave as documented."""
    import torch
    exe = _build_consumer(tmp_path)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert ("gpu ok" if torch.cuda.is_available() else "nogpu ok") in r.stdout


@pytest.mark.gpu
def test_c_consumer_runs_every_entry_point_on_the_gpu(tmp_path):
    exe = _build_consumer(tmp_path)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "gpu ok" in r.stdout, r.stdout + r.stderr
