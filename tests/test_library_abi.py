"""CPU-side checks of the boundary: libodb.so builds (nvcc cross-compiles without a GPU), loads, and
exports every symbol include/odb.h declares; the ctypes structs match the C layout; without a CUDA
device the product path fails loudly instead of falling back."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "odb.h")


def _declared_symbols():
    text = open(HEADER).read()
    return sorted(set(re.findall(r"^ODB_API[^;(]*?\b(odb_[a-z_]+)\(", text, flags=re.M)))


def test_header_declares_the_entry_points():
    names = _declared_symbols()
    for must in ("odb_form_groups", "odb_align", "odb_collate", "odb_run", "odb_run_host", "odb_create",
                 "odb_destroy", "odb_plan_query", "odb_round_status"):
        assert must in names


def test_library_loads_and_exports_every_declared_symbol():
    import paper_2606_19989_b200 as P
    L = P.load()
    declared = _declared_symbols()
    assert sorted(P.SYMBOLS) == declared          # the binding covers the header, nothing more
    for name in declared:
        assert hasattr(L, name), name
    out = subprocess.check_output(["nm", "-D", "--defined-only", P.library_path()], text=True)
    exported = {ln.split()[-1] for ln in out.splitlines() if " T " in ln}
    assert set(declared) <= exported


def test_struct_layouts_match_the_header():
    """Compile a tiny C program against odb.h and compare sizeof / offsetof with the ctypes structs."""
    import paper_2606_19989_b200 as P
    fields = {
        "odb_params": [f for f, _ in P.odb_params._fields_],
        "odb_plan_info": [f for f, _ in P.odb_plan_info._fields_],
        "odb_outputs": [f for f, _ in P.odb_outputs._fields_],
    }
    src = ["#include <stdio.h>", "#include <stddef.h>", '#include "odb.h"', "int main(void){"]
    for s, fs in fields.items():
        src.append('printf("%s %%zu\\n", sizeof(%s));' % (s, s))
        for f in fs:
            src.append('printf("%s.%s %%zu\\n", offsetof(%s, %s));' % (s, f, s, f))
    src.append("return 0;}")
    tmp = os.path.join(ROOT, "tests", ".abi_probe_%d" % os.getpid())
    try:
        with open(tmp + ".c", "w") as f:
            f.write("\n".join(src))
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", tmp, tmp + ".c"])
        out = subprocess.check_output([tmp], text=True)
    finally:
        for p in (tmp, tmp + ".c"):
            if os.path.exists(p):
                os.remove(p)
    got = dict(line.split() for line in out.splitlines())
    for s in fields:
        cls = getattr(P, s)
        assert int(got[s]) == ctypes.sizeof(cls), s
        for f in fields[s]:
            assert int(got["%s.%s" % (s, f)]) == getattr(cls, f).offset, (s, f)


def test_status_strings_and_param_validation_need_no_gpu():
    import paper_2606_19989_b200 as P
    assert P.status_string(P.ODB_OK) == "ok"
    assert "capacity" in P.status_string(P.ODB_ERR_CAPACITY)
    with pytest.raises(P.OdbError) as ei:
        P.odb_create(P.make_params(0, 1024), 0, 16)          # n_ranks < 1
    assert ei.value.status == P.ODB_ERR_INVALID_ARG
    with pytest.raises(P.OdbError) as ei:
        P.odb_create(P.make_params(2, 0), 0, 16)             # budget < 1
    assert ei.value.status == P.ODB_ERR_INVALID_ARG


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_2606_19989_b200 as P
    with pytest.raises(P.OdbError) as ei:
        P.odb_create(P.make_params(2, 2048), 0, 128)
    assert ei.value.status == P.ODB_ERR_CUDA


def test_product_never_imports_the_oracle():
    """The CUDA package and the oracle share nothing and neither imports the other."""
    pkg = os.path.join(ROOT, "paper_2606_19989_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), fn
                assert "odb_oracle" not in text, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", fn)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2606_19989_b200\b", text, flags=re.M), fn
            assert '#include "odb.h"' not in text, fn
