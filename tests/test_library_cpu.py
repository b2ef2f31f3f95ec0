"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol of include/omnimem.h."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "omnimem.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2606_07577_b200 import build
    return ctypes.CDLL(build.build())


def declared_functions():
    src = open(HEADER).read()
    return re.findall(r"^OMNIMEM_API\s+[\w\s\*]+?\b(omnimem_\w+)\s*\(", src, flags=re.M)


def test_header_declares_the_five_calls():
    names = declared_functions()
    for f in ("omnimem_score", "omnimem_allocate", "omnimem_select", "omnimem_compact", "omnimem_compress_chunk"):
        assert f in names
    assert len(names) == len(set(names)) >= 14


def test_library_exports_every_declared_symbol(lib):
    from paper_2606_07577_b200 import omnimem
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} declared in include/omnimem.h but not exported"
    assert set(omnimem.EXPORTS) == set(declared_functions())


def test_strerror_and_argument_validation_without_a_device(lib):
    lib.omnimem_strerror.restype = ctypes.c_char_p
    assert lib.omnimem_strerror(0) == b"ok"
    assert b"workspace" in lib.omnimem_strerror(-3)
    assert lib.omnimem_create(None, None) == -1          # INVALID_ARG before any CUDA call
    assert lib.omnimem_workspace_bytes(None) == 0


def test_binding_struct_matches_header_field_order():
    """The ctypes mirror of omnimem_config lists the fields in the header's order (names aside: `lambda` is a keyword)."""
    from paper_2606_07577_b200 import omnimem
    src = open(HEADER).read()
    body = src[src.index("typedef struct {", src.index("omnimem_ctx omnimem_ctx")):src.index("} omnimem_config;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S).replace("typedef struct {", "")
    fields = []
    for decl in body.split(";"):
        m = re.match(r"\s*(int32_t|float)\s+(.*)", decl.strip(), flags=re.S)
        if m:
            fields += [(m.group(1), f.strip()) for f in m.group(2).split(",")]
    mirror = omnimem.omnimem_config._fields_
    assert len(fields) == len(mirror)
    for (ctype, name), (pname, ptype) in zip(fields, mirror):
        assert ptype is (ctypes.c_int32 if ctype == "int32_t" else ctypes.c_float)
        assert pname == ("lam" if name == "lambda" else name)


def test_no_cpu_fallback_when_no_device():
    import torch
    from paper_2606_07577_b200 import omnimem
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(omnimem.OmniMemError):
        omnimem.OmniMem(L=1, Hq=2, Hkv=1, D=64, dtype="fp32", cache_cap=8, max_chunk_v=4, max_chunk_a=4)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_07577_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "omnimem_ref" not in text and "from oracle" not in text and "import oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_07577_b200" not in text and "from paper_2606_07577_b200" not in text
            assert "csrc" not in text.replace("paper_2606_07577_b200/csrc", "") or f.endswith(".c")


def test_build_refuses_a_source_list_with_a_missing_file(monkeypatch):
    """A SOURCES entry that is not on disk is an error at build time, not an unresolved symbol at load time."""
    from paper_2606_07577_b200 import build
    monkeypatch.setattr(build, "SOURCES", build.SOURCES + ["no_such_file.cu"])
    with pytest.raises(FileNotFoundError, match="no_such_file.cu"):
        build.build()
