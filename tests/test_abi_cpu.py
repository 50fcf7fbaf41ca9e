"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/chime_bf.h declares; argument validation fails loudly without a GPU."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bf():
    import __graft_entry__ as g
    g.build()
    import paper_1702_04728_b200 as bf
    return bf


def test_every_declared_symbol_is_exported(bf):
    hdr = open(os.path.join(ROOT, "include", "chime_bf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(chime_bf_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(bf.EXPORTS), declared ^ set(bf.EXPORTS)
    lib = bf.load_library()
    for name in declared:
        assert getattr(lib, name) is not None


def test_params_struct_matches_header(bf):
    hdr = open(os.path.join(ROOT, "include", "chime_bf.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} chime_bf_params;", hdr, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        for part in decl.split(","):
            names.append(re.findall(r"([A-Za-z_][A-Za-z0-9_]*)\s*$", part.strip())[0])
    assert names == [f[0] for f in bf.chime_bf_params._fields_]


def test_invalid_arguments_fail_loudly(bf):
    import torch
    with pytest.raises(bf.ChimeBfError, match="zero_pad"):
        bf.plan_create(1, zero_pad=300)
    with pytest.raises(bf.ChimeBfError, match="upchan_len"):
        bf.plan_create(1, upchan_len=64)
    with pytest.raises(bf.ChimeBfError, match="n_time"):
        bf.plan_create_ex(1, n_time=1000)
    with pytest.raises(bf.ChimeBfError, match="n_coarse"):
        bf.plan_create(0)
    if not torch.cuda.is_available():
        # no CPU fallback: a valid request without a device must raise, not compute
        with pytest.raises(bf.ChimeBfError, match="no CUDA device"):
            bf.plan_create(1)
    lib = bf.load_library()
    assert lib.chime_bf_execute(None, None, None, None) == -1
    assert b"null" in lib.chime_bf_last_error()
    lib.chime_bf_destroy(None)  # NULL-safe


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1702_04728_b200")
    for dp, _, fns in os.walk(pkg):
        for fn in fns:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dp, fn)).read()
                assert "oracle" not in src.lower(), f"{fn} mentions the oracle"
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", fn)).read()
            code = "\n".join(l for l in src.splitlines()
                             if re.match(r"\s*(import\s+[\w.]+(\s+as\s+\w+)?\s*$|from\s+[\w.]+\s+import\s|#include)", l))
            assert "paper_1702_04728_b200" not in code and "csrc" not in code and "chime_bf.h" not in code
