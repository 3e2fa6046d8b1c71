"""CPU checks of the boundary: the C-ABI library loads and exports every symbol include/nnp.h declares."""
import os
import re

from paper_2405_01491_b200 import nnp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "nnp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nnp_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_all_exported_and_bound():
    import __graft_entry__
    __graft_entry__.build()
    names = _declared()
    assert len(names) >= 16
    L = nnp.lib()
    for n in names:
        assert hasattr(L, n), n
        assert n in nnp.EXPORTS and hasattr(nnp, n), n
    assert sorted(nnp.EXPORTS) == names


def test_status_codes_match_header():
    src = open(os.path.join(ROOT, "include", "nnp.h")).read()
    for name, val in re.findall(r"(NNP_[A-Z]+)\s*=\s*(-?\d+)", src):
        assert getattr(nnp, name) == int(val)


def test_params_struct_matches_header_field_order():
    src = open(os.path.join(ROOT, "include", "nnp.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} nnp_params;", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        fptr = re.search(r"\(\s*\*\s*([A-Za-z_0-9]+)\s*\)\s*\(", decl)     # function pointer: ret (*name)(args)
        if fptr:
            fields.append(fptr.group(1))
            continue
        for part in decl.split(","):
            fields.append(re.findall(r"[A-Za-z_0-9]+", part)[-1])
    assert fields == [f[0] for f in nnp.nnp_params._fields_]
