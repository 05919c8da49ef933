"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a without a GPU, loads,
and exports every symbol include/nb.h declares; the Python binding mirrors the header (struct
layouts, enum values, names).  No compute call is made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "nb.h")


@pytest.fixture(scope="module")
def header_text():
    with open(HEADER) as fh:
        return fh.read()


@pytest.fixture(scope="module")
def built_lib():
    from paper_2006_09167_b200 import build
    return C.CDLL(build.build())


def declared_functions(text):
    body = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"^\s*(?:int|void|const char\*)\s+(nb_[a-z0-9_]+)\s*\(", body, flags=re.M)))


def test_header_declares_the_five_working_calls(header_text):
    names = declared_functions(header_text)
    for n in ("nb_init", "nb_put_atoms", "nb_search", "nb_prune", "nb_forces"):   # BASELINE.json north_star
        assert n in names


def test_library_exports_every_declared_symbol(header_text, built_lib):
    names = declared_functions(header_text)
    assert len(names) >= 15
    for n in names:
        assert hasattr(built_lib, n), f"{n} declared in include/nb.h but not exported"


def test_binding_mirrors_header(header_text):
    from paper_2006_09167_b200 import nb
    assert sorted(nb.EXPORTS) == declared_functions(header_text)
    enums = dict(re.findall(r"(NB_[A-Z_0-9]+)\s*=\s*(-?\d+)", header_text))
    for code, name in nb.NB_ERR.items():
        assert int(enums[name]) == code
    assert int(enums["NB_COUL_EWALD"]) == nb.NB_COUL_EWALD and int(enums["NB_COUL_RF"]) == nb.NB_COUL_RF
    assert int(enums["NB_MOD_POTSHIFT"]) == nb.NB_MOD_POTSHIFT
    assert int(enums["NB_T_NKINDS"]) == len(nb.NB_T_NAMES)
    for i, k in enumerate(nb.NB_T_NAMES):
        assert int(enums["NB_T_" + k.upper()]) == i
    # struct layouts: field order and C types of nb_params / nb_stats
    def fields(struct):
        m = re.search(r"typedef struct \{([^}]*)\} " + struct + ";", header_text, flags=re.S)
        body = re.sub(r"/\*.*?\*/", "", m.group(1), flags=re.S)
        out = []
        for decl in body.split(";"):
            decl = decl.strip()
            if not decl:
                continue
            typ, rest = re.match(r"((?:const\s+)?[a-z0-9_]+\s*\*?)\s*(.*)", decl, flags=re.S).groups()
            for nm in rest.split(","):
                out.append((nm.strip().lstrip("*").strip(), typ.replace(" ", "")))
        return out
    cmap = {"int32_t": C.c_int32, "int64_t": C.c_int64, "float": C.c_float, "void*": C.c_void_p,
            "constfloat*": C.c_void_p, "constint32_t*": C.c_void_p}
    for struct, cls in (("nb_params", nb.nb_params), ("nb_stats", nb.nb_stats)):
        want = fields(struct)
        got = [(n, t) for n, t in cls._fields_]
        assert [n for n, _ in want] == [n for n, _ in got], struct
        for (n, t), (_, ct) in zip(want, got):
            assert cmap[t] is ct, (struct, n, t)


def test_product_path_does_not_touch_the_oracle():
    """The oracle is test infrastructure: nothing under the package may import or link it."""
    pkg = os.path.join(ROOT, "paper_2006_09167_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".h", ".cpp", ".c")):
                with open(os.path.join(dirpath, fn)) as fh:
                    src = fh.read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), fn
                assert "nb_oracle" not in src and "libnb_oracle" not in src, fn


def test_missing_library_fails_loudly(monkeypatch):
    from paper_2006_09167_b200 import nb
    monkeypatch.setattr(nb, "_lib", None)
    monkeypatch.setattr(nb, "LIB_PATH", "/nonexistent/libnb_b200.so")
    with pytest.raises(RuntimeError, match="no CPU or PyTorch fallback"):
        nb.lib()
