"""Host-side checks of the C-ABI boundary that need no GPU: the library builds for sm_100a, loads, and
exports every symbol include/lartpc.h declares; the binding's structs match the header field for field."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2212_09807_b200 import build, lartpc
    build.build()
    return lartpc.load_library()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "lartpc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lartpc_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    names = _declared_functions()
    assert "lartpc_run_spill" in names and "lartpc_sim_create" in names and len(names) >= 14
    for n in names:
        assert getattr(lib, n) is not None, n
    from paper_2212_09807_b200 import lartpc
    assert sorted(lartpc.EXPORTS) == names


def test_strerror(lib):
    assert lib.lartpc_strerror(0) == b"ok"
    assert b"capacity" in lib.lartpc_strerror(-2).lower() or b"small" in lib.lartpc_strerror(-2).lower()


def _header_struct_fields(name):
    src = open(os.path.join(ROOT, "include", "lartpc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    body = re.search(r"typedef struct \{((?:(?!typedef).)*?)\}\s*" + name + r"\s*;", src, flags=re.S).group(1)
    fields = []
    for stmt in body.split(";"):
        stmt = stmt.strip()
        if not stmt:
            continue
        parts = stmt.replace("const ", "").split(None, 1)
        for f in parts[1].split(","):
            fields.append(f.replace("*", "").strip())
    return fields


@pytest.mark.parametrize("cname,pyname", [
    ("lartpc_params_t", "Params"), ("lartpc_tpc_t", "Tpc"), ("lartpc_segments_t", "Segments"),
    ("lartpc_drifted_t", "Drifted"), ("lartpc_pixmap_t", "Pixmap"), ("lartpc_pixmap_info_t", "PixmapInfo"),
    ("lartpc_signals_t", "Signals"), ("lartpc_waveforms_t", "Waveforms"), ("lartpc_hits_t", "Hits"),
    ("lartpc_stats_t", "Stats"), ("lartpc_truth_t", "Truth"), ("lartpc_light_params_t", "LightParams")])
def test_binding_structs_follow_the_header(cname, pyname):
    from paper_2212_09807_b200 import lartpc
    want = _header_struct_fields(cname)
    got = [f[0] for f in getattr(lartpc, pyname)._fields_]
    assert got == want


def test_workload_param_names_match_header():
    from paper_2212_09807_b200 import lartpc, workloads
    assert set(workloads.default_params()) == {f[0] for f in lartpc.Params._fields_}


def test_sim_create_rejects_bad_arguments_without_a_gpu(lib):
    """Argument validation happens before any device work, so NULL arguments fail cleanly even here."""
    out = ctypes.c_void_p()
    rc = lib.lartpc_sim_create(None, None, 0, None, ctypes.c_size_t(0), ctypes.byref(out))
    assert rc == -1
    assert lib.lartpc_quench(None, None, ctypes.c_int64(0), None, None, None) == -1


def test_no_product_import_of_the_oracle():
    """The product path must never route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2212_09807_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "lartpc_oracle" not in txt, f
    txt = open(os.path.join(ROOT, "oracle", "lartpc_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "lartpc.h" not in txt and "liblartpc.so" not in txt and "from paper_2212_09807_b200 import lartpc" not in txt
