"""CPU-only checks of the boundary: libmk.so loads, exports every symbol include/mk.h declares, the header and the
binding agree, and the library refuses to work without a GPU (no CPU fallback).  No compute calls."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = (ROOT / "include" / "mk.h").read_text()


@pytest.fixture(scope="module")
def lib():
    from paper_2106_04649_b200 import build, binding
    build.build()
    return binding.load()


def declared_functions():
    body = re.sub(r"/\*.*?\*/", "", HEADER, flags=re.S)
    return sorted(set(re.findall(r"\b(mk_[a-zA-Z_]+)\s*\(", body)))


def test_header_cites_the_paper_for_every_entry_point():
    assert "PAPER.md" in HEADER and "eq. (1)" in HEADER
    for nm in ("mk_create", "mk_load_R", "mk_run", "mk_begin", "mk_step", "mk_finish", "mk_synthesis"):
        assert nm in HEADER


def test_every_declared_symbol_is_exported(lib):
    from paper_2106_04649_b200 import binding
    names = declared_functions()
    assert set(names) == set(binding.SYMBOLS), (names, binding.SYMBOLS)
    for nm in names:
        assert getattr(lib, nm) is not None


def test_enum_values_match_header():
    from paper_2106_04649_b200 import binding
    body = re.sub(r"/\*.*?\*/", "", HEADER, flags=re.S)
    for nm, val in re.findall(r"\b(MK_[A-Z_0-9]+)\s*=\s*(-?\d+)", body):
        assert getattr(binding, nm) == int(val), nm


def test_outputs_struct_layout_matches_header():
    from paper_2106_04649_b200 import binding
    m = re.search(r"typedef struct mk_outputs \{(.*?)\} mk_outputs;", HEADER, flags=re.S)
    fields = re.findall(r"float\*\s*(\w+);", m.group(1))
    assert tuple(fields) == binding.OUTPUT_FIELDS
    assert C.sizeof(binding.mk_outputs) == 6 * C.sizeof(C.c_void_p)


def test_operand_view_struct_layout_matches_header():
    from paper_2106_04649_b200 import binding
    m = re.search(r"typedef struct mk_operand_view \{(.*?)\} mk_operand_view;", HEADER, flags=re.S)
    ints = [x.strip() for x in re.search(r"int ([^;]+);", m.group(1)).group(1).split(",")]
    assert "float* plane[2];" in m.group(1)
    assert [nm for nm, _ in binding.mk_operand_view._fields_] == ["plane"] + ints
    assert C.sizeof(binding.mk_operand_view) == 2 * C.sizeof(C.c_void_p) + 4 * len(ints) + (4 * len(ints)) % 8


def test_sharded_create_rejects_bad_row_ranges(lib):
    h = C.c_void_p()
    for row0, nrows in ((-1, 4), (0, 0), (8, 4), (0, 11)):
        assert lib.mk_create_sharded(C.byref(h), 10, 10, 64, 0.004, 10.0, 5.0, 60.0, row0, nrows) == -1
        assert not h


def test_streamed_create_rejects_bad_row_counts(lib):
    h = C.c_void_p()
    for resident, window in ((-1, 0), (11, 0), (4, -2)):
        assert lib.mk_create_streamed(C.byref(h), 10, 10, 64, 0.004, 10.0, 5.0, 60.0, resident, window) == -1
        assert not h


def test_invalid_arguments_are_rejected_before_touching_the_device(lib):
    h = C.c_void_p()
    assert lib.mk_create(C.byref(h), 0, 11, 64, 0.004, 10.0, 5.0, 60.0) == -1       # no shots
    assert not h
    assert lib.mk_create_sharded(C.byref(h), 10, 11, 64, 0.004, 10.0, 5.0, 60.0, 0, 5) == -1   # row sharding needs nshot == nrec
    assert not h
    assert lib.mk_create(C.byref(h), 10, 10, 100, 0.004, 10.0, 5.0, 60.0) == -1     # nt not a power of two
    assert lib.mk_create(C.byref(h), 10, 10, 64, -1.0, 10.0, 5.0, 60.0) == -1
    assert lib.mk_create(C.byref(h), 10, 10, 64, 0.004, 10.0, 60.0, 5.0) == -1      # fmax < fmin
    assert lib.mk_create(C.byref(h), 10, 10, 64, 0.004, 10.0, 5.0, 500.0) == -1     # above Nyquist
    assert lib.mk_create(None, 10, 10, 64, 0.004, 10.0, 5.0, 60.0) == -1
    assert lib.mk_destroy(None) == 0
    assert lib.mk_version().decode().startswith("libmk")


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    assert lib.mk_create(C.byref(h), 10, 10, 64, 0.004, 10.0, 5.0, 60.0) == -4      # MK_ERR_CUDA: fails loudly
    from paper_2106_04649_b200 import binding
    with pytest.raises(RuntimeError):
        binding.Marchenko(10, 10, 64, 0.004, 10.0, 5.0, 60.0)


def test_product_path_does_not_touch_the_oracle():
    pkg = ROOT / "paper_2106_04649_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")):
        txt = f.read_text()
        assert "import oracle" not in txt and "from oracle" not in txt and "marchenko_oracle" not in txt, f
    for f in (ROOT / "oracle").rglob("*"):
        if f.suffix in (".py", ".cpp"):
            txt = f.read_text()
            assert "binding" not in txt.replace("paper_2106_04649_b200.binding / csrc", "") or f.name == "__init__.py"
            assert "import paper_2106_04649_b200" not in txt and "from paper_2106_04649_b200" not in txt, f
