"""CPU-only checks of the boundary: libhepk.so loads without a GPU and exports every symbol that
include/hepk.h declares; argument validation (host side) returns error codes and messages."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1906_06242_b200 import build
    return C.CDLL(build.build())


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "hepk.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hepk_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = declared_symbols()
    for n in ["hepk_select_mask", "hepk_segmented_reduce_sum", "hepk_segmented_reduce_max", "hepk_segmented_reduce_min",
              "hepk_segmented_reduce_count", "hepk_segmented_reduce_argmax", "hepk_deltar_mask", "hepk_pair_invmass",
              "hepk_lookup_binned", "hepk_fill_histogram", "hepk_analysis_chain", "hepk_chain_workspace_bytes",
              "hepk_analysis_chain_host", "hepk_last_error", "hepk_version"]:
        assert n in names


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), f"libhepk.so does not export {name}"


def test_host_side_validation_without_gpu(lib):
    lib.hepk_last_error.restype = C.c_char_p
    assert lib.hepk_version() >= 100
    # negative sizes / NULL required pointers -> HEPK_ERR_INVALID (-1) before any CUDA call
    assert lib.hepk_select_mask(None, None, C.c_int64(-1), C.c_float(0), C.c_float(0), None, None) == -1
    assert b"n < 0" in lib.hepk_last_error()
    assert lib.hepk_select_mask(None, None, C.c_int64(5), C.c_float(0), C.c_float(0), None, None) == -1
    assert lib.hepk_segmented_reduce_sum(None, None, C.c_int64(3), C.c_int64(0), None, None, None, C.c_int32(0), None) == -1
    assert lib.hepk_segmented_reduce_sum(None, None, C.c_int64(0), C.c_int64(0), None, None, None, C.c_int32(7), None) == -1
    assert lib.hepk_fill_histogram(None, None, C.c_int64(4), None, C.c_int32(0), None, None, None) == -1
    assert lib.hepk_fill_histogram(None, None, C.c_int64(4), C.c_void_p(8), C.c_int32(1 << 20), None, None, None) == -2
    assert lib.hepk_lookup_binned(None, None, C.c_int64(4), None, C.c_int32(3), None, C.c_int32(0), None, None, None) == -1
    assert lib.hepk_analysis_chain(None, None, C.c_size_t(0), None) == -1
    # empty inputs are fine and touch nothing
    assert lib.hepk_select_mask(None, None, C.c_int64(0), C.c_float(0), C.c_float(0), None, None) == 0
    assert lib.hepk_deltar_mask(None, None, None, C.c_int64(0), None, None, None, None, C.c_int64(0), None,
                                C.c_int64(0), C.c_float(0.4), None, None) == 0


def test_binding_struct_matches_header():
    from paper_1906_06242_b200 import binding
    # field-by-field the ctypes mirror follows include/hepk.h; the size is what the C compiler computes
    import subprocess, tempfile
    src = '#include "hepk.h"\n#include <stdio.h>\nint main(){printf("%zu %zu\\n", sizeof(hepk_chain_desc), sizeof(hepk_collection));return 0;}\n'
    with tempfile.TemporaryDirectory() as td:
        c = os.path.join(td, "s.c")
        open(c, "w").write(src)
        exe = os.path.join(td, "s")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe], check=True)
        sz_desc, sz_coll = map(int, subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split())
    assert C.sizeof(binding.ChainDesc) == sz_desc
    assert C.sizeof(binding.Collection) == sz_coll


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1906_06242_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "hepo" not in text and "import oracle" not in text and "from oracle" not in text, f


def test_bench_algorithmic_bytes_matches_survey_8d():
    """bench.py's algorithmic bytes per event equal SURVEY.md 8(d)'s table (config 2: 210.3 B/event) on a sample."""
    import importlib.util
    import hepgen
    spec = importlib.util.spec_from_file_location("bench", os.path.join(ROOT, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    wl = hepgen.generate(2, n_events=200_000)
    per_event = bench.algorithmic_bytes(wl) / wl.n_events
    nj = wl.jets.n_objects / wl.n_events
    nm = wl.muons.n_objects / wl.n_events
    ne = wl.electrons.n_objects / wl.n_events
    want = 24 + 16 * nj + 12 * nm + 12 * ne + 4 + 20
    assert abs(per_event - want) < 0.01
    assert 205 < per_event < 216                       # 210.3 B/event for config 2
    assert bench.algorithmic_bytes(wl, event_outputs=False) == bench.algorithmic_bytes(wl) - 20 * wl.n_events
