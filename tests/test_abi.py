"""CPU-side checks of the boundary: libg3.so builds for sm_100a, loads, and exports every
symbol include/g3.h declares.  No compute calls (no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1708_08619_b200 import build
    build.build()
    import paper_1708_08619_b200 as g3
    return g3.load()


def declared_symbols(header="g3.h", macro="G3_API"):
    text = open(os.path.join(ROOT, "include", header)).read()
    return re.findall(macro + r"\s+[\w\s\*]+?\b(g3_\w+)\s*\(", text)


def test_header_symbols_exported(lib):
    names = declared_symbols()
    assert len(names) >= 10 and "g3_plan_create" in names and "g3_finalize" in names
    for name in names:
        assert hasattr(lib, name), name


def test_binding_lists_the_same_names(lib):
    import paper_1708_08619_b200 as g3
    assert sorted(g3.EXPORTS) == sorted(declared_symbols())


def test_every_header_has_its_library():
    """every include/*.h is covered: g3.h -> libg3.so, g3_bench.h -> libg3bench.so (bench.py's
    measurement aid, kept out of the product library)"""
    import paper_1708_08619_b200 as g3
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["g3.h", "g3_bench.h"]
    names = declared_symbols("g3_bench.h", "G3_BENCH_API")
    assert sorted(names) == sorted(g3.BENCH_EXPORTS) == ["g3_microbench"]
    blib = g3.load_bench()
    for name in names:
        assert hasattr(blib, name), name
    assert not hasattr(g3.load(), "g3_microbench")          # not part of the product ABI
    rate = ctypes.c_double()
    assert blib.g3_microbench(7, 64, 1024, ctypes.byref(rate), None) == g3.G3_EINVAL


def test_strerror_and_argument_errors(lib):
    import paper_1708_08619_b200 as g3
    assert g3.strerror(g3.G3_OK) == "ok"
    assert "capacity" in g3.strerror(g3.G3_ECAPACITY)
    h = ctypes.c_void_p()
    bins = g3.binding.g3_bins(8, 8)
    # argument validation happens before any CUDA call
    assert lib.g3_plan_create(None, 100, 1.0, 0.2, bins) == g3.G3_EINVAL
    assert lib.g3_plan_create(ctypes.byref(h), 2, 1.0, 0.2, bins) == g3.G3_EINVAL        # n < 3
    assert lib.g3_plan_create(ctypes.byref(h), 100, 1.0, 0.5, bins) == g3.G3_EINVAL      # r_max >= box/2
    assert lib.g3_plan_create(ctypes.byref(h), 100, -1.0, 0.2, bins) == g3.G3_EINVAL
    assert lib.g3_plan_create(ctypes.byref(h), 100, 1.0, 0.2, g3.binding.g3_bins(0, 8)) == g3.G3_EINVAL
    assert h.value is None
    assert lib.g3_accumulate_frame(None, None, None) == g3.G3_EINVAL
    assert lib.g3_finalize(None, None, None, None, None) == g3.G3_EINVAL
    lib.g3_plan_destroy(None)


def test_no_allocation_entry_point_limits_and_errors(lib):
    """g3_msd_static (the MSD entry point for callers that cannot allocate device memory): the limit
    the binding quotes is the header's, the scratch size follows from it, its own status code has a
    description, and argument errors are reported before any CUDA call"""
    import paper_1708_08619_b200 as g3
    text = open(os.path.join(ROOT, "include", "g3.h")).read()
    limit = int(re.search(r"#define G3_MSD_STATIC_MAX_PARTIALS (\d+)", text).group(1))
    assert limit == g3.G3_MSD_STATIC_MAX_PARTIALS == 1 << 19
    assert "#define G3_MSD_STATIC_SCRATCH_BYTES (256 + 16 * G3_MSD_STATIC_MAX_PARTIALS)" in text
    assert (32768 // 32) * 500 <= limit                      # the config-4 shape with every lag fits
    assert int(re.search(r"G3_ELIMIT = (\d+)", text).group(1)) == g3.G3_ELIMIT
    assert "scratch" in g3.strerror(g3.G3_ELIMIT)
    assert lib.g3_msd_static(None, 10, 10, 30, 1.0, 5, None, None, None) == g3.G3_EINVAL     # null positions
    buf = ctypes.create_string_buffer(8)                     # never dereferenced: the arguments are refused first
    assert lib.g3_msd_static(buf, 10, 10, 29, 1.0, 5, None, None, None) == g3.G3_EINVAL      # stride < 3 n
    assert lib.g3_msd_static(buf, 10, 10, 30, 1.0, 10, None, None, None) == g3.G3_EINVAL     # max_lag > F - 1
    assert lib.g3_msd_static(buf, 10, 10, 30, 0.0, 5, None, None, None) == g3.G3_EINVAL      # box


def test_no_cpu_fallback_without_gpu(lib):
    """On a box without a CUDA device plan creation must fail loudly, never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_1708_08619_b200 as g3
    with pytest.raises(g3.G3Error) as e:
        g3.Plan(100, 1.0, 0.2, 8)
    assert e.value.code == g3.G3_ECUDA


def test_product_does_not_touch_oracle():
    """The product package must not import, read or link anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1708_08619_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in text.lower(), os.path.join(dirpath, fn)
