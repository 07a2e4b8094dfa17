"""The C-ABI library builds, loads, and exports every symbol include/rips.h declares (no compute calls:
those need a GPU).  Also the host-only error paths that do not touch the device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "rips.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rips_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2003_07989_b200 import build, rips
    build.build()
    return rips.lib()


def test_header_and_binding_agree():
    from paper_2003_07989_b200 import rips
    assert declared_symbols() == sorted(rips.SYMBOLS)


def test_every_declared_symbol_is_exported(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_struct_sizes_match_header():
    from paper_2003_07989_b200 import rips
    # rips_stats_t: 15 int64 + 4 int32; rips_timings_t: 13 floats
    assert ctypes.sizeof(rips.RipsStats) == 15 * 8 + 4 * 4
    assert ctypes.sizeof(rips.RipsTimings) == 13 * 4
    text = open(os.path.join(ROOT, "include", "rips.h")).read()
    stats = re.search(r"typedef struct \{(.*?)\} rips_stats_t;", text, flags=re.S).group(1)
    stats = re.sub(r"/\*.*?\*/", "", stats, flags=re.S)
    fields = re.findall(r"int(?:64|32)_t\s+([a-z_0-9]+);", stats)
    assert fields == [f for f, _ in rips.RipsStats._fields_]
    tim = re.search(r"typedef struct \{(.*?)\} rips_timings_t;", text, flags=re.S).group(1)
    tim = re.sub(r"/\*.*?\*/", "", tim, flags=re.S)
    assert re.findall(r"float\s+([a-z_0-9]+);", tim) == [f for f, _ in rips.RipsTimings._fields_]


def test_host_only_error_paths(lib):
    from paper_2003_07989_b200 import rips
    b = ctypes.c_int64()
    assert lib.rips_workspace_bytes(192, 3, ctypes.byref(b)) == rips.RIPS_OK and b.value > 0
    assert lib.rips_workspace_bytes(0, 3, ctypes.byref(b)) == rips.RIPS_EINVAL
    assert lib.rips_workspace_bytes(60000, 4, ctypes.byref(b)) == rips.RIPS_EOVERFLOW
    assert lib.rips_strerror(rips.RIPS_ECUDA).decode() == "CUDA error"
    h = ctypes.c_void_p()
    assert lib.rips_init(ctypes.byref(h), None, 0, 1, 1.0, None, 0, None) == rips.RIPS_EINVAL
    assert lib.rips_init(ctypes.byref(h), None, 5, 9, 1.0, None, 0, None) == rips.RIPS_EINVAL
    assert lib.rips_last_required_bytes() == 0
    assert lib.rips_compute(None) == rips.RIPS_EINVAL


def test_no_cpu_fallback_without_a_device(lib):
    """On a machine without a GPU the product fails loudly instead of computing on the host."""
    import numpy as np
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2003_07989_b200 import rips
    with pytest.raises(rips.RipsError) as e:
        rips.Rips(np.ones(3, dtype=np.float32), 3, 1)
    assert e.value.code == rips.RIPS_ECUDA


def test_product_does_not_import_the_oracle():
    """Neither side imports, includes or loads the other (comments may name it)."""
    pkg = os.path.join(ROOT, "paper_2003_07989_b200")
    bad = re.compile(r'^\s*(from|import)\s+oracle\b|#\s*include\s*[<"][^>"]*oracle|liboracle|oracle\.(lib|build|barcodes|stage)',
                     re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not bad.search(src), os.path.join(dirpath, f)
    ora = os.path.join(ROOT, "oracle")
    for f in os.listdir(ora):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ora, f)).read()
            assert not re.search(r'^\s*(from|import)\s+paper_2003_07989_b200(?!\.inputs|\s+import\s+inputs)|#\s*include\s*[<"][^>"]*(rips\.h|csrc)|librips',
                                 src, re.M), f
