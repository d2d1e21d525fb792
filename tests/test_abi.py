"""The C-ABI library loads and exports every symbol include/tofmlem.h declares (no GPU, no compute calls)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "tofmlem.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tofmlem_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_exported():
    import paper_1706_07075_b200 as pkg

    L = pkg.lib()
    declared = _declared_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(L, name), f"{name} declared in include/tofmlem.h but not exported"
    assert sorted(pkg.SYMBOLS) == declared  # the binding knows every call
    assert b"sm_100a" in L.tofmlem_version()


def test_struct_layouts_match_header():
    import paper_1706_07075_b200 as pkg

    assert ctypes.sizeof(pkg.Grid) == 36 and ctypes.sizeof(pkg.Scanner) == 8
    assert ctypes.sizeof(pkg.Events) == 7 * ctypes.sizeof(ctypes.c_void_p)
    assert ctypes.sizeof(pkg.Stats) == 64 and ctypes.sizeof(pkg.Plan) == 40


def test_argument_errors_without_gpu():
    """NULL / invalid arguments are rejected before any CUDA work."""
    import paper_1706_07075_b200 as pkg

    L = pkg.lib()
    assert L.tofmlem_create(None, None, ctypes.c_float(300.0), None, None) == -1
    h = ctypes.c_void_p()
    g = pkg.make_grid(0, 4, 4, 2.0)
    sc = pkg.Scanner(100.0, 100.0)
    assert L.tofmlem_create(ctypes.byref(sc), ctypes.byref(g), ctypes.c_float(300.0), None, ctypes.byref(h)) == -1
    assert L.tofmlem_destroy(None) == 0
    assert L.tofmlem_num_bins(None) == 0
    assert L.tofmlem_iterate(None, None, ctypes.c_uint64(0), None, None, 1) == -1
    # widened rows: a NULL context is rejected by every entry point
    assert L.tofmlem_iterate_weighted(None, None, ctypes.c_uint64(0), None, None, None, 1) == -1
    assert L.tofmlem_em_correction_weighted(None, None, ctypes.c_uint64(0), None, None, None) == -1
    assert L.tofmlem_median3(None, None, None) == -1
    assert L.tofmlem_attenuation_weights(None, None, ctypes.c_uint64(0), None, None) == -1
    assert L.tofmlem_gather_f32(None, None, None, ctypes.c_uint64(0), None) == -1
    assert L.tofmlem_scatter_reject(None, None, ctypes.c_uint64(0), None, 1, ctypes.c_float(0.0), None, None, None) == -1


def test_no_cpu_fallback():
    import torch

    import paper_1706_07075_b200 as pkg

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        pkg.Context(200.0, 128.0, pkg.make_grid(8, 8, 8, 4.0), 300.0)


def test_product_does_not_import_oracle():
    """The product path and the oracle share nothing and neither imports the other."""
    for base, banned in (("paper_1706_07075_b200", ("oracle", "synth")), ("oracle", ("paper_1706_07075_b200", "synth")),
                         ("synth", ("oracle", "paper_1706_07075_b200"))):
        for dirpath, _, files in os.walk(os.path.join(ROOT, base)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".c", ".h")):
                    src = open(os.path.join(dirpath, f)).read()
                    for b in banned:
                        assert not re.search(rf"^\s*(from|import)\s+{b}\b", src, flags=re.M), (f, b)
                        assert f'#include "{b}' not in src
