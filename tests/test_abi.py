"""The C-ABI library loads and exports every symbol include/ile.h declares; argument checking that needs no GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1902_04934_b200 import build as b

    b.build()
    import paper_1902_04934_b200 as ile

    return ile.load()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "ile.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ile_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = declared_symbols()
    assert {"ile_create", "ile_eval", "ile_eval_all", "ile_evidence", "ile_status", "ile_destroy", "ile_strerror",
            "ile_run_host"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/ile.h but not exported"


def test_binding_lists_every_export():
    import paper_1902_04934_b200 as ile

    assert sorted(ile.EXPORTS) == declared_symbols()


def test_strerror_and_bad_arguments(lib):
    assert lib.ile_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4, -5, -99):
        assert len(lib.ile_strerror(code)) > 0
    # NULL arguments are rejected before any CUDA call
    assert lib.ile_create(None, None, None, None, None) == -1
    assert lib.ile_eval(None, 0, 10, *([None] * 7), None, None, None) == -1
    assert lib.ile_evidence(None, 1, 10, None, None, None, None, None, None) == -1
    assert lib.ile_status(None, None, 0, None) == -1
    assert lib.ile_set_variant(None, 0) == -1
    assert lib.ile_launch_count(None) == 0
    lib.ile_destroy(None)  # no-op


def test_create_validates_config_before_touching_the_device(lib):
    import ile_inputs as gi
    import paper_1902_04934_b200 as ile

    cfg = gi.make_config(0, n=4)
    bad = dict(cfg)
    bad["n_t"] = cfg["n_q"] + 1
    with pytest.raises(ile.IleError) as ei:
        ile.Context(bad)
    assert ei.value.code == -1
    bad = dict(cfg)
    bad["l"] = np.array([1, 2], dtype=np.int32)  # l < 2 has no spin-weight -2 harmonic
    with pytest.raises(ile.IleError) as ei:
        ile.Context(bad)
    assert ei.value.code == -1
    bad = dict(cfg)
    bad["fs_hz"] = 0.0
    with pytest.raises(ile.IleError) as ei:
        ile.Context(bad)
    assert ei.value.code == -1


def test_no_device_is_an_error_not_a_fallback(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is visible")
    import ile_inputs as gi
    import paper_1902_04934_b200 as ile

    with pytest.raises(ile.IleError) as ei:
        ile.Context(gi.make_config(0, n=4))
    assert ei.value.code == -3
    tf, ms = ctypes.c_double(), ctypes.c_double()
    assert lib.ile_measure_fp64_peak(16, ctypes.byref(tf), ctypes.byref(ms)) == -3


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or any CPU fallback), and the oracle must not use the
    product: no import / #include in either direction."""
    imp_oracle = re.compile(r"^\s*(import|from)\s+oracle\b|^\s*#\s*include\s+[\"<].*oracle", re.M)
    imp_product = re.compile(r"^\s*(import|from)\s+paper_1902_04934_b200\b|^\s*#\s*include\s+[\"<].*(csrc|ile\.h)", re.M)
    pkg = os.path.join(ROOT, "paper_1902_04934_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not imp_oracle.search(open(os.path.join(dirpath, f)).read()), f
    for f in os.listdir(os.path.join(ROOT, "ile_inputs")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "ile_inputs", f)).read()
            assert not imp_oracle.search(src) and not imp_product.search(src), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            assert not imp_product.search(open(os.path.join(ROOT, "oracle", f)).read()), f
