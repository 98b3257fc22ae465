"""The C-ABI library loads and exports every symbol include/hlb.h declares; the metric is
the paper's SUPS definition. No compute calls (this file runs without a GPU)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1906_11925_b200 as hlb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "hlb.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = re.findall(r"\b(hlb_[a-z_]+)\s*\(", text)
    return sorted(set(n for n in names if n != "hlb_alloc_fn"))


def test_header_symbols_are_exported():
    lib = ctypes.CDLL(hlb.LIB_PATH)
    names = declared_functions()
    assert len(names) >= 16
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/hlb.h but not exported"
    assert sorted(hlb.EXPORTED) == names          # the binding wraps exactly the header


def test_no_torch_or_cpp_types_in_signatures():
    text = open(os.path.join(ROOT, "include", "hlb.h")).read()
    code = re.sub(r"/\*.*?\*/", "", text, flags=re.S)            # declarations without comments
    assert "torch" not in code.lower() and "std::" not in code and "at::" not in code
    assert 'extern "C"' in code


def test_errors_without_a_device_or_with_bad_arguments():
    st = np.ones((2, 2, 2), dtype=np.uint8)
    p = hlb.hlb_params()
    p.nx = p.ny = p.nz = 2
    p.tau = 0.4                                     # invalid tau is reported before any CUDA call
    out = ctypes.c_void_p()
    lib = ctypes.CDLL(hlb.LIB_PATH)
    lib.hlb_geometry_create.restype = ctypes.c_int
    lib.hlb_last_error.restype = ctypes.c_char_p
    rc = lib.hlb_geometry_create(st.ctypes.data_as(ctypes.c_void_p), ctypes.byref(p), ctypes.byref(out))
    assert rc == hlb.HLB_EINVAL and out.value is None
    assert b"tau" in lib.hlb_last_error()
    assert lib.hlb_geometry_create(None, ctypes.byref(p), ctypes.byref(out)) == hlb.HLB_EINVAL
    p.tau = 0.8
    p.n_iolets = 1
    bad_rho = (ctypes.c_double * 1)(-1.0)                 # a density must be positive
    p.iolet_rho = ctypes.cast(bad_rho, ctypes.c_void_p)
    assert lib.hlb_geometry_create(st.ctypes.data_as(ctypes.c_void_p), ctypes.byref(p), ctypes.byref(out)) == hlb.HLB_EINVAL
    assert b"positive" in lib.hlb_last_error()
    lib.hlb_num_sites.restype = ctypes.c_int64
    assert lib.hlb_num_sites(None) == hlb.HLB_EINVAL
    lib.hlb_geometry_destroy(None)                  # NULL is a no-op


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(hlb.HlbError) as e:
        hlb.hlb_geometry_create(np.ones((2, 2, 2), dtype=np.uint8), 7, 0.8)
    assert e.value.code == hlb.HLB_ECUDA


def test_sups_reproduces_the_papers_table():
    """Table III = sites x steps / seconds from Table II."""
    rows = [l for l in open(os.path.join(ROOT, "tests", "golden", "paper_tables_II_III.txt"))
            if not l.startswith("#")]
    assert len(rows) == 2
    for line in rows:
        name, sites, blocks, secs, steps, sups = [s.strip() for s in line.split(",")]
        assert int(hlb.sups(int(sites), int(steps), float(secs))) == int(sups)
        assert hlb.msups(int(sites), int(steps), float(secs)) == pytest.approx(int(sups) / 1e6, rel=1e-7)


def test_bytes_per_site_model():
    assert hlb.algorithmic_bytes_per_site("two_lattice", "f64") == 15 * 8 * 2 + 14 * 4
    assert hlb.algorithmic_bytes_per_site("aa", "f64") == 15 * 8 * 2 + 14 * 4 / 2
    assert hlb.algorithmic_bytes_per_site("two_lattice", "f32") == 15 * 4 * 2 + 14 * 4
    assert hlb.algorithmic_bytes_per_site("aa", "f32") == 15 * 4 * 2 + 14 * 4 / 2
    assert hlb.algorithmic_bytes_per_site("two_lattice", "f64", 19) == 19 * 8 * 2 + 18 * 4   # 376
    assert hlb.algorithmic_bytes_per_site("aa", "f64", 19) == 19 * 8 * 2 + 18 * 4 / 2
    assert hlb.algorithmic_bytes_per_site("two_lattice", "f32", 19) == 19 * 4 * 2 + 18 * 4


def test_moved_bytes_model():
    """What the selected variant really reads and writes (bench.py roofline.frac_moved_model)."""
    m = hlb.moved_bytes_per_site
    assert m("two_lattice", "f64", 15, records=False) == 240 + 56 + 0.125
    assert m("two_lattice", "f64", 15, records=True, sentinel_fraction=0.0) == 240 + 7 + 0.125
    assert m("two_lattice", "f64", 15, records=True, sentinel_fraction=0.5) == 240 + 7 + 28 + 0.125
    assert m("aa", "f64", 15, records=True, phase="even") == 240 + 0.125
    assert m("aa", "f64", 15, records=True, phase="odd") == 240 + 7 + 0.125
    assert m("aa", "f64", 15, records=True) == 240 + 3.5 + 0.125
    assert m("aa", "f32", 19, records=False, phase="odd") == 152 + 72 + 0.125
    # interpolated walls: one index word per 32 sites, one 64-byte (D3Q19: 80-byte) row per flagged site
    assert m("aa", "f64", 15, phase="even", bfl_site_fraction=0.25) == 240 + 0.125 + 0.25 + 16
    assert m("two_lattice", "f64", 19, bfl_site_fraction=0.5) == 304 + 9 + 0.125 + 0.25 + 40
