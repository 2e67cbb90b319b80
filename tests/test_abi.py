"""CPU-side checks of the boundary: libphotons.so loads and exports every symbol include/photons.h declares,
the ctypes structs match the header, and without a CUDA device the product path fails loudly (no fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2107_14008_b200 import build, binding
    build.build()
    return binding.load()


def _header():
    src = open(os.path.join(ROOT, "include", "photons.h")).read()
    return re.sub(r"/\*.*?\*/", "", src, flags=re.S)


def _declared():
    return sorted(set(re.findall(r"\b(photons_[a-z0-9_]+)\s*\(", _header())))


def test_header_symbols_are_exported(lib):
    from paper_2107_14008_b200 import binding
    names = _declared()
    assert {"photons_create", "photons_set_particles", "photons_build_leaves", "photons_short_range_acc",
            "photons_destroy"} <= set(names)
    for name in names:
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == names


def test_struct_layouts_match_header(lib):
    from paper_2107_14008_b200 import binding
    src = _header()
    for cname, cls in (("photons_params", binding.Params), ("photons_stats", binding.Stats)):
        body = re.search(r"typedef struct \{([^{}]*)\} " + cname + ";", src).group(1)
        fields = []
        for decl in body.split(";"):
            decl = decl.strip()
            if not decl:
                continue
            m = re.match(r"(long long|double|int)\s+(.*)", decl)
            ctype = {"long long": ctypes.c_longlong, "double": ctypes.c_double, "int": ctypes.c_int}[m.group(1)]
            for name in m.group(2).split(","):
                fields.append((name.strip(), ctype))
        assert [(n, t) for n, t in cls._fields_] == fields


def test_default_params_are_the_papers(lib):
    from paper_2107_14008_b200 import binding
    p = binding.default_params()
    assert (p.boxsize, p.n_pm, p.rs_over_cell, p.rcut_over_rs, p.G, p.maxleaf) == (1.0, 32, 1.2, 6.0, 1.0, 32)
    assert p.table_nodes == 512 and p.table_level == 2


def test_parameter_validation_needs_no_device(lib):
    # argument checks come before device selection: they answer EINVAL / EBOX on a CPU-only box too
    from paper_2107_14008_b200 import binding as B
    for bad, code in ((dict(maxleaf=48), B.EINVAL), (dict(n_pm=8), B.EBOX), (dict(precision=9), B.EINVAL),
                      (dict(boxsize=0.0), B.EINVAL), (dict(g_mode="table", table_level=7), B.EINVAL)):
        with pytest.raises(B.PhotonsError) as e:
            B.Photons(**bad)
        assert e.value.code == code


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2107_14008_b200 import binding as B
    with pytest.raises(B.PhotonsError) as e:
        B.Photons()
    assert e.value.code == B.ENODEVICE
    out = ctypes.c_double()
    assert lib.photons_peak_probe(0, 0, ctypes.byref(out)) != B.OK


def test_generated_m2l_header_is_in_sync_with_its_generator():
    import importlib.util
    path = os.path.join(ROOT, "paper_2107_14008_b200", "csrc", "gen_m2l.py")
    spec = importlib.util.spec_from_file_location("gen_m2l", path)
    gen = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(gen)
    assert open(os.path.join(os.path.dirname(path), "m2l_generated.cuh")).read() == gen.render()


def test_m2l_argument_checks_need_no_device(lib):
    import numpy as np
    from paper_2107_14008_b200 import binding as B
    c = np.zeros((2, 3)); c[1, 0] = 1.0
    ptr = np.array([0, 1, 1], dtype=np.int64)
    src = np.array([1], dtype=np.int32)
    with pytest.raises(B.PhotonsError) as e:
        B.m2l(c, np.zeros((2, B.m2l_n_coeffs(5))), ptr, src, p=5, r_s=0.1)        # order above 4
    assert e.value.code == B.EINVAL
    with pytest.raises(B.PhotonsError) as e:
        B.m2l(c, np.zeros((2, 4)), ptr, src, p=1, r_s=-1.0)
    assert e.value.code == B.EINVAL
    with pytest.raises(ValueError):
        B.m2l(c, np.zeros((2, 5)), ptr, src, p=1, r_s=0.1)
    assert [B.m2l_n_coeffs(p) for p in range(5)] == [1, 4, 10, 20, 35]


def test_product_does_not_touch_the_oracle():
    # the CUDA path and its binding never import, read or link anything under oracle/ (and vice versa)
    pkg = os.path.join(ROOT, "paper_2107_14008_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) in ("build", "__pycache__"):
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "p2p_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2107_14008_b200", text, flags=re.M), f
            assert '#include "' not in text, f
