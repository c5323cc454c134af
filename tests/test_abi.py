"""Host-side checks that need no GPU: libkcs.so builds for sm_100a, loads, and exports every symbol that
include/kcs.h declares; the Python binding's struct mirrors the header; the product path refuses to run
without a CUDA device (no CPU fallback); the product never imports the oracle."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_functions(name="kcs.h"):
    src = open(os.path.join(ROOT, "include", name)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(kcs_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import paper_1803_10045_b200 as kcs
    lib = kcs.load()
    names = _header_functions()
    assert {"kcs_forward_project", "kcs_back_project", "kcs_osl_update", "kcs_kinetic_eval", "kcs_map_lm",
            "kcs_icm_iteration"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(kcs.EXPORTS) == names
    assert "kcs_probe_peak" not in names  # measuring tools are not part of the product ABI


def test_every_header_has_its_library():
    """include/ holds kcs.h (libkcs.so, the product) and kcs_probe.h (libkcs_probe.so, bench-only peak probes)."""
    from paper_1803_10045_b200 import build as kb
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["kcs.h", "kcs_probe.h"]
    lib = ctypes.CDLL(kb.build_probe())
    for n in _header_functions("kcs_probe.h"):
        assert hasattr(lib, n), n


def test_built_for_sm_100a():
    import subprocess

    import paper_1803_10045_b200 as kcs
    kcs.load()
    out = subprocess.run(["cuobjdump", "-lelf", kcs.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_config_struct_matches_header():
    """Field order of the ctypes mirror == field order of kcs_config in the header."""
    import paper_1803_10045_b200 as kcs
    src = open(os.path.join(ROOT, "include", "kcs.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} kcs_config;", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        names = decl.split(None, 1)[1] if not decl.startswith("const") else decl.split(None, 2)[2]
        if decl.startswith("const unsigned"):
            names = decl.split(None, 3)[3]
        for n in names.split(","):
            fields.append(re.sub(r"[\*\s]|\[\d+\]", "", n))
    assert fields == [f[0] for f in kcs._Config._fields_]


def test_no_cpu_fallback():
    import torch

    import kcs_inputs as ki
    import paper_1803_10045_b200 as kcs
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError):
        kcs.Context(ki.small_config())
    # straight through the C ABI: kcs_create must fail with KCS_ERR_CUDA, not compute on the host
    lib = kcs.load()
    import numpy as np
    cfg = ki.small_config()
    c = kcs._Config()
    for k in ("nx", "ny", "nz", "n_angles", "n_bins", "n_steps", "n_subsets"):
        setattr(c, k, int(cfg[k]))
    for k in ("vx", "vy", "vz", "bin_mm", "step_mm"):
        setattr(c, k, float(cfg[k]))
    ts = np.ascontiguousarray(cfg["t_start_min"])
    te = np.ascontiguousarray(cfg["t_end_min"])
    c.n_frames = len(ts)
    c.t_start_min = ts.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
    c.t_end_min = te.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
    c.feng_A = (ctypes.c_float * 3)(*cfg["feng_A"])
    c.feng_lambda = (ctypes.c_float * 3)(*cfg["feng_lambda"])
    h = ctypes.c_void_p()
    rc = lib.kcs_create(ctypes.byref(h), ctypes.byref(c), None)
    assert rc == -5 and not h.value
    assert b"no CUDA device" in lib.kcs_last_error(None)


def test_product_and_oracle_are_independent():
    """Neither side imports or includes the other (prompt section 3)."""
    pkg = os.path.join(ROOT, "paper_1803_10045_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                assert "kcs_oracle" not in s and "import oracle" not in s and "from oracle" not in s, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            s = open(os.path.join(ROOT, "oracle", f)).read()
            assert "include/kcs.h" not in s and "import paper_1803_10045_b200" not in s and "libkcs.so" not in s, f
    s = open(os.path.join(ROOT, "kcs_inputs", "__init__.py")).read()
    assert "import oracle" not in s and "paper_1803_10045_b200" not in s
