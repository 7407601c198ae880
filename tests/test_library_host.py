"""CPU-side checks of the CUDA library: it loads, exports every symbol include/sas.h declares,
validates descriptors, builds the same quadrature rules as the oracle (two independent
constructions: Sturm bisection + Christoffel numbers vs numpy eigh), and fails loudly -- never
falls back -- when no device is present."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import sas_workloads as W
from oracle import oracle as O
from paper_2501_06054_b200 import binding as B
from paper_2501_06054_b200 import build as libbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    libbuild.build()
    return B.load_library()


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "sas.h")).read()
    declared = set(re.findall(r"\b(sas_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(B.EXPORTED_SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.sas_version()


def test_struct_layouts_match_the_header(lib):
    # sizes the C compiler gives for the header's structs
    import subprocess, tempfile
    src = ('#include "sas.h"\n#include <stdio.h>\nint main(){printf("%zu %zu %zu %zu\\n", sizeof(sas_instrument_desc), '
           'sizeof(sas_model_desc), sizeof(sas_radial_desc), sizeof(sas_launch_record));return 0;}\n')
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "t.c"), "w").write(src)
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", os.path.join(d, "t"), os.path.join(d, "t.c")])
        a, b, r, l = map(int, subprocess.check_output([os.path.join(d, "t")]).split())
    assert a == C.sizeof(B.InstrumentDesc) and b == C.sizeof(B.ModelDesc)
    assert r == C.sizeof(B.RadialDesc) and l == C.sizeof(B.LaunchRecord)


def test_quadrature_rules_agree_with_the_oracles(lib):
    for p, n in ((0.15, 32), (0.1, 16), (0.3, 64), (0.05, 5), (0.5, 40)):
        s, w = B.quadrature_nodes("schulz", p, n)
        so, wo = O.schulz_nodes(p, n)
        assert np.allclose(s, so, rtol=2e-13, atol=0)
        assert np.allclose(w, wo, rtol=1e-9, atol=1e-16)   # eigh resolves tiny weights only absolutely
        assert abs(w.sum() - 1) < 1e-14 and abs((w * s).sum() - 1) < 1e-13
        assert abs((w * s * s).sum() - (1 + p * p)) < 1e-13
    for sig, n in ((np.radians(10), 24), (0.3, 64), (0.01, 7)):
        d, w = B.quadrature_nodes("gauss_tilt", sig, n)
        do, wo = O.gauss_tilts(sig, n)
        assert np.allclose(d, do, rtol=0, atol=2e-15 * 3 * sig * 10)
        assert np.allclose(w, wo, rtol=1e-11, atol=1e-300)
    s, w = B.quadrature_nodes("schulz", 0.0, 4)      # degenerate: one node of weight 1
    assert s[0] == 1.0 and w[0] == 1.0 and w[1:].sum() == 0.0


def test_bad_descriptors_are_rejected_without_touching_a_device(lib):
    ctx = C.c_void_p()
    ins = B.instrument_desc(W.instrument())
    ins.struct_size = 8
    assert lib.sas_create_instrument(C.byref(ins), C.byref(ctx)) == 1
    assert b"struct_size" in lib.sas_last_error(None)
    for bad in (dict(q_min=0.3, q_max=0.1), dict(lambda_min=0.0), dict(det_nx=0), dict(sample_shape=7),
                dict(focus_z=0.0), dict(slit2_xw=-1.0)):
        d = W.instrument(**bad)
        ins = B.instrument_desc(d)
        assert lib.sas_create_instrument(C.byref(ins), C.byref(ctx)) == 1, bad
    v = (C.c_double * 4)()
    assert lib.sas_quadrature_nodes(0, 1.5, 4, v, v) == 1
    assert lib.sas_quadrature_nodes(3, 0.1, 4, v, v) == 1
    assert lib.sas_quadrature_nodes(0, 0.1, 65, v, v) == 1


def test_no_device_means_an_error_not_a_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    ctx = C.c_void_p()
    ins = B.instrument_desc(W.instrument())
    assert lib.sas_create_instrument(C.byref(ins), C.byref(ctx)) == 3      # SAS_ECUDA
    assert not ctx.value
    with pytest.raises(B.SasError):
        B.Tracer(W.instrument(), W.model())


def test_product_code_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2501_06054_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
                assert "sas_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2501_06054_b200 import" not in txt and "libsas_b200" not in txt, f
            assert "import paper_2501_06054_b200" not in txt, f
