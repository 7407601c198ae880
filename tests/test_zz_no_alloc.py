"""sas_reduce_radial_static (include/sas.h): the ring average for callers that must not allocate (CUDA graph capture,
tight serving loops, harnesses that forbid cudaMalloc) -- static device scratch of SAS_STATIC_MAX_RINGS rings, device
inputs and outputs, no allocation inside the library.  Checked against the existing path, sas_reduce_radial, within
the tolerance the ring-average tests use (q and pixel counts exactly, I and sigma to 1e-12), on calls in a row that
share the static scratch.  Collected last on purpose (the suite runs with pytest -x)."""
import os
import re

import numpy as np
import pytest

import sas_workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
STATIC_MAX_RINGS = 512


@pytest.fixture(scope="module")
def sas():
    import paper_2501_06054_b200 as S
    from paper_2501_06054_b200 import build
    build.build()
    S.load_library()
    return S


def test_the_static_entry_point_contains_no_allocating_call():
    src = open(os.path.join(ROOT, "paper_2501_06054_b200", "csrc", "reduce_static.cu")).read()
    code = re.sub(r"//[^\n]*", "", src)                       # comments name the calls it avoids
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaEventCreate", "cudaStreamCreate", "std::vector", " new ", "malloc("):
        assert banned not in code, banned
    assert "static __device__ __align__(256)" in code and "cudaGetSymbolAddress" in code
    hdr = open(os.path.join(ROOT, "include", "sas.h")).read()
    assert f"#define SAS_STATIC_MAX_RINGS {STATIC_MAX_RINGS}" in hdr


@pytest.mark.gpu
def test_static_ring_average_equals_the_existing_path_on_calls_in_a_row(sas):
    import torch
    # two different images: c1's polydisperse spheres on 256 x 256 pixels, a rod on a 128 x 96 detector further away
    ca = W.config(1)
    ins_a, n_a = ca["instrument"], 6 * 10**6
    ins_b = W.instrument(det_nx=128, det_ny=96, det_dist=5.0, det_xw=0.5, det_yh=0.375)
    mod_b = W.model(model="cylinder", precision="fp64", size=[30.0, 300.0, 0, 0], orient_kind="isotropic_mc")
    n_b = 4 * 10**6
    ta, tb = sas.Tracer(ins_a, ca["model"]), sas.Tracer(ins_b, mod_b)
    ta.trace(n_a, ca["seed"])
    tb.trace(n_b, 77)
    cases = [(ta, ins_a, n_a, 6.0, 0.0, 0.08, 200), (tb, ins_b, n_b, 5.4, 0.002, 0.05, 64), (ta, ins_a, n_a, 6.0, 0.0, 0.08, 200),
             (tb, ins_b, n_b, 6.6, 0.001, 0.04, STATIC_MAX_RINGS), (ta, ins_a, n_a, 6.3, 0.01, 0.07, 1)]
    # the existing path first (it allocates its own scratch and synchronises)
    want = [tr.reduce_radial(lam, q_lo, q_hi, nb) for tr, _, _, lam, q_lo, q_hi, nb in cases]
    # caller-owned device outputs, made before the calls; then every call back to back on one stream, no
    # synchronisation in between: each must clear what the one before left in the shared static scratch
    outs = [tuple(torch.full((nb,), -1, dtype=dt, device="cuda") for dt in (torch.float64, torch.float64, torch.float64, torch.int64))
            for *_, nb in cases]
    sas.reduce_radial_static(ins_a, ta.sum_p[0], ta.sum_p2[0], n_a, 6.0, 0.0, 0.08, 8)     # once-per-device set-up, module load
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for (tr, ins, n, lam, q_lo, q_hi, nb), out in zip(cases, outs):
        got = sas.reduce_radial_static(ins, tr.sum_p[0], tr.sum_p2[0], n, lam, q_lo, q_hi, nb, out=out)
        assert got is out
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before          # nothing was allocated on the device
    for k, ((q, I, s, n), out) in enumerate(zip(want, outs)):
        gq, gI, gs, gn = (t.cpu().numpy() for t in out)
        assert np.array_equal(gq, q), k
        assert np.array_equal(gn.view(np.uint64), n), k
        m = I > 0
        assert m.sum() >= 1 and np.all(gI[~m] == 0) and np.all(gs[~m] == 0), k
        assert np.abs(gI[m] / I[m] - 1).max() < 1e-12 and np.abs(gs[m] / s[m] - 1).max() < 1e-12, k
    # the inputs are not modified, and the existing path still gives what it gave
    q, I, s, n = ta.reduce_radial(6.0, 0.0, 0.08, 200)
    assert np.array_equal(n, want[0][3]) and np.allclose(I, want[0][1], rtol=1e-12, atol=0)
    ta.close()
    tb.close()


@pytest.mark.gpu
def test_static_ring_average_refuses_what_does_not_fit(sas):
    import torch
    ins = W.instrument(det_nx=64, det_ny=64)
    img = torch.ones(64, 64, dtype=torch.float64, device="cuda")
    with pytest.raises(sas.SasError) as err:
        sas.reduce_radial_static(ins, img, img, 1000, 6.0, 0.0, 0.08, STATIC_MAX_RINGS + 1)
    assert err.value.status == 1 and "SAS_STATIC_MAX_RINGS = 512" in str(err.value)
    with pytest.raises(sas.SasError) as err:
        sas.reduce_radial_static(ins, img, img, 0, 6.0, 0.0, 0.08, 16)
    assert err.value.status == 1 and "n_launched" in str(err.value)
    with pytest.raises(sas.SasError):
        sas.reduce_radial_static(ins, img, img, 1000, 6.0, 0.05, 0.01, 16)
    # a valid call after the refusals: a constant image gives I = sum P / (sum dOmega * launched) ring by ring
    q, I, s, n = (t.cpu().numpy() for t in sas.reduce_radial_static(ins, img, img, 1000, 6.0, 0.0, 0.08, 16))
    assert n.sum() > 0 and np.all(I[n > 0] > 0) and np.all(I[n == 0] == 0)
