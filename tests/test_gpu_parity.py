"""Parity of the CUDA path (through the C ABI) with the CPU oracle on the same seeded inputs.

Per neutron: detector pixel bit-exact, drawn |Q| bit-exact, weight within
    |dp| <= tol * max(|p_oracle|, 1e-4 * p_env),  tol = 1e-12 (fp64 model) / 1e-5 (fp32 model)
where p_env is the oracle's weight with every shape factor set to 1 (DESIGN.md R-C15: a purely
relative bound cannot hold at a form-factor zero in any finite precision).
Per histogram: counts exact, bins within 1e-9 relative (fp64), counters exact."""
import math

import numpy as np
import pytest

import sas_workloads as W
from oracle import oracle as O

pytestmark = pytest.mark.gpu

TOL = {"fp64": 1e-12, "fp32": 1e-5}


@pytest.fixture(scope="module")
def sas():
    import paper_2501_06054_b200 as S
    from paper_2501_06054_b200 import build
    build.build()
    S.load_library()
    return S


def check_dump(sas, ins, model, seed, first, n, exp_index=0, tol=None, min_detected=1):
    tol = tol or TOL[model["precision"]]
    tr = sas.Tracer(ins, model)
    px, wt, qq = tr.trace_dump(first, n, seed, exp_index)
    tr.close()
    ref = O.trace_range(ins, model, seed, first, n, exp_index=exp_index, hist=False)
    assert np.array_equal(px, ref["pixel"]), f"{(px != ref['pixel']).sum()} pixel mismatches"
    # the oracle reports q for every neutron that reached the draw; the library likewise
    reached = ref["q"] > 0
    assert np.array_equal(qq[reached], ref["q"][reached])
    det = ref["pixel"] >= 0
    assert det.sum() >= min_detected
    assert np.all(wt[~det] == 0.0)
    bound = tol * np.maximum(np.abs(ref["weight"][det]), 1e-4 * np.abs(ref["weight_env"][det]))
    err = np.abs(wt[det] - ref["weight"][det])
    worst = float((err / bound).max())
    print(f"[parity] worst weight error {worst:.3g} x tolerance (tol {tol:g}, {int(det.sum())} detected)")
    assert worst <= 1.0, f"worst weight error {worst:.3g} x tolerance"
    return worst


def assert_bins(got, ref, key, tol, what=""):
    """R-C16 with R-C15's floor: |bin - oracle bin| <= tol * max(oracle bin, 1e-4 * envelope bin), the envelope bin
    being the sum of the oracle's weights with every shape factor set to 1 (a bin that holds one hit at a
    form-factor zero cannot meet a purely relative bound in any precision, exactly as a single weight cannot).
    `ref` is an oracle run with dump and hist."""
    det = ref["pixel"] >= 0
    env = np.zeros(ref[key].size)
    np.add.at(env, ref["pixel"][det], ref["weight_env"][det] ** (2 if key == "sum_p2" else 1))
    bound = tol * np.maximum(np.abs(ref[key]), (1e-4 if key == "sum_p" else 1e-8) * env)
    err = np.abs(got.reshape(-1) - ref[key])
    assert np.all(err <= bound), f"{what}: worst bin error {float((err[bound > 0] / bound[bound > 0]).max()):.3g} x bound"
    assert np.all(got.reshape(-1)[ref[key] == 0] == 0), what


def check_prefix(sas, ins, model, seed, n, exp_index=0, tol=None, min_detected=1, tracer=None):
    """Ids [0, n) of one experiment against ONE oracle run: per neutron (R-C15: pixels and |Q| bit-exact, weights
    within tol) and per histogram (R-C16: counts exact; fp64 model: bins <= 1e-9 of the oracle's; fp32 model: bins
    <= 1e-9 of an fp64 re-accumulation of the library's own dumped weights and <= 1e-5 of the oracle's)."""
    tol = tol or TOL[model["precision"]]
    tr = tracer or sas.Tracer(ins, model)
    px, wt, qq = tr.trace_dump(0, n, seed, exp_index)
    ref = O.trace_range(ins, model, seed, 0, n, exp_index=exp_index)
    assert np.array_equal(px, ref["pixel"]), f"{(px != ref['pixel']).sum()} pixel mismatches"
    reached = ref["q"] > 0
    assert np.array_equal(qq[reached], ref["q"][reached])
    det = ref["pixel"] >= 0
    assert det.sum() >= min_detected and np.all(wt[~det] == 0.0)
    bound = tol * np.maximum(np.abs(ref["weight"][det]), 1e-4 * np.abs(ref["weight_env"][det]))
    worst = float((np.abs(wt[det] - ref["weight"][det]) / bound).max())
    assert worst <= 1.0, f"worst weight error {worst:.3g} x tolerance"
    if tracer is None and exp_index == 0:
        tr.reset()
        tr.trace(n, seed)
        sp, sp2, cn = (a.reshape(-1) for a in tr.read_detector())
        assert np.array_equal(cn, ref["counts"])
        assert np.array_equal(tr.counters()[:7], ref["counters"][:7])
        m = ref["sum_p"] > 0
        assert np.all(sp[~m] == 0)
        if tol <= 1e-11:
            assert_bins(sp, ref, "sum_p", 1e-9)
            assert_bins(sp2, ref, "sum_p2", 1e-9)
        else:
            acc, acc2 = np.zeros(sp.size), np.zeros(sp.size)
            np.add.at(acc, px[det], wt[det])
            np.add.at(acc2, px[det], wt[det] ** 2)
            assert np.abs(sp[m] / acc[m] - 1).max() < 1e-9 and np.abs(sp2[m] / acc2[m] - 1).max() < 1e-9
            assert_bins(sp, ref, "sum_p", 1e-5)
    if tracer is None:
        tr.close()
    print(f"[parity] {int(det.sum())} detected of {n}: worst weight error {worst:.3g} x tolerance ({tol:g})")
    return ref, px, wt


def test_c0_sphere_fp64_per_neutron(sas):
    c = W.config(0)
    check_dump(sas, c["instrument"], c["model"], c["seed"], 0, 10**6, min_detected=40000)


def test_c0_histogram_and_counters(sas):
    c = W.config(0)
    n = c["n_neutrons"]
    tr = sas.Tracer(c["instrument"], c["model"])
    tr.trace(n, c["seed"])
    sp, sp2, cn = tr.read_detector()
    cnt = tr.counters()
    ref = O.trace_range(c["instrument"], c["model"], c["seed"], 0, n, dump=False)
    assert np.array_equal(cnt[:7], ref["counters"][:7])
    assert np.array_equal(cn.reshape(-1), ref["counts"])
    m = ref["sum_p"] > 0
    assert np.all(sp.reshape(-1)[~m] == 0)
    assert np.abs(sp.reshape(-1)[m] / ref["sum_p"][m] - 1).max() < 1e-9
    assert np.abs(sp2.reshape(-1)[m] / ref["sum_p2"][m] - 1).max() < 1e-9
    # the torch-owned buffers the library was bound to hold the same numbers (no hidden copy)
    assert np.array_equal(tr.sum_p.cpu().numpy(), sp)
    # accumulation: a second trace of the next id range adds on top; reset clears
    tr.trace_range(n, 1000, c["seed"])
    assert tr.counters()[0] == n + 1000
    tr.reset()
    assert tr.counters().sum() == 0 and float(tr.sum_p.sum()) == 0.0
    tr.close()


# per-neutron parity on ids [0, 1e6) of every config, histogram parity on the same prefix
@pytest.mark.parametrize("precision", ["fp32", "fp64"])
def test_c1_polydisperse_sphere_py(sas, precision):
    c = W.config(1, precision)
    check_prefix(sas, c["instrument"], c["model"], c["seed"], 10**6, min_detected=40000)


def test_c2_oriented_cylinder_fp32(sas):
    c = W.config(2)
    check_prefix(sas, c["instrument"], c["model"], c["seed"], 10**6, min_detected=100000)


def test_c3_core_shell_triaxial_fp32(sas):
    c = W.config(3)
    check_prefix(sas, c["instrument"], c["model"], c["seed"], 10**6, min_detected=40000)


def test_c4_batch_small(sas):
    c = W.batch_config(12, 30000, 20250110)
    # per neutron, experiment by experiment, with the experiment index in the Philox counter
    for e in (0, 1, 6, 11):
        check_dump(sas, c["instruments"][e], c["models"][e], c["seed"], 0, 30000, exp_index=e, min_detected=100)
    bt = sas.BatchTracer(c["instruments"], c["models"])
    bt.trace(30000, c["seed"])
    sp, sp2, cn = bt.read_detector()
    cnt = bt.counters()
    tot = np.zeros(8, np.uint64)
    for e in range(12):
        ref = O.trace_range(c["instruments"][e], c["models"][e], c["seed"], 0, 30000, exp_index=e)
        tot += ref["counters"]
        assert np.array_equal(cn[e].reshape(-1), ref["counts"]), e
        # monodisperse models are served in fp64 whatever precision was asked: R-C16's fp64 bound
        assert_bins(sp[e], ref, "sum_p", 1e-9, e)
        assert_bins(sp2[e], ref, "sum_p2", 1e-9, e)
    assert np.array_equal(cnt[:7], tot[:7])
    bt.close()


def test_fp32_histogram_is_an_fp64_accumulation_of_the_dumped_weights(sas):
    c = W.config(1, "fp32")
    n = 500000
    tr = sas.Tracer(c["instrument"], c["model"])
    px, wt, _ = tr.trace_dump(0, n, c["seed"])
    tr.trace(n, c["seed"])
    sp, sp2, cn = tr.read_detector()
    tr.close()
    det = px >= 0
    acc = np.zeros(sp.size)
    np.add.at(acc, px[det], wt[det])
    acc2 = np.zeros(sp.size)
    np.add.at(acc2, px[det], wt[det] ** 2)
    m = acc > 0
    assert np.abs(sp.reshape(-1)[m] / acc[m] - 1).max() < 1e-9
    assert np.abs(sp2.reshape(-1)[m] / acc2[m] - 1).max() < 1e-9
    assert np.array_equal(cn.reshape(-1), np.bincount(px[det], minlength=sp.size).astype(np.uint64))
    ref = O.trace_range(c["instrument"], c["model"], c["seed"], 0, n, dump=False)
    assert np.abs(sp.reshape(-1)[m] / ref["sum_p"][m] - 1).max() < 1e-5


MODELS = [
    ("core_shell_sphere_pd", dict(model="core_shell_sphere", size=[40.0, 10.0, 0, 0], sld=[3e-6, 1e-6, 0],
                                  pd_kind=["schulz", "schulz"], pd_rel=[0.1, 0.2], pd_nodes=[12, 7])),
    ("cylinder_fixed_60_60", dict(model="cylinder", size=[20.0, 400.0, 0, 0], theta=math.radians(60), phi=math.radians(60))),
    ("cylinder_pd_iso", dict(model="cylinder", size=[119.0, 800.0, 0, 0], pd_kind=["schulz", "schulz"],
                             pd_rel=[0.05, 0.05], pd_nodes=[8, 8], orient_kind="isotropic_mc")),
    ("cylinder_quad_tilted", dict(model="cylinder", size=[30.0, 150.0, 0, 0], orient_kind="gauss_quad", theta=0.4, phi=1.1,
                                  psi=0.3, sigma_theta=0.1, sigma_phi=0.2, n_theta=9, n_phi=5,
                                  pd_kind=["schulz", "none"], pd_rel=[0.1, 0], pd_nodes=[6, 1])),
    ("triaxial_fixed", dict(model="triaxial", size=[30.0, 50.0, 80.0, 0], theta=0.7, phi=2.0, psi=0.5,
                            pd_kind=["schulz", "none"], pd_rel=[0.1, 0], pd_nodes=[10, 1])),
    ("cs_triaxial_fixed", dict(model="core_shell_triaxial", size=[30.0, 50.0, 80.0, 10.0], sld=[3e-6, 1e-6, 0],
                               theta=1.2, phi=0.3, psi=2.5)),
    ("sphere_bkg_py", dict(model="sphere", size=[80.0, 0, 0, 0], background=0.05, sq_kind="hard_sphere_py",
                           sq_radius_eff=85.0, sq_volfrac=0.3)),
    ("flat", dict(model="flat", scale=2.5, background=0.5)),
]


@pytest.mark.parametrize("precision", ["fp32", "fp64"])
@pytest.mark.parametrize("name,over", MODELS, ids=[m[0] for m in MODELS])
def test_model_library(sas, name, over, precision):
    model = W.model(precision=precision, **over)
    tol = TOL[precision]
    if precision == "fp64" and model["model"] == "cylinder":
        tol = 1e-12
    check_dump(sas, W.instrument(det_dist=3.0), model, 424242, 0, 150000, tol=tol, min_detected=5000)


def test_geometry_variants(sas):
    m = W.config(0)["model"]
    # slit 1 downstream of the source (no integer prefilter), wide focus so that slit 2 cuts
    ins = W.instrument(slit1_z=1.0, slit1_xw=0.004, focus_xw=0.008, focus_yh=0.008)
    ref = O.trace_range(ins, m, 5, 0, 50000, dump=False, hist=False)
    assert ref["counters"][1] > 0 and ref["counters"][2] > 0
    check_dump(sas, ins, m, 5, 0, 200000, min_detected=2000)
    # cylinder sample shorter than the beam: misses; attenuation on
    ins = W.instrument(sample_shape="cyl_y", sample_yh=0.003, mu_abs_2200=20.0, mu_inc=40.0)
    ref = O.trace_range(ins, m, 6, 0, 50000, dump=False, hist=False)
    assert ref["counters"][3] > 0
    check_dump(sas, ins, m, 6, 0, 200000, min_detected=2000)
    # box with attenuation; long wavelength so that some |Q| are unreachable
    ins = W.instrument(mu_abs_2200=5.0, mu_inc=10.0, lambda_min=25.0, lambda_max=30.0, q_max=0.6, det_dist=0.3)
    ref = O.trace_range(ins, m, 7, 0, 50000, dump=False, hist=False)
    assert ref["counters"][4] > 0
    check_dump(sas, ins, m, 7, 0, 200000, min_detected=2000)
    # counters of the general path
    tr = sas.Tracer(W.instrument(slit1_z=1.0, slit1_xw=0.004, focus_xw=0.008, focus_yh=0.008), m)
    tr.trace(50000, 5)
    assert np.array_equal(tr.counters()[:7], O.trace_range(W.instrument(slit1_z=1.0, slit1_xw=0.004, focus_xw=0.008,
                          focus_yh=0.008), m, 5, 0, 50000, dump=False, hist=False)["counters"][:7])
    assert tr.counters()[7] == 0          # slit 1 off the source plane: the classifier must stay off
    tr.close()


def test_edge_cases(sas):
    c = W.config(0)
    tr = sas.Tracer(c["instrument"], c["model"])
    tr.trace(0, 1)                                   # empty
    assert tr.counters().sum() == 0
    for n in (1, 31, 33, 12345):                     # ragged tails
        tr.reset()
        tr.trace(n, c["seed"])
        ref = O.trace_range(c["instrument"], c["model"], c["seed"], 0, n, dump=False)
        assert np.array_equal(tr.counters()[:7], ref["counters"][:7])
        assert np.array_equal(tr.read_detector()[2].reshape(-1), ref["counts"])
    # ranges are additive, and ids above 2^32 use the high counter word
    tr.reset()
    tr.trace_range(0, 70000, c["seed"])
    tr.trace_range(70000, 30000, c["seed"])
    a = tr.read_detector()
    tr.reset()
    tr.trace(100000, c["seed"])
    b = tr.read_detector()
    assert np.array_equal(a[2], b[2]) and np.allclose(a[0], b[0], rtol=1e-12, atol=0)
    tr.close()
    big = (1 << 33) + 12345
    check_dump(sas, c["instrument"], c["model"], c["seed"], big, 100000, min_detected=3000)
    # a range that crosses a multiple of 2^32: the library splits the launch there (dump and histogram paths)
    cross = (1 << 32) - 50001
    check_dump(sas, c["instrument"], c["model"], c["seed"], cross, 100000, min_detected=3000)
    tr = sas.Tracer(c["instrument"], c["model"])
    tr.trace_range(cross, 100000, c["seed"])
    ref = O.trace_range(c["instrument"], c["model"], c["seed"], cross, 100000, dump=False)
    assert np.array_equal(tr.counters()[:7], ref["counters"][:7])
    assert np.array_equal(tr.read_detector()[2].reshape(-1), ref["counts"])
    assert tr.launch_info()["n_launches"] == 2
    tr.close()


def test_slit_narrower_than_the_source_grid(sas):
    """A slit 1 in the source plane that no 32-bit source draw can pass (its aperture is below the spacing of the
    source coordinates, 10 mm / 2^32): every neutron is absorbed at slit 1, as the oracle finds; and a slit that
    passes a handful of words keeps exactly those."""
    c = W.config(0)
    for width, expect_none in ((1.0e-12, True), (2.0e-8, False)):
        ins = dict(c["instrument"], slit1_xw=width)
        n = 3_000_000
        tr = sas.Tracer(ins, c["model"])
        tr.trace(n, c["seed"])
        cnt = tr.counters()
        counts = tr.read_detector()[2]
        tr.close()
        ref = O.trace_range(ins, c["model"], c["seed"], 0, n, dump=False)
        assert np.array_equal(cnt[:7], ref["counters"][:7])
        assert np.array_equal(counts.reshape(-1), ref["counts"])
        assert (cnt[1] == n) == expect_none


def test_error_paths(sas):
    tr = sas.Tracer(W.instrument())
    with pytest.raises(sas.SasError) as e:
        tr.trace(10, 1)
    assert e.value.status == 2
    with pytest.raises(sas.SasError) as e:
        tr.set_model(W.model(model="triaxial", size=[1.0, 2.0, 3.0, 0], orient_kind="gauss_quad", n_theta=3, n_phi=3,
                             sigma_theta=0.1, sigma_phi=0.1))
    assert e.value.status == 5
    with pytest.raises(sas.SasError) as e:
        tr.set_model(W.model(size=[-1.0, 0, 0, 0]))
    assert e.value.status == 1
    tr.close()


def test_certain_miss_classifier_never_changes_an_outcome(sas):
    """Stage B0 decides 'misses the detector' from q*lambda alone when the host can prove it
    (include/sas.h, counters[7]).  Outcomes and pixels must stay those of the oracle in instruments
    where it is busy, idle, and disqualified."""
    m = W.config(0)["model"]
    cases = [
        (W.instrument(), True),                                                   # c0: ~73 % decided early
        (W.instrument(det_dist=10.0, det_xw=0.2, det_yh=0.3), True),              # far, small, non-square detector
        (W.instrument(det_dist=0.4, det_xw=1.0, det_yh=1.0), False),              # everything can hit: idle
        (W.instrument(lambda_min=2.0, lambda_max=12.0), True),                    # wide band: threshold varies 6x
        (W.instrument(sample_shape="cyl_y", det_nx=64, det_ny=32), True),         # cylinder sample
        (W.instrument(focus_xw=0.012, slit2_xw=0.012), False),                    # beam wider than the sample
        (W.instrument(focus_xw=0.006, focus_yh=0.006), False),                    # slit 2 cuts: disqualified
    ]
    for k, (ins, busy) in enumerate(cases):
        n = 300000
        check_dump(sas, ins, m, 31 + k, 0, n, min_detected=100)
        tr = sas.Tracer(ins, m)
        tr.trace(n, 31 + k)
        cnt = tr.counters()
        tr.close()
        ref = O.trace_range(ins, m, 31 + k, 0, n, dump=False, hist=False)["counters"]
        assert np.array_equal(cnt[:7], ref[:7]), (k, cnt, ref)
        assert cnt[7] <= cnt[5]
        assert (cnt[7] > 0) == busy, (k, cnt)


# ---- NEXT-1: the paper's own stochastic averaging (DESIGN.md R-N1..R-N3)
PAPER_SAMPLING = [
    ("sphere_gauss", dict(model="sphere", size=[50.0, 0, 0, 0], pd_kind=["gauss_mc", "none"], pd_rel=[0.15, 0.0])),
    ("sphere_gauss_wide_py", dict(model="sphere", size=[40.0, 0, 0, 0], pd_kind=["gauss_mc", "none"], pd_rel=[0.9, 0.0],
                                  scale=0.2, sq_kind="hard_sphere_py", sq_radius_eff=40.0, sq_volfrac=0.2)),
    ("core_shell_gauss2", dict(model="core_shell_sphere", size=[40.0, 10.0, 0, 0], sld=[3e-6, 1e-6, 0],
                               pd_kind=["gauss_mc", "gauss_mc"], pd_rel=[0.1, 0.6])),
    ("cylinder_paper", dict(model="cylinder", size=[119.0, 800.0, 0, 0], pd_kind=["gauss_mc", "gauss_mc"],
                            pd_rel=[0.05, 0.05], orient_kind="uniform_angles_mc")),
    ("cylinder_gauss_fixed", dict(model="cylinder", size=[20.0, 400.0, 0, 0], pd_kind=["none", "gauss_mc"],
                                  pd_rel=[0.0, 0.2], theta=1.0, phi=0.4)),
    ("triaxial_gauss_iso", dict(model="triaxial", size=[30.0, 50.0, 80.0, 0], pd_kind=["gauss_mc", "none"],
                                pd_rel=[0.1, 0.0], orient_kind="isotropic_mc")),
    ("cs_triaxial_paper", dict(model="core_shell_triaxial", size=[30.0, 50.0, 80.0, 10.0], sld=[3e-6, 1e-6, 0],
                               pd_kind=["gauss_mc", "gauss_mc"], pd_rel=[0.1, 0.1], orient_kind="uniform_angles_mc")),
    ("cylinder_uniform_angles_nodes", dict(model="cylinder", size=[30.0, 150.0, 0, 0], orient_kind="uniform_angles_mc",
                                           pd_kind=["schulz", "none"], pd_rel=[0.1, 0], pd_nodes=[6, 1])),
]


@pytest.mark.parametrize("name,over", PAPER_SAMPLING, ids=[m[0] for m in PAPER_SAMPLING])
def test_paper_sampling_per_neutron(sas, name, over):
    # per-event sizes are one fp64 evaluation per neutron whatever precision is asked for
    precision = "fp32" if name == "cylinder_uniform_angles_nodes" else "fp64"
    model = W.model(precision=precision, **over)
    tol = TOL[precision]
    check_dump(sas, W.instrument(det_dist=3.0), model, 20250111, 0, 150000, tol=tol, min_detected=5000)


def test_paper_sampling_histogram_and_fp32_request(sas):
    ins = W.instrument(det_dist=3.0, det_nx=64, det_ny=64)
    over = dict(PAPER_SAMPLING[3][1])
    n = 300000
    ref = O.trace_range(ins, W.model(precision="fp64", **over), 7, 0, n, dump=False)
    for precision in ("fp64", "fp32"):      # the fp32 request is served by the same fp64 event evaluation
        tr = sas.Tracer(ins, W.model(precision=precision, **over))
        tr.trace(n, 7)
        sp, sp2, cn = tr.read_detector()
        cnt = tr.counters()
        tr.close()
        assert np.array_equal(cnt[:7], ref["counters"][:7]) and np.array_equal(cn.reshape(-1), ref["counts"])
        m = ref["sum_p"] > 0
        assert np.abs(sp.reshape(-1)[m] / ref["sum_p"][m] - 1).max() < 1e-9
        assert np.abs(sp2.reshape(-1)[m] / ref["sum_p2"][m] - 1).max() < 1e-9


def test_paper_sampling_rejects_mixtures(sas):
    ins = W.instrument()
    for over in (dict(model="sphere", pd_kind=["gauss_mc", "none"], pd_rel=[0.1, 0], orient_kind="fixed",
                      size=[50.0, 0, 0, 0]),):
        sas.Tracer(ins, W.model(**over)).close()        # fine on its own
    bad = [dict(model="core_shell_sphere", size=[40.0, 10.0, 0, 0], pd_kind=["gauss_mc", "schulz"], pd_rel=[0.1, 0.1],
                pd_nodes=[1, 8]),
           dict(model="cylinder", size=[20.0, 400.0, 0, 0], pd_kind=["gauss_mc", "none"], pd_rel=[0.1, 0],
                orient_kind="gauss_quad", sigma_theta=0.1, sigma_phi=0.1, n_theta=4, n_phi=4)]
    for over in bad:
        with pytest.raises(sas.SasError) as e:
            sas.Tracer(ins, W.model(**over))
        assert e.value.status == 5                      # SAS_EUNSUPPORTED


# ---- NEXT-2: parallelepiped, core-shell cylinder, ellipsoid of revolution (fp64 node loops)
MORE_MODELS = [
    ("parallelepiped_fixed", dict(model="parallelepiped", size=[35.0, 75.0, 120.0, 0], theta=0.7, phi=2.0, psi=0.5)),
    ("parallelepiped_pd_iso", dict(model="parallelepiped", size=[35.0, 75.0, 120.0, 0], pd_kind=["schulz", "none"],
                                   pd_rel=[0.1, 0], pd_nodes=[8, 1], orient_kind="isotropic_mc")),
    ("cs_cylinder_pd_fixed", dict(model="core_shell_cylinder", size=[20.0, 300.0, 8.0, 0], sld=[3e-6, 1e-6, 0],
                                  pd_kind=["schulz", "schulz"], pd_rel=[0.1, 0.05], pd_nodes=[6, 5], theta=1.0, phi=0.3)),
    ("cs_cylinder_paper", dict(model="core_shell_cylinder", size=[20.0, 300.0, 8.0, 0], sld=[3e-6, 1e-6, 0],
                               pd_kind=["gauss_mc", "gauss_mc"], pd_rel=[0.1, 0.1], orient_kind="uniform_angles_mc")),
    ("ellipsoid_pd_iso_py", dict(model="ellipsoid", size=[30.0, 70.0, 0, 0], pd_kind=["schulz", "schulz"],
                                 pd_rel=[0.1, 0.1], pd_nodes=[5, 7], orient_kind="isotropic_mc",
                                 sq_kind="hard_sphere_py", sq_radius_eff=45.0, sq_volfrac=0.15, background=0.01)),
    ("ellipsoid_paper", dict(model="ellipsoid", size=[30.0, 70.0, 0, 0], pd_kind=["gauss_mc", "none"], pd_rel=[0.2, 0],
                             theta=0.5, phi=1.0)),
    ("barbell_pd_fixed", dict(model="barbell", size=[20.0, 200.0, 40.0, 0], pd_kind=["schulz", "schulz"], pd_rel=[0.1, 0.1],
                              pd_nodes=[4, 3], theta=0.8, phi=0.5)),
    ("barbell_paper", dict(model="barbell", size=[20.0, 200.0, 40.0, 0], pd_kind=["gauss_mc", "gauss_mc"],
                           pd_rel=[0.05, 0.1], orient_kind="uniform_angles_mc")),
    ("capped_cylinder_iso", dict(model="capped_cylinder", size=[20.0, 200.0, 25.0, 0], orient_kind="isotropic_mc",
                                 pd_kind=["none", "schulz"], pd_rel=[0, 0.2], pd_nodes=[1, 5])),
    ("elliptical_cylinder_pd", dict(model="elliptical_cylinder", size=[20.0, 35.0, 300.0, 0], theta=1.1, phi=0.4, psi=0.9,
                                    pd_kind=["schulz", "schulz"], pd_rel=[0.1, 0.1], pd_nodes=[5, 4])),
    ("hollow_cylinder_paper", dict(model="hollow_cylinder", size=[20.0, 300.0, 8.0, 0], pd_kind=["gauss_mc", "gauss_mc"],
                                   pd_rel=[0.1, 0.05], orient_kind="uniform_angles_mc")),
    ("core_shell_ellipsoid_iso", dict(model="core_shell_ellipsoid", size=[30.0, 70.0, 8.0, 0], sld=[3e-6, 1e-6, 0],
                                      orient_kind="isotropic_mc", pd_kind=["schulz", "none"], pd_rel=[0.15, 0],
                                      pd_nodes=[9, 1])),
    # polymer micelle (R-M4): monodisperse, Schulz core radii with a hard-sphere S(q), the paper's per-event sizes
    ("micelle_mono", dict(model="polymer_micelle", size=[40.0, 15.0, 4000.0, 30.0], sld=[2e-6, 1e-6, 0])),
    ("micelle_pd_py", dict(model="polymer_micelle", size=[40.0, 15.0, 4000.0, 30.0], sld=[2e-6, -1e-6, 0],
                           pd_kind=["schulz", "none"], pd_rel=[0.12, 0], pd_nodes=[12, 1], sq_kind="hard_sphere_py",
                           sq_radius_eff=60.0, sq_volfrac=0.1, background=0.005)),
    ("micelle_paper", dict(model="polymer_micelle", size=[40.0, 15.0, 4000.0, 30.0], sld=[2e-6, 1e-6, 0],
                           pd_kind=["gauss_mc", "none"], pd_rel=[0.1, 0])),
    # thin-walled hollow rectangular prism (R-M5): fixed orientation, Schulz scale with random orientation, the
    # paper's per-event scheme
    ("hollow_prism_fixed", dict(model="hollow_prism_thin", size=[35.0, 75.0, 120.0, 2.0], theta=0.7, phi=2.0, psi=0.5)),
    ("hollow_prism_pd_iso", dict(model="hollow_prism_thin", size=[35.0, 75.0, 120.0, 2.0], pd_kind=["schulz", "none"],
                                 pd_rel=[0.1, 0], pd_nodes=[8, 1], orient_kind="isotropic_mc", background=0.002)),
    ("hollow_prism_paper", dict(model="hollow_prism_thin", size=[35.0, 75.0, 120.0, 2.0], pd_kind=["gauss_mc", "none"],
                                pd_rel=[0.1, 0], orient_kind="uniform_angles_mc")),
]


@pytest.mark.parametrize("precision", ["fp32", "fp64"])
@pytest.mark.parametrize("name,over", MORE_MODELS, ids=[m[0] for m in MORE_MODELS])
def test_more_models_per_neutron(sas, name, over, precision):
    # these models have an fp64 node loop only: an fp32 request is served in fp64 and meets the fp64 bound
    model = W.model(precision=precision, **over)
    check_dump(sas, W.instrument(det_dist=3.0), model, 777, 0, 150000, tol=1e-12, min_detected=5000)


def test_more_models_in_one_batch(sas):
    # one launch per kernel variant present, fixed-node and per-event kernels side by side
    ins = [W.instrument(det_dist=2.0 + 0.5 * i, det_nx=64, det_ny=64) for i in range(len(MORE_MODELS))]
    models = [W.model(precision="fp64", **over) for _, over in MORE_MODELS]
    bt = sas.BatchTracer(ins, models)
    bt.trace(40000, 31)
    sp, sp2, cn = bt.read_detector()
    cnt = bt.counters()
    tot = np.zeros(8, np.uint64)
    for e in range(len(models)):
        ref = O.trace_range(ins[e], models[e], 31, 0, 40000, exp_index=e, dump=False)
        tot += ref["counters"]
        assert np.array_equal(cn[e].reshape(-1), ref["counts"]), e
        m = ref["sum_p"] > 0
        assert np.abs(sp[e].reshape(-1)[m] / ref["sum_p"][m] - 1).max() < 1e-9, e
    assert np.array_equal(cnt[:7], tot[:7])
    bt.close()
    with pytest.raises(sas.SasError) as e:
        sas.Tracer(ins[0], W.model(model="ellipsoid", size=[30.0, 70.0, 0, 0], orient_kind="gauss_quad",
                                   sigma_theta=0.1, sigma_phi=0.1, n_theta=4, n_phi=4))
    assert e.value.status == 5


# ---- full sizes, in the launch configuration bench.py times (BASELINE.json configs 1-4)
def _sampled_windows(sas, ins, model, seed, n_total, exp_index=0, n_win=6, width=4096, tol=None):
    rng = np.random.Generator(np.random.PCG64(seed ^ 0x5EED))
    firsts = [0, n_total - width] + [int(v) for v in rng.integers(0, n_total - width, n_win - 2)]
    tr = sas.Tracer(ins, model)
    n_det = 0
    for first in firsts:
        px, wt, qq = tr.trace_dump(first, width, seed, exp_index)
        ref = O.trace_range(ins, model, seed, first, width, exp_index=exp_index, hist=False)
        assert np.array_equal(px, ref["pixel"]), first
        det = ref["pixel"] >= 0
        bound = tol * np.maximum(np.abs(ref["weight"][det]), 1e-4 * np.abs(ref["weight_env"][det]))
        assert np.all(np.abs(wt[det] - ref["weight"][det]) <= bound), first
        n_det += int(det.sum())
    tr.close()
    return n_det


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_full_size_run_properties_and_sampled_ids(sas, cfg):
    c = W.config(cfg)
    n, seed, ins, model = c["n_neutrons"], c["seed"], c["instrument"], c["model"]
    tr = sas.Tracer(ins, model)
    tr.trace(n, seed)                                  # the launch bench.py times
    sp, sp2, cn = tr.read_detector()
    cnt = tr.counters().astype(np.int64)
    info = tr.launch_info()
    assert info["grid"] % 148 == 0 and info["grid"] * info["block"] in (148 * 640, 148 * 1024)   # 20 (unified kernel) or 32 (warp-specialised) resident warps per SM
    # every neutron has exactly one outcome; the histogram holds exactly the detected ones
    assert cnt[0] == n and cnt[1:7].sum() == n and int(cn.sum()) == cnt[6]
    assert abs(cnt[1] / n - 0.75) < 5 * math.sqrt(0.75 * 0.25 / n)      # slit 1 passes the central quarter
    assert np.all((cn == 0) == (sp == 0)) and np.all(sp2 <= sp * sp * (1 + 1e-12)) and np.all(sp >= 0)
    # the image has the symmetry of the instrument: left/right and up/down halves agree statistically
    tot = sp.sum()
    lr = sp[:, : sp.shape[1] // 2].sum() / tot
    ud = sp[: sp.shape[0] // 2, :].sum() / tot
    rel_err = math.sqrt(float(sp2.sum())) / tot
    assert abs(lr - 0.5) < 6 * rel_err and abs(ud - 0.5) < 6 * rel_err
    # a second launch of the same ids in two halves adds up to the same detector (counts exactly)
    tr.reset()
    tr.trace_range(0, n // 2, seed)
    tr.trace_range(n // 2, n - n // 2, seed)
    sp_b, sp2_b, cn_b = tr.read_detector()
    assert np.array_equal(cn, cn_b)
    m = sp > 0
    assert np.abs(sp_b[m] / sp[m] - 1).max() < 1e-9
    tr.close()
    # the oracle's image of an id prefix is the same estimator: mean weight per hit, pixel ring by ring
    n_pre = 300000
    ref = O.trace_range(ins, model, seed, 0, n_pre, dump=False)
    ny, nx = sp.shape
    yy, xx = np.mgrid[0:ny, 0:nx]
    ring = np.minimum((np.hypot(xx - (nx - 1) / 2, yy - (ny - 1) / 2) / (nx / 2) * 12).astype(int), 15).reshape(-1)
    gp, gc = np.bincount(ring, sp.reshape(-1), 16), np.bincount(ring, cn.reshape(-1).astype(float), 16)
    op, oc = np.bincount(ring, ref["sum_p"], 16), np.bincount(ring, ref["counts"].astype(float), 16)
    op2 = np.bincount(ring, ref["sum_p2"], 16)
    ok = oc > 200
    mean_g, mean_o = gp[ok] / gc[ok], op[ok] / oc[ok]
    sig_o = np.sqrt(np.maximum(op2[ok] / oc[ok] - mean_o ** 2, 0) / oc[ok])
    assert ok.sum() >= 8 and np.all(np.abs(mean_g - mean_o) < 5 * sig_o + 1e-3 * mean_o)
    # ids sampled over the whole range, one by one against the oracle
    assert _sampled_windows(sas, ins, model, seed, n, tol=TOL[model["precision"]]) > 300


def test_full_size_batch_properties_and_sampled_ids(sas):
    c = W.config(4)
    n_each, seed = c["n_neutrons_each"], c["seed"]
    bt = sas.BatchTracer(c["instruments"], c["models"])
    bt.trace(n_each, seed)
    sp, sp2, cn = bt.read_detector()
    cnt = bt.counters().astype(np.int64)
    n_exp = len(c["models"])
    assert cnt[0] == n_exp * n_each and cnt[1:7].sum() == cnt[0] and int(cn.sum()) == cnt[6]
    per_exp = cn.reshape(n_exp, -1).sum(axis=1)
    assert per_exp.min() > 0                           # every experiment wrote its own histogram
    bt.close()
    # three experiments one by one: same Philox word, same detector as a single-experiment run of those ids
    for e in (0, 511, 1023):
        tr = sas.Tracer(c["instruments"][e], c["models"][e])
        px, wt, _ = tr.trace_dump(n_each - 50000, 50000, seed, e)
        tr.close()
        ref = O.trace_range(c["instruments"][e], c["models"][e], seed, n_each - 50000, 50000, exp_index=e, hist=False)
        assert np.array_equal(px, ref["pixel"])
        det = ref["pixel"] >= 0
        bound = 1e-5 * np.maximum(np.abs(ref["weight"][det]), 1e-4 * np.abs(ref["weight_env"][det]))
        assert np.all(np.abs(wt[det] - ref["weight"][det]) <= bound)
        # the batch histogram of experiment e counts what the oracle counts over a prefix, scaled: detected fraction
        frac = per_exp[e] / n_each
        pre = O.trace_range(c["instruments"][e], c["models"][e], seed, 0, 200000, exp_index=e, dump=False, hist=False)
        f0 = pre["counters"][6] / 200000
        assert abs(frac - f0) < 6 * math.sqrt(f0 * (1 - f0) / 200000) + 1e-4


def test_c4_every_experiment_prefix_per_neutron_and_per_bin(sas):
    """ids [0, 1e4) of EACH of the 1024 experiments of config 4, per neutron against the oracle
    (pixels and |Q| bit-exact; weights within 1e-12: the batch is served in fp64), and the batch histogram of the
    same prefix per bin (counts exact, bins <= 1e-9)."""
    c = W.config(4)
    seed, n_exp, n = c["seed"], len(c["models"]), 10**4
    bt = sas.BatchTracer(c["instruments"], c["models"])
    bt.trace(n, seed)
    sp, sp2, cn = (a.reshape(n_exp, -1).copy() for a in bt.read_detector())
    cnt = bt.counters()
    recs = bt.launch_records()
    bt.close()
    assert len(recs) == 2 and all(r["precision"] == 1 for r in recs) and sum(r["n_exp"] for r in recs) == n_exp
    tot = np.zeros(8, np.uint64)
    n_det = 0
    for e in range(n_exp):
        ins, model = c["instruments"][e], c["models"][e]
        tr = sas.Tracer(ins, model)
        px, wt, qq = tr.trace_dump(0, n, seed, e)
        tr.close()
        ref = O.trace_range(ins, model, seed, 0, n, exp_index=e)
        assert np.array_equal(px, ref["pixel"]), e
        reached = ref["q"] > 0
        assert np.array_equal(qq[reached], ref["q"][reached]), e
        det = ref["pixel"] >= 0
        bound = 1e-12 * np.maximum(np.abs(ref["weight"][det]), 1e-4 * np.abs(ref["weight_env"][det]))
        assert np.all(np.abs(wt[det] - ref["weight"][det]) <= bound), e
        assert np.array_equal(cn[e], ref["counts"]), e
        assert_bins(sp[e], ref, "sum_p", 1e-9, e)
        assert_bins(sp2[e], ref, "sum_p2", 1e-9, e)
        tot += ref["counters"]
        n_det += int(det.sum())
    assert np.array_equal(cnt[:7], tot[:7]) and n_det > 400000


def test_batch_id_ranges_add_up_and_shard(sas):
    """sas_trace_batch_range: two half ranges give the detector of the whole range (counts
    exactly), a resumed range continues it, and each rank's shard of a weak-scaling run is such a range."""
    c = W.batch_config(12, 50000, 20250110)
    n, seed = 50000, c["seed"]
    bt = sas.BatchTracer(c["instruments"], c["models"])
    bt.trace(n, seed)
    sp, sp2, cn = (a.copy() for a in bt.read_detector())
    cnt = bt.counters()
    bt.reset()
    bt.trace_range(0, 20001, seed)
    bt.trace_range(20001, n - 20001, seed)
    sp_b, sp2_b, cn_b = (a.copy() for a in bt.read_detector())
    assert np.array_equal(cn, cn_b) and np.array_equal(cnt[:7], bt.counters()[:7])
    m = sp > 0
    assert np.abs(sp_b[m] / sp[m] - 1).max() < 1e-12
    # a range that does not start at 0, against the oracle, experiment by experiment
    bt.reset()
    bt.trace_range(n, 30000, seed)
    cn_c = bt.read_detector()[2].copy()
    bt.close()
    for e in (0, 5, 11):
        ref = O.trace_range(c["instruments"][e], c["models"][e], seed, n, 30000, exp_index=e, dump=False)
        assert np.array_equal(cn_c[e].reshape(-1), ref["counts"]), e
    tr = sas.Tracer(c["instruments"][0], c["models"][0])   # a single-experiment context refuses the batch call
    assert tr.L.sas_trace_batch_range(tr.ctx, 0, 10, 1) == 2
    tr.close()


def test_precision_is_decided_per_experiment(sas):
    """An fp32 batch that mixes a Schulz-polydisperse sphere (node loop: fp32) with a monodisperse sphere whose
    first form-factor zero lies on the detector (one evaluation per neutron: served in fp64):
    two launches of different precision, each experiment within ITS tolerance."""
    ins = W.instrument(det_nx=128, det_ny=128)
    poly = W.model(precision="fp32", size=[60.0, 0, 0, 0], pd_kind=["schulz", "none"], pd_rel=[0.1, 0.0], pd_nodes=[24, 1])
    mono = W.model(precision="fp32", size=[80.0, 0, 0, 0])          # zero at q = 4.4934 / 80 = 0.056: on the detector
    seed, n = 77, 200000
    bt = sas.BatchTracer([ins, ins, ins], [poly, mono, poly])
    bt.trace(n, seed)
    sp, sp2, cn = (a.reshape(3, -1).copy() for a in bt.read_detector())
    recs = bt.launch_records()
    bt.close()
    assert sorted((r["precision"], r["n_exp"]) for r in recs) == [(0, 2), (1, 1)]
    for e, (model, tol) in enumerate(((poly, 1e-5), (mono, 1e-12), (poly, 1e-5))):
        tr = sas.Tracer(ins, model)
        check_prefix(sas, ins, model, seed, n, exp_index=e, tol=tol, min_detected=5000, tracer=tr)
        tr.close()
        ref = O.trace_range(ins, model, seed, 0, n, exp_index=e)
        assert np.array_equal(cn[e], ref["counts"]), e
        assert_bins(sp[e], ref, "sum_p", 1e-9 if tol < 1e-11 else 1e-5, e)


def test_producer_consumer_split_is_chosen_per_launch_group(sas):
    """The warp-specialised kernel exists in two block splits: one producer + one consumer
    warpgroup (256 threads) and one + three (512 threads) for launches bound by stages B and C.  A barbell and a
    32-node fp64 sphere take the heavy split, a monodisperse sphere and the fp32 node loop the default one; an fp64
    batch whose sphere group holds two 32-node experiments and one monodisperse one is launched once, in the heavy
    split (majority), and every experiment is the oracle's per neutron and per bin whichever split served it."""
    ins = W.instrument(det_nx=128, det_ny=128)
    mono = W.model(precision="fp64", size=[80.0, 0, 0, 0])
    poly64 = W.model(precision="fp64", size=[60.0, 0, 0, 0], pd_kind=["schulz", "none"], pd_rel=[0.1, 0.0], pd_nodes=[32, 1])
    poly32 = dict(poly64, precision="fp32")
    barbell = W.config(6)["model"]
    for model, block in ((mono, 256), (poly64, 512), (poly32, 256), (barbell, 512)):
        tr = sas.Tracer(ins, model)
        tr.trace(100000, 5)
        recs = tr.launch_records()
        tr.close()
        assert [(r["warp_specialised"], r["block"]) for r in recs] == [(1, block)], (model["model"], recs)
    seed, n = 78, 200000
    models = [poly64, mono, poly64]
    bt = sas.BatchTracer([ins] * 3, models)
    bt.trace(n, seed)
    sp, sp2, cn = (a.reshape(3, -1).copy() for a in bt.read_detector())
    recs = bt.launch_records()
    bt.close()
    assert [(r["n_exp"], r["block"]) for r in recs] == [(3, 512)], recs
    for e, model in enumerate(models):
        tr = sas.Tracer(ins, model)
        check_prefix(sas, ins, model, seed, n, exp_index=e, tol=1e-12, min_detected=5000, tracer=tr)
        tr.close()
        ref = O.trace_range(ins, model, seed, 0, n, exp_index=e)
        assert np.array_equal(cn[e], ref["counts"]), e
        assert_bins(sp[e], ref, "sum_p", 1e-9, e)


def test_fp32_request_with_phases_beyond_the_proven_range_runs_in_fp64(sas):
    """The fp32 argument reductions are proven for |x| < 1e3 rad (device_math.cuh).  A Schulz-polydisperse sphere of
    4000 A at q_max = 0.3 reaches 1.6e3: the library serves that experiment in fp64 (include/sas.h) and meets the
    fp64 tolerance; just inside the range (2800 A, largest node factor about 1.1: below 950 rad) it stays in fp32 within 1e-5."""
    ins = W.instrument(det_nx=64, det_ny=64)
    for R, expect in ((4000.0, 1), (2800.0, 0)):
        model = W.model(precision="fp32", size=[R, 0, 0, 0], pd_kind=["schulz", "none"], pd_rel=[0.03, 0.0], pd_nodes=[8, 1])
        tr = sas.Tracer(ins, model)
        tr.trace(1000, 5)
        assert tr.launch_records()[-1]["precision"] == expect
        tr.reset()
        check_prefix(sas, ins, model, 5, 200000, tol=1e-12 if expect else 1e-5, min_detected=5000, tracer=tr)
        tr.close()


@pytest.mark.parametrize("name,over", [
    ("big_cylinder_iso", dict(model="cylinder", size=[300.0, 3000.0, 0, 0], orient_kind="isotropic_mc")),
    ("big_cylinder_event", dict(model="cylinder", size=[300.0, 3000.0, 0, 0], pd_kind=["gauss_mc", "gauss_mc"],
                                pd_rel=[0.1, 0.1], orient_kind="uniform_angles_mc")),
    ("big_sphere_schulz", dict(model="sphere", size=[2000.0, 0, 0, 0], pd_kind=["schulz", "none"], pd_rel=[0.05, 0],
                               pd_nodes=[16, 1])),
    ("big_core_shell_sphere", dict(model="core_shell_sphere", size=[800.0, 150.0, 0, 0], sld=[3e-6, 1e-6, 0],
                                   pd_kind=["schulz", "schulz"], pd_rel=[0.05, 0.1], pd_nodes=[6, 5])),
    ("big_hollow_cylinder", dict(model="hollow_cylinder", size=[250.0, 2000.0, 40.0, 0], orient_kind="isotropic_mc")),
])
def test_large_arguments_of_the_fp64_special_functions(sas, name, over):
    """The tracer's own fp64 sin/cos, sin u - u cos u and Lambda = 2 J1(x)/x far beyond the arguments of the
    BASELINE.json workloads: q x size up to 600 rad (sphere), 450 rad (sinc of the rod) and x = 90 (Lambda: the
    Hankel range, x > 12, for most detected neutrons), against the oracle's glibc sin, cos, j1 at 1e-12."""
    model = W.model(precision="fp64", **over)
    check_dump(sas, W.instrument(det_dist=3.0), model, 4242, 0, 200000, tol=1e-12, min_detected=8000)


def test_pixels_stay_bit_exact_over_2e7_ids(sas):
    """R-C10: the azimuth's sin/cos come from the tracer's own fp64 routine on the device and from glibc in the
    oracle (about an ulp apart): a pixel could flip only for a hit within ~1e-16 of a pixel edge.  2e7 ids of c0
    (9.7e5 detected neutrons), far from the id ranges of the other tests: not one pixel, not one drawn |Q| differs."""
    c = W.config(0)
    tr = sas.Tracer(c["instrument"], c["model"])
    n_det = 0
    for first in range(7 * 10**9, 7 * 10**9 + 2 * 10**7, 2 * 10**6):
        px, wt, qq = tr.trace_dump(first, 2 * 10**6, c["seed"])
        ref = O.trace_range(c["instrument"], c["model"], c["seed"], first, 2 * 10**6, hist=False)
        assert np.array_equal(px, ref["pixel"]), first
        reached = ref["q"] > 0
        assert np.array_equal(qq[reached], ref["q"][reached]), first
        n_det += int((px >= 0).sum())
    tr.close()
    assert n_det > 9 * 10**5


MSA = dict(sq_kind="hayter_msa", sq_radius_eff=45.0, sq_volfrac=0.2, sq_contact_kT=5.0, sq_kappa_sigma=2.0)


@pytest.mark.parametrize("name,over,tol", [
    ("sphere_mono_fp64", dict(model="sphere", precision="fp64", size=[40.0, 0, 0, 0], **MSA), 1e-12),
    ("sphere_schulz_fp32", dict(model="sphere", precision="fp32", size=[40.0, 0, 0, 0], pd_kind=["schulz", "none"],
                                pd_rel=[0.15, 0], pd_nodes=[32, 1], scale=0.2, **MSA), 1e-5),
    ("sphere_schulz_fp64", dict(model="sphere", precision="fp64", size=[40.0, 0, 0, 0], pd_kind=["schulz", "none"],
                                pd_rel=[0.15, 0], pd_nodes=[32, 1], scale=0.2, **MSA), 1e-12),
    ("ellipsoid_paper", dict(model="ellipsoid", precision="fp64", size=[30.0, 60.0, 0, 0], pd_kind=["gauss_mc", "none"],
                             pd_rel=[0.1, 0], orient_kind="uniform_angles_mc", **MSA), 1e-12),
    ("micelle_schulz", dict(model="polymer_micelle", precision="fp64", size=[40.0, 15.0, 4000.0, 30.0], sld=[2e-6, 1e-6, 0],
                            pd_kind=["schulz", "none"], pd_rel=[0.1, 0], pd_nodes=[8, 1],
                            **dict(MSA, sq_volfrac=0.35, sq_contact_kT=6.0, sq_kappa_sigma=6.0)), 1e-12),
])
def test_hayter_msa_structure_factor(sas, name, over, tol):
    """R-S2: the library solves the closure on the host with its own Newton iteration and Gauss-Legendre rule and
    evaluates S(q) on the device; per neutron against the oracle (own solver, own rule)."""
    check_dump(sas, W.instrument(det_dist=3.0), W.model(**over), 909, 0, 200000, tol=tol, min_detected=8000)


def test_hayter_msa_in_a_batch_and_its_refusals(sas):
    ins = [W.instrument(det_nx=64, det_ny=64, det_dist=2.0 + e) for e in range(4)]
    models = [W.model(size=[30.0 + 5 * e, 0, 0, 0], **dict(MSA, sq_contact_kT=1.0 + 2.0 * e, sq_volfrac=0.1 + 0.08 * e)) for e in range(4)]
    models[2] = W.model(size=[40.0, 0, 0, 0], sq_kind="hard_sphere_py", sq_radius_eff=45.0, sq_volfrac=0.2)
    bt = sas.BatchTracer(ins, models)
    bt.trace(60000, 5)
    sp, sp2, cn = (a.reshape(4, -1).copy() for a in bt.read_detector())
    bt.close()
    for e in range(4):
        ref = O.trace_range(ins[e], models[e], 5, 0, 60000, exp_index=e)
        assert np.array_equal(cn[e], ref["counts"]), e
        assert_bins(sp[e], ref, "sum_p", 1e-9, e)
    # the closure's known failure: a dilute, strongly charged system has g(1+) < 0 -> refused, as is a q range
    # beyond the quadrature rule
    with pytest.raises(sas.SasError) as err:
        sas.Tracer(ins[0], W.model(**dict(MSA, sq_volfrac=0.05, sq_contact_kT=50.0, sq_kappa_sigma=0.5)))
    assert err.value.status == 5 and "contact" in str(err.value)
    with pytest.raises(sas.SasError) as err:
        sas.Tracer(ins[0], W.model(**dict(MSA, sq_radius_eff=150.0)))
    assert err.value.status == 5
    with pytest.raises(sas.SasError) as err:                 # a sphere-sphere S(q) is not offered for rods
        sas.Tracer(ins[0], W.model(model="cylinder", size=[20.0, 400.0, 0, 0], orient_kind="isotropic_mc", **MSA))
    assert err.value.status == 5 and "globular" in str(err.value)
    with pytest.raises(sas.SasError) as err:
        sas.Tracer(ins[0], W.model(**dict(MSA, sq_kappa_sigma=0.0)))
    assert err.value.status == 1


@pytest.mark.parametrize("cfg", [5, 6, 7, 8, 9])
def test_paper_scheme_workloads_of_the_bench_per_neutron(sas, cfg):
    """The n1..n5 workloads exactly as bench.py configures them (the paper's per-event averaging on its rod, a
    barbell, a micelle, charged spheres with the Hayter MSA S(q), a thin-walled hollow prism): an id prefix per neutron and per bin."""
    c = W.config(cfg)
    check_prefix(sas, c["instrument"], c["model"], c["seed"], 150000, min_detected=6000)


def test_back_to_back_steps_without_launch_timing_are_each_a_clean_step(sas):
    """sas_set_launch_timing(0) leaves reset -> trace adjacent in the stream, where the trace kernel is launched
    programmatically dependent on the zeroing kernel (sas_api.cu: launch): 300 steps in a row, no host
    synchronisation in between, each must leave exactly the image of a single step (a trace kernel that touched
    the detector before the zeroing finished, or a zeroing that overtook the previous trace, would show)."""
    c = W.config(0)
    for ins, model in ((c["instrument"], c["model"]), (W.instrument(det_dist=3.0), W.model(model="cylinder", size=[20.0, 400.0, 0, 0], orient_kind="isotropic_mc", precision="fp32"))):
        tr = sas.Tracer(ins, model)
        tr.trace(100000, 3)
        want = [a.copy() for a in tr.read_detector()]
        want_c = tr.counters().copy()
        assert len(tr.launch_records()) == 1
        tr.kernel_time_ms(reset=True)
        tr.set_launch_timing(False)
        for n in (100000, 777, 100000):           # a different step in between: leftovers of it would show too
            for _ in range(100):
                tr.reset()
                tr.trace(n, 3)
        got = tr.read_detector()
        assert tr.launch_records() == [] and tr.kernel_time_ms()[1] == 0
        assert np.array_equal(got[2], want[2]) and np.array_equal(tr.counters(), want_c)
        assert np.allclose(got[0], want[0], rtol=1e-12, atol=0) and np.allclose(got[1], want[1], rtol=1e-12, atol=0)
        tr.set_launch_timing(True)
        tr.reset(); tr.trace(100000, 3)
        assert len(tr.launch_records()) == 1 and np.array_equal(tr.read_detector()[2], want[2])
        tr.close()


def test_context_stays_on_its_device(sas):
    """A context lives on the device it was created on, whatever torch's current device is (multi-GPU ranks);
    with one GPU only the default-device behaviour can be checked."""
    import torch
    c = W.config(0)
    dev = torch.device("cuda", torch.cuda.device_count() - 1)
    tr = sas.Tracer(c["instrument"], c["model"], device=dev)
    assert tr.sum_p.device == dev and tr.device == dev
    with torch.cuda.device(0):
        tr.trace(100000, c["seed"])
        cnt = tr.counters()
    tr.close()
    ref = O.trace_range(c["instrument"], c["model"], c["seed"], 0, 100000, dump=False)
    assert np.array_equal(cnt[:7], ref["counters"][:7])
    tr = sas.Tracer(c["instrument"], c["model"])          # default: torch's current device, left unchanged
    assert tr.device == torch.device("cuda", torch.cuda.current_device())
    tr.close()


def test_triangular_wavelength_law_per_neutron(sas):
    """R-L1: the velocity-selector law through every stage (the fp64 classifier takes over from the fp32 one):
    c0 and c1-fp32 with lambda_dist = triangle, per neutron and per bin against the oracle."""
    for idx in (0, 1):
        c = W.config(idx)
        ins = dict(c["instrument"], lambda_dist="triangle")
        check_prefix(sas, ins, c["model"], c["seed"], 400000, min_detected=15000)
    tr = sas.Tracer(dict(W.instrument(), lambda_dist="triangle"), W.config(0)["model"])
    tr.trace(10**7, 3)
    cnt = tr.counters()
    tr.close()
    assert cnt[7] > 0.6 * (cnt[0] - cnt[1])               # the classifier still removes most survivors


def test_resolution_smeared_curve_of_the_paper_rod_against_the_oracle(sas):
    """NEXT-4: the randomly oriented R = 119 A, L = 800 A rod with 5 % Gaussian sizes on an
    instrument with a 10 % FWHM velocity-selector band, 5 mm slits and 3.9 mm pixels: the GPU image reduced by
    sas_reduce_radial is the same resolution-smeared I(q) as the oracle's ring average of its own, smaller, image,
    ring by ring within the standard errors both carry from sum P^2 (the measured curve of PAPER.md:173 and the
    KWS-1 file are not in the container; the oracle's curve stands in for them)."""
    lam = 6.0
    ins = W.instrument(lambda_min=0.9 * lam, lambda_max=1.1 * lam, lambda_dist="triangle", det_nx=128, det_ny=128, q_max=0.12)
    model = W.model(model="cylinder", precision="fp64", size=[119.0, 800.0, 0, 0], pd_kind=["gauss_mc", "gauss_mc"],
                    pd_rel=[0.05, 0.05], orient_kind="isotropic_mc")
    n_gpu, n_orc, seed, nb = 3 * 10**8, 2 * 10**7, 1731, 40
    tr = sas.Tracer(ins, model)
    tr.trace(n_gpu, seed)
    q, I, sig, npix = tr.reduce_radial(lam, 0.004, 0.064, nb)
    tr.close()
    ref = O.trace_range(ins, model, seed, n_gpu, n_orc, dump=False)          # ids the GPU run did not use
    qo, Io, so, no = O.reduce_radial(ins, ref["sum_p"], ref["sum_p2"], n_orc, lam, 0.004, 0.064, nb)
    assert np.array_equal(npix, no) and np.allclose(q, qo, rtol=1e-15)
    ok = (npix > 0) & (Io > 0)
    z = (I[ok] - Io[ok]) / np.sqrt(sig[ok] ** 2 + so[ok] ** 2)
    assert ok.sum() >= 35 and np.abs(z).max() < 4.5 and abs(float((z * z).mean()) - 1.0) < 5 * math.sqrt(2.0 / ok.sum())
    # the smearing is visible: the first minimum (Q ~ 0.032 1/A) is shallower than on the narrow-band instrument of
    # the test above, but still there
    i_min = int(np.argmin(np.where((q > 0.026) & (q < 0.040), I, np.inf)))
    assert 0.029 <= q[i_min] <= 0.036 and I[i_min] < 0.8 * I[i_min + 4]


def test_ring_average_normalises_by_the_neutrons_the_buffers_hold(sas):
    """sas_radial_desc.n_launched: buffers that hold more than this context traced (the detector merged from two
    ranks on rank 0) are normalised by the figure the caller gives; 0 keeps the context's own count."""
    c = W.config(0)
    a = sas.Tracer(c["instrument"], c["model"])
    b = sas.Tracer(c["instrument"], c["model"])
    a.trace_range(0, 300000, c["seed"])
    b.trace_range(300000, 300000, c["seed"])
    q, I_a, s_a, _ = a.reduce_radial(6.0, 0.004, 0.07, 30)
    a.sum_p += b.sum_p                                    # what merge_detectors does on rank 0
    a.sum_p2 += b.sum_p2
    a.torch.cuda.synchronize()
    _, I_m, s_m, _ = a.reduce_radial(6.0, 0.004, 0.07, 30, n_launched=600000)
    _, I_wrong, _, _ = a.reduce_radial(6.0, 0.004, 0.07, 30)
    ref = O.trace_range(c["instrument"], c["model"], c["seed"], 0, 600000, dump=False)
    _, I_o, s_o, _ = O.reduce_radial(c["instrument"], ref["sum_p"], ref["sum_p2"], 600000, 6.0, 0.004, 0.07, 30)
    m = I_o > 0
    assert np.allclose(I_m[m], I_o[m], rtol=1e-11) and np.allclose(s_m[m], s_o[m], rtol=1e-11)
    assert np.allclose(I_wrong[m], 2.0 * I_m[m], rtol=1e-12)
    a.close()
    b.close()


def test_paper_pin_first_minimum_of_the_random_rod_end_to_end(sas):
    """a randomly oriented cylinder R = 119 A, L = 800 A with 5 % polydispersity has its lowest-Q
    minimum at Q ~ 0.032 1/A (R = 3.78 / Q_min).  Here the whole CUDA path produces it: 4e8 neutrons through the
    instrument (narrow wavelength band so that the ring is not smeared away), the paper's own per-event size and
    orientation draws, the detector image averaged over rings with numpy."""
    lam = 6.0
    ins = W.instrument(lambda_min=lam - 0.05, lambda_max=lam + 0.05, det_nx=256, det_ny=256, q_max=0.12)
    model = W.model(model="cylinder", precision="fp64", size=[119.0, 800.0, 0, 0], pd_kind=["gauss_mc", "gauss_mc"],
                    pd_rel=[0.05, 0.05], orient_kind="isotropic_mc")
    tr = sas.Tracer(ins, model)
    tr.trace(4 * 10**8, 173)
    sp, sp2, cn = tr.read_detector()
    tr.close()
    ny, nx = sp.shape
    yy, xx = np.mgrid[0:ny, 0:nx]
    X = (xx + 0.5) / nx * ins["det_xw"] - 0.5 * ins["det_xw"]
    Y = (yy + 0.5) / ny * ins["det_yh"] - 0.5 * ins["det_yh"]
    two_theta = np.arctan(np.hypot(X, Y) / ins["det_dist"])
    q = 4 * math.pi / lam * np.sin(0.5 * two_theta)
    # solid angle per pixel ~ cos^3(2 theta): divide it out so that the profile is I(q)
    img = sp / np.cos(two_theta) ** 3
    edges = np.linspace(0.010, 0.060, 51)
    idx = np.digitize(q.reshape(-1), edges) - 1
    ok = (idx >= 0) & (idx < 50)
    prof = np.bincount(idx[ok], img.reshape(-1)[ok], 50) / np.maximum(np.bincount(idx[ok], None, 50), 1)
    qc = 0.5 * (edges[1:] + edges[:-1])
    # first local minimum of the smoothed profile
    sm = np.convolve(prof, np.ones(3) / 3, mode="same")
    i_min = next(i for i in range(2, 47) if sm[i] < sm[i - 1] and sm[i] < sm[i + 1] and sm[i] < sm[i - 2] and sm[i] < sm[i + 2])
    assert 0.030 <= qc[i_min] <= 0.034, qc[i_min]
    assert 3.5 < 119.0 * qc[i_min] < 4.1                  # the paper's R = 3.78 / Q_min


def test_detector_image_agrees_with_the_analytic_intensity_within_3_sigma(sas):
    """north_star: "the detector image agrees with the analytic I(Q) within 3 sigma statistical error".
    Monochromatic pencil beam (DESIGN.md R-C17), 2e8 neutrons on a 64 x 64 detector through the CUDA path; the
    expectation per pixel is the closed-form sphere intensity (numpy, nothing of the oracle but the source
    weight p0 of one ray) integrated over the pixel's solid angle."""
    ins = W.pencil_instrument(det_nx=64, det_ny=64, q_min=0.004, q_max=0.3)
    m = W.config(0)["model"]
    n = 2 * 10**8
    tr = sas.Tracer(ins, m)
    tr.trace(n, 4242)
    sp, sp2, cn = tr.read_detector()
    tr.close()
    p0, ell = O.trace_one(ins, m, 4242, 0).p0, 1e-3
    R, drho, scale = m["size"][0], m["sld"][0], m["scale"]
    nx = ny = 64
    Wd, D, k = ins["det_xw"], ins["det_dist"], 2 * math.pi / ins["lambda_min"]
    g, gw = np.polynomial.legendre.leggauss(5)
    xs = ((np.arange(nx)[:, None] + 0.5 + 0.5 * g[None, :]) * (Wd / nx) - 0.5 * Wd).reshape(-1)
    w1 = np.tile(0.5 * gw * (Wd / nx), nx)
    X, Y = xs[None, :], xs[:, None]
    R2 = X * X + Y * Y
    q = 2 * k * np.sin(0.5 * np.arctan2(np.sqrt(R2), D))
    u = q * R
    V = 4 * math.pi / 3 * R ** 3
    Iq = 1e8 * scale * drho ** 2 * V * (3 * (np.sin(u) - u * np.cos(u)) / u ** 3) ** 2
    Iq = np.where((q >= ins["q_min"]) & (q <= ins["q_max"]), Iq, 0.0)
    f = Iq * D / (D * D + R2) ** 1.5 * w1[None, :] * w1[:, None]
    E = n * p0 * 100 * ell * f.reshape(ny, 5, nx, 5).sum(axis=(1, 3))
    ok = cn > 100
    ok[30:34, 30:34] = False                      # pixels cut by the q_min circle
    z = (sp[ok] - E[ok]) / np.sqrt(sp2[ok])
    chi2 = float((z * z).mean())
    assert ok.sum() > 3000
    assert abs(chi2 - 1) < 5 * math.sqrt(2 / ok.sum()), chi2
    assert (np.abs(z) > 3).mean() <= 0.01
    assert abs(sp[ok].sum() / E[ok].sum() - 1) < 1e-3


def test_host_proved_skips_at_their_margins(sas):
    """Stage B skips the sample's lateral slabs and the slit arithmetic when the host has proved them idle
    (DESIGN.md section 5).  Instruments just inside and just outside those proofs must give the oracle's
    outcomes and pixels exactly."""
    m = W.config(0)["model"]
    base = W.instrument()
    # beam envelope at the far face of the sample (the host's own bound): focus half-width + divergence beyond it
    z_far = base["sample_z"] + 0.5 * base["sample_zd"]
    bx = 0.5 * base["focus_xw"] + (z_far - base["focus_z"]) * (0.5 * base["focus_xw"] + 0.5 * base["src_xw"]) / base["focus_z"]
    for scale in (1 + 3e-6, 1 - 3e-6, 0.9, 0.5):           # proof holds / fails by a hair / lateral faces really cut
        ins = W.instrument(sample_xw=2 * bx * scale, sample_yh=2 * bx * scale)
        check_dump(sas, ins, m, 31337, 0, 120000, min_detected=1000)
        tr = sas.Tracer(ins, m)
        tr.trace(120000, 31337)
        ref = O.trace_range(ins, m, 31337, 0, 120000, dump=False)
        assert np.array_equal(tr.counters()[:7], ref["counters"][:7]), scale
        tr.close()
    # slit 2 a hair narrower than the focus rectangle: it cuts, the slit arithmetic must run
    ins = W.instrument(slit2_xw=base["focus_xw"] * (1 - 1e-9))
    ref = O.trace_range(ins, m, 31337, 0, 400000, dump=False, hist=False)
    check_dump(sas, ins, m, 31337, 0, 400000, min_detected=1000)
    tr = sas.Tracer(ins, m)
    tr.trace(400000, 31337)
    assert np.array_equal(tr.counters()[:7], ref["counters"][:7])
    tr.close()


def test_many_tiny_experiments_in_one_batch(sas):
    # 150 experiments of 700 neutrons each: work items shorter than the minimum item, ragged rows, an experiment
    # change at every item, all three kernel variants of c4-like batches plus a per-event one
    c = W.batch_config(150, 700, 555)
    models = list(c["models"])
    models[7] = W.model(model="sphere", precision="fp32", size=[60.0, 0, 0, 0], pd_kind=["gauss_mc", "none"], pd_rel=[0.2, 0])
    bt = sas.BatchTracer(c["instruments"], models)
    bt.trace(700, 555)
    sp, sp2, cn = bt.read_detector()
    cnt = bt.counters()
    bt.close()
    tot = np.zeros(8, np.uint64)
    for e in range(150):
        ref = O.trace_range(c["instruments"][e], models[e], 555, 0, 700, exp_index=e, dump=False)
        tot += ref["counters"]
        assert np.array_equal(cn[e].reshape(-1), ref["counts"]), e
        m = ref["sum_p"] > 0
        if m.any():
            assert np.abs(sp[e].reshape(-1)[m] / ref["sum_p"][m] - 1).max() < 1e-9, e
    assert np.array_equal(cnt[:7], tot[:7])


# ---- NEXT-4 (first part): ring average of the detector into I(q) on the GPU
def test_radial_reduction_matches_the_oracle(sas):
    c = W.config(1)
    tr = sas.Tracer(c["instrument"], c["model"])
    tr.trace(2 * 10**7, c["seed"])
    sp, sp2, cn = tr.read_detector()
    launched = int(tr.counters()[0])
    for lam, q_lo, q_hi, nb in ((6.0, 0.0, 0.08, 64), (5.4, 0.004, 0.05, 1), (6.6, 0.01, 0.0733, 1024)):
        q, I, s, n = tr.reduce_radial(lam, q_lo, q_hi, nb)
        rq, rI, rs, rn = O.reduce_radial(c["instrument"], sp, sp2, launched, lam, q_lo, q_hi, nb)
        assert np.array_equal(n, rn) and np.array_equal(q, rq)
        m = rI > 0
        assert m.sum() >= min(nb, 40) * 0.8
        assert np.abs(I[m] / rI[m] - 1).max() < 1e-12 and np.abs(s[m] / rs[m] - 1).max() < 1e-12
        assert np.all(I[~m] == 0) and np.all(s[~m] == 0)
    # 2e7 neutrons give every populated ring a positive intensity with a small relative error
    q, I, s, n = tr.reduce_radial(6.0, 0.004, 0.07, 66)
    assert np.all(I[n > 0] > 0) and np.all(s[n > 0] < 0.2 * I[n > 0]) and (n > 0).sum() >= 60
    with pytest.raises(sas.SasError):
        tr.reduce_radial(6.0, 0.05, 0.01, 10)
    with pytest.raises(sas.SasError):
        tr.reduce_radial(6.0, 0.0, 0.1, 5000)
    with pytest.raises(sas.SasError):
        tr.reduce_radial(6.0, 0.0, 0.1, 10, exp_index=1)
    tr.close()
    # a batch: each experiment's own detector distance and histogram
    b = W.batch_config(6, 400000, 77)
    bt = sas.BatchTracer(b["instruments"], b["models"])
    bt.trace(400000, 77)
    sp, sp2, cn = bt.read_detector()
    for e in (0, 3, 5):
        lam = 0.5 * (b["instruments"][e]["lambda_min"] + b["instruments"][e]["lambda_max"])
        q, I, s, n = bt.reduce_radial(lam, 0.0, 0.1, 40, exp_index=e)
        rq, rI, rs, rn = O.reduce_radial(b["instruments"][e], sp[e], sp2[e], 400000, lam, 0.0, 0.1, 40)
        m = rI > 0
        assert np.array_equal(n, rn) and np.abs(I[m] / rI[m] - 1).max() < 1e-12 and np.abs(s[m] / rs[m] - 1).max() < 1e-12
    bt.close()
