"""Pins of the oracle's tracer (source, slits, sample, Q choice, detector, weight):
worked example, closed-form geometry, weight conservation, and the pencil-beam
chi^2 test against the numerically integrated I(Q) (DESIGN.md R-C17)."""
import math
import os

import numpy as np

import sas_workloads as W
from oracle import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")
TWO_PI = 2 * math.pi


def _gold():
    with open(os.path.join(GOLD, "worked_example_c0.txt")) as f:
        return [l.split() for l in f if l.strip() and not l.startswith("#")]


def test_worked_example_c0():
    c = W.config(0)
    for t in _gold():
        if t[0].isdigit():
            r = O.trace_one(c["instrument"], c["model"], c["seed"], int(t[0]))
            assert r.status == 0 and r.pixel == int(t[1])
            assert abs(r.q - float(t[2])) < 1e-14
            assert abs(r.weight - float(t[3])) < 1e-13 * float(t[3])
        elif t[0] == "id3":
            r = O.trace_one(c["instrument"], c["model"], c["seed"], 3)
            lam, ell, p0, I, qx, qy, qz = map(float, t[1:])
            assert abs(r.lam - lam) < 1e-14 and abs(r.ell - ell) < 1e-17
            assert abs(r.p0 - p0) < 1e-20 and abs(r.intensity - I) < 1e-14
            for a, b in zip(r.Q, (qx, qy, qz)):
                assert abs(a - b) < 1e-13 * r.q       # the probe formed Q as k(d - d'), which cancels: 2e-14 |Q|
        elif t[0] == "counters":
            out = O.trace_range(c["instrument"], c["model"], c["seed"], 0, 200000, dump=False, hist=False)
            cn = out["counters"]
            assert [int(cn[1]), int(cn[5]), int(cn[6])] == [int(v) for v in t[1:]]
            assert int(cn[0]) == 200000 and int(cn[1:7].sum()) == 200000
    for i in (0, 1, 2):      # id 3 is the first detected neutron
        assert O.trace_one(c["instrument"], c["model"], c["seed"], i).status != 0


def test_counters_and_histogram_bookkeeping():
    c = W.config(0)
    n = 100000
    out = O.trace_range(c["instrument"], c["model"], c["seed"], 0, n)
    cn = out["counters"].astype(np.int64)
    # slit 1 (5x5 mm in the plane of a 10x10 mm source) passes 1/4 +- binomial
    assert abs((n - cn[1]) / n - 0.25) < 4 * math.sqrt(0.25 * 0.75 / n)
    assert cn[2] == 0 and cn[3] == 0 and cn[4] == 0      # focus = slit 2, beam inside the sample
    det = out["pixel"] >= 0
    assert det.sum() == cn[6] == out["counts"].sum()
    # histograms are the id-ordered sums of the dump
    sp = np.zeros_like(out["sum_p"])
    np.add.at(sp, out["pixel"][det], out["weight"][det])
    assert np.allclose(sp, out["sum_p"], rtol=1e-13, atol=0)
    sp2 = np.zeros_like(sp)
    np.add.at(sp2, out["pixel"][det], out["weight"][det] ** 2)
    assert np.allclose(sp2, out["sum_p2"], rtol=1e-13, atol=0)
    # ranges are additive and independent of where they start (counter-based RNG)
    a = O.trace_range(c["instrument"], c["model"], c["seed"], 0, 40000)
    b = O.trace_range(c["instrument"], c["model"], c["seed"], 40000, 60000)
    assert np.array_equal(a["counts"] + b["counts"], out["counts"])
    assert np.array_equal(np.concatenate([a["pixel"], b["pixel"]]), out["pixel"])
    assert np.array_equal(np.concatenate([a["weight"], b["weight"]]), out["weight"])
    # another seed / another experiment index gives another stream
    o2 = O.trace_range(c["instrument"], c["model"], c["seed"] + 1, 0, 1000)
    o3 = O.trace_range(c["instrument"], c["model"], c["seed"], 0, 1000, exp_index=1)
    assert not np.array_equal(o2["pixel"], out["pixel"][:1000])
    assert not np.array_equal(o3["pixel"], out["pixel"][:1000])


def test_linearity_is_bit_exact():
    c = W.config(0)
    a = O.trace_range(c["instrument"], c["model"], 7, 0, 20000, hist=False)
    m2 = dict(c["model"], scale=0.02)
    b = O.trace_range(c["instrument"], m2, 7, 0, 20000, hist=False)
    assert np.array_equal(a["pixel"], b["pixel"])
    assert np.array_equal(2.0 * a["weight"], b["weight"])
    m4 = dict(c["model"], sld=[2.0e-6, 0, 0])
    d = O.trace_range(c["instrument"], m4, 7, 0, 20000, hist=False)
    assert np.allclose(4.0 * a["weight"], d["weight"], rtol=4e-16, atol=0)


def test_on_axis_pencil_geometry_closed_form():
    # a 1 nm "pencil": the ray is the z axis to ~1e-9; pixel from X = D tan(2 theta) cos(chi) etc.
    ins = W.pencil_instrument(src_xw=1e-9, src_yh=1e-9, slit1_xw=1e-6, slit1_yh=1e-6, slit2_xw=1e-6,
                              slit2_yh=1e-6, focus_xw=1e-9, focus_yh=1e-9)
    m = W.model(model="flat", scale=1.0)
    k = TWO_PI / 6.0
    n_checked = 0
    for i in range(400):
        r = O.trace_one(ins, m, 11, i)
        assert r.status in (0, 5)
        two_theta = 2 * math.asin(r.q / (2 * k))
        chi = TWO_PI * r.u[7]
        zs = r.u[5] * 1e-3 + (5.01 - 0.5e-3)
        D = 5.01 + 5.0 - zs
        X, Y = D * math.tan(two_theta) * math.cos(chi), D * math.tan(two_theta) * math.sin(chi)
        inside = abs(X) < 0.25 and abs(Y) < 0.25
        assert (r.status == 0) == inside
        assert abs(r.ell - 1e-3) < 1e-12
        assert abs(r.lam - 6.0) == 0.0
        if inside:
            fx, fy = (X + 0.25) * 256, (Y + 0.25) * 256
            if min(fx % 1, 1 - fx % 1, fy % 1, 1 - fy % 1) > 1e-5:
                assert r.pixel == int(fy) * 128 + int(fx)
                n_checked += 1
            # |Q| = q, Q perpendicular-ish: Qz = -k(1 - cos 2theta) ... sign: Q = k(d - d')
            assert abs(math.sqrt(sum(v * v for v in r.Q)) - r.q) < 1e-12 * r.q
            assert abs(r.Q[2] - k * (1 - math.cos(two_theta))) < 1e-9 * r.q
            assert abs(r.Q[0] + k * math.sin(two_theta) * math.cos(chi)) < 1e-7 * r.q
            # flat model, T = 1: p = p0 * 100 ell * q/k^2 * 2 pi (qmax - qmin)
            p = r.p0 * 0.1 * r.q / k ** 2 * TWO_PI * 0.299
            assert abs(r.weight - p) < 1e-9 * p
    assert n_checked > 50


def test_source_weight_is_the_solid_angle_of_the_focus_rectangle():
    # sum of p0 over launched neutrons / N -> flux * A_src[cm^2] * Omega(focus rect from source) * dlambda
    ins = W.instrument(slit1_xw=1.0, slit1_yh=1.0)      # nothing absorbed at slit 1
    m = W.model(model="flat", scale=1.0)
    p0 = np.array([O.trace_one(ins, m, 3, i).p0 for i in range(4000)])
    omega = 0.005 * 0.005 / 25.0                        # small-angle: A / z^2
    expect = 1.0 * (0.01 * 0.01 * 1e4) * omega * 1.2
    assert abs(p0.mean() / expect - 1) < 1e-5


def test_flat_model_weight_conservation():
    """I == 1/cm: the mean scattered weight per sample-crossing neutron is
    p0 * 100 ell * pi (qmax^2 - qmin^2) / k^2 (total cross-section of the q window)."""
    ins = W.pencil_instrument(det_dist=0.05, det_xw=4.0, det_yh=4.0)   # a detector that catches everything
    m = W.model(model="flat", scale=1.0)
    out = O.trace_range(ins, m, 5, 0, 200000, hist=False)
    assert out["counters"][6] == 200000
    k = TWO_PI / 6.0
    r0 = O.trace_one(ins, m, 5, 0)
    expect = r0.p0 * 100 * 1e-3 * math.pi * (0.3 ** 2 - 0.001 ** 2) / k ** 2
    mean = out["weight"].mean()
    sem = out["weight"].std() / math.sqrt(out["weight"].size)
    assert abs(mean - expect) < 4 * sem and sem < 0.003 * expect


def _expected_pencil_image(ins, model_d, p0, ell, nsub=6):
    """E[P(pixel)]/N = p0 * 100 ell * integral over the pixel of I(q(X,Y)) dOmega,
    dOmega = D dX dY / (D^2+X^2+Y^2)^(3/2), restricted to q in [qmin, qmax]; scattering point at the
    sample centre (sample thickness 1 mm << D)."""
    nx, ny, Wd, H, D = ins["det_nx"], ins["det_ny"], ins["det_xw"], ins["det_yh"], ins["det_dist"]
    k = TWO_PI / ins["lambda_min"]
    g, gw = np.polynomial.legendre.leggauss(nsub)
    xs = (np.arange(nx)[:, None] + 0.5 + 0.5 * g[None, :]) * (Wd / nx) - 0.5 * Wd
    ys = (np.arange(ny)[:, None] + 0.5 + 0.5 * g[None, :]) * (H / ny) - 0.5 * H
    wx = 0.5 * gw * (Wd / nx)
    wy = 0.5 * gw * (H / ny)
    X = xs.reshape(-1)[None, :]
    Y = ys.reshape(-1)[:, None]
    R2 = X * X + Y * Y
    two_theta = np.arctan2(np.sqrt(R2), D)
    q = 2 * k * np.sin(0.5 * two_theta)
    Iq = np.vectorize(lambda qq: O.intensity(model_d, [qq, 0.0, 0.0]))(q)
    Iq = np.where((q >= ins["q_min"]) & (q <= ins["q_max"]), Iq, 0.0)
    f = Iq * D / (D * D + R2) ** 1.5
    f = f.reshape(ny, nsub, nx, nsub)
    return p0 * 100 * ell * np.einsum("iajb,a,b->ij", f, wy, wx)


def test_pencil_beam_image_matches_integrated_intensity_chi2():
    # 16x16 detector at 5 m, monochromatic pencil beam, sphere R = 50 A
    ins = W.pencil_instrument(det_nx=16, det_ny=16, q_min=0.004, q_max=0.3)
    m = W.config(0)["model"]
    n = 600000
    out = O.trace_range(ins, m, 99, 0, n, dump=False)
    r0 = O.trace_one(ins, m, 99, 0)
    E = n * _expected_pencil_image(ins, m, r0.p0, 1e-3).reshape(-1)
    P, P2, N = out["sum_p"], out["sum_p2"], out["counts"]
    ok = N > 30
    # pixels crossed by the q_min circle have a discontinuous integrand: exclude the 4 central ones
    centre = np.zeros((16, 16), bool)
    centre[7:9, 7:9] = True
    ok &= ~centre.reshape(-1)
    z = (P[ok] - E[ok]) / np.sqrt(P2[ok])
    chi2 = float((z * z).mean())
    assert ok.sum() > 200
    assert abs(chi2 - 1) < 5 * math.sqrt(2 / ok.sum()), chi2
    assert (np.abs(z) > 3).mean() <= 0.02
    assert abs(P[ok].sum() / E[ok].sum() - 1) < 0.01
    # 4-fold symmetry of an isotropic image (statistical)
    img = P.reshape(16, 16)
    s = np.sqrt(P2.reshape(16, 16))
    d = (img - img[::-1, ::-1]) / np.sqrt(s ** 2 + s[::-1, ::-1] ** 2 + 1e-300)
    assert np.abs(d[ok.reshape(16, 16)]).max() < 5


def test_attenuation_closed_form_on_axis():
    ins = W.pencil_instrument(src_xw=1e-9, src_yh=1e-9, focus_xw=1e-9, focus_yh=1e-9,
                              mu_abs_2200=30.0, mu_inc=50.0)
    ref = W.pencil_instrument(src_xw=1e-9, src_yh=1e-9, focus_xw=1e-9, focus_yh=1e-9)
    m = W.model(model="flat", scale=1.0)
    k = TWO_PI / 6.0
    n = 0
    for i in range(300):
        a, b = O.trace_one(ins, m, 21, i), O.trace_one(ref, m, 21, i)
        assert a.status == b.status and a.pixel == b.pixel
        if a.status:
            continue
        mu = 30.0 * 6.0 / 1.7982 + 50.0
        d_in = a.u[5] * 1e-3
        two_theta = 2 * math.asin(a.q / (2 * k))
        T = math.exp(-mu * (d_in + (1e-3 - d_in) / math.cos(two_theta)))
        assert abs(a.weight / b.weight - T) < 1e-7 * T
        n += 1
    assert n > 30


def test_cylinder_sample_chord():
    # y-axis cylinder, radius 5 mm: an on-axis ray has chord 2R; a ray displaced by x has 2 sqrt(R^2-x^2)
    ins = W.pencil_instrument(sample_shape="cyl_y", src_xw=1e-9, src_yh=1e-9, focus_xw=1e-9, focus_yh=1e-9)
    m = W.model(model="flat", scale=1.0)
    r = O.trace_one(ins, m, 1, 0)
    assert abs(r.ell - 0.010) < 1e-12
    wide = W.instrument(sample_shape="cyl_y")
    for i in range(2000):
        r = O.trace_one(wide, m, 1, i)
        if r.status in (1, 2):
            continue
        # reconstruct the x of the (nearly parallel) ray at the sample
        x0 = (r.u[0] - 0.5) * 0.01
        xt = (r.u[2] - 0.5) * 0.005
        xs = x0 + (xt - x0) * 5.01 / 5.0
        assert abs(r.ell - 2 * math.sqrt(0.005 ** 2 - xs ** 2)) < 2e-8
    # taller beam than the cylinder: misses above the top are dropped
    short = W.instrument(sample_shape="cyl_y", sample_yh=0.002)
    out = O.trace_range(short, m, 1, 0, 20000, dump=False, hist=False)
    assert out["counters"][3] > 0


def test_unreachable_q_is_dropped():
    ins = W.pencil_instrument(lambda_min=30.0, lambda_max=30.0, q_max=0.6)   # 2k = 0.419 < q_max
    out = O.trace_range(ins, W.model(model="flat", scale=1.0), 2, 0, 5000, hist=False)
    q = out["q"]
    k = TWO_PI / 30.0
    assert out["counters"][4] == (q >= 2 * k).sum() > 0


def test_triangular_wavelength_law_of_a_velocity_selector():
    """R-L1 (the selector fixes the wavelength spread): the wavelengths the oracle draws follow the
    symmetric triangle on [lambda_min, lambda_max] -- mean at the centre, variance (d lambda)^2 / 24,
    Kolmogorov-Smirnov against the triangle's distribution function -- from the same uniform draw 4 as the uniform
    law (continuous at u = 1/2, monotone), and nothing else of the neutron changes."""
    import math
    ins_u = W.instrument()
    ins_t = W.instrument(lambda_dist="triangle")
    lam_u, lam_t = [], []
    c = W.config(0)
    for nid in range(60000):
        ru, rt = O.trace_one(ins_u, c["model"], 99, nid), O.trace_one(ins_t, c["model"], 99, nid)
        if ru.status == 1:                                 # died at slit 1: no wavelength drawn
            continue
        assert ru.status == rt.status or {ru.status, rt.status} <= {0, 4, 5}   # only outcomes that depend on lambda may differ
        assert ru.u[4] == rt.u[4] and ru.p0 == rt.p0 and ru.q == rt.q
        u4 = ru.u[4]
        t = math.sqrt(0.5 * u4) if u4 < 0.5 else 1.0 - math.sqrt(0.5 * (1.0 - u4))
        assert rt.lam == 5.4 + t * (6.6 - 5.4) and ru.lam == 5.4 + u4 * (6.6 - 5.4)
        lam_u.append(ru.lam)
        lam_t.append(rt.lam)
    lam_t = np.sort(np.array(lam_t))
    n = lam_t.size
    assert n > 14000
    d = 6.6 - 5.4
    assert abs(lam_t.mean() - 6.0) < 5 * d / math.sqrt(24 * n)
    assert abs(lam_t.var() - d * d / 24) < 0.03 * d * d / 24
    t = (lam_t - 5.4) / d
    cdf = np.where(t < 0.5, 2 * t * t, 1 - 2 * (1 - t) ** 2)
    ks = np.abs(cdf - (np.arange(n) + 0.5) / n).max()
    assert ks < 1.63 / math.sqrt(n)                        # 1 % level
    # the uniform law is not a triangle (the test has power)
    tu = (np.sort(np.array(lam_u)) - 5.4) / d
    assert np.abs(np.where(tu < 0.5, 2 * tu * tu, 1 - 2 * (1 - tu) ** 2) - (np.arange(n) + 0.5) / n).max() > 5 / math.sqrt(n)
