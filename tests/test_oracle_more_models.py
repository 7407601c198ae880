"""Pins of the oracle's NEXT-2 models: parallelepiped (Eq. 6, Table I group E),
core-shell cylinder and ellipsoid of revolution (Eq. 7, groups A and B).  Each amplitude is checked against
PAPER.md Eq. 1 integrated numerically over the body with numpy Gauss-Legendre rules (nothing of the oracle in
the reference values), plus the reductions to models pinned elsewhere and the Guinier radii."""
import math

import numpy as np

import sas_workloads as W
from oracle import oracle as O


def _gl(n, a, b):
    x, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (b - a) * x + 0.5 * (b + a), 0.5 * (b - a) * w


def _brute_box(Q, a, b, c, n=40):
    """Re integral of exp(-iQ.r) over |x|<=a/2, |y|<=b/2, |z|<=c/2 (Eq. 1, drho = 1)."""
    x, wx = _gl(n, -0.5 * a, 0.5 * a)
    y, wy = _gl(n, -0.5 * b, 0.5 * b)
    z, wz = _gl(n, -0.5 * c, 0.5 * c)
    X, Y, Z = np.meshgrid(x, y, z, indexing="ij")
    return np.einsum("ijk,i,j,k->", np.cos(Q[0] * X + Q[1] * Y + Q[2] * Z), wx, wy, wz)


def _brute_cylinder(Q, R, L, n=48):
    r, wr = _gl(n, 0.0, R)
    ph, wp = _gl(2 * n, 0.0, 2 * math.pi)
    z, wz = _gl(n, -0.5 * L, 0.5 * L)
    RR, P, Z = np.meshgrid(r, ph, z, indexing="ij")
    f = np.cos(Q[0] * RR * np.cos(P) + Q[1] * RR * np.sin(P) + Q[2] * Z) * RR
    return np.einsum("ijk,i,j,k->", f, wr, wp, wz)


def _brute_ellipsoid(Q, a, b, c, n=48):
    r, wr = _gl(n, 0.0, 1.0)
    mu, wm = _gl(n, -1.0, 1.0)
    ph, wp = _gl(2 * n, 0.0, 2 * math.pi)
    R, M, P = np.meshgrid(r, mu, ph, indexing="ij")
    s = np.sqrt(1 - M * M)
    x, y, z = a * R * s * np.cos(P), b * R * s * np.sin(P), c * R * M
    f = np.cos(Q[0] * x + Q[1] * y + Q[2] * z) * (a * b * c) * R * R
    return np.einsum("ijk,i,j,k->", f, wr, wm, wp)


QS = [np.array(v) for v in ((0.02, 0.0, 0.0), (0.0, 0.03, 0.0), (0.0, 0.0, 0.011), (0.013, -0.021, 0.017),
                            (0.07, 0.05, -0.09), (1e-4, 2e-4, -1e-4))]


def test_parallelepiped_is_eq1_integrated():
    a, b, c = 35.0, 75.0, 120.0
    m = W.model(model="parallelepiped", size=[a, b, c, 0], sld=[1.0, 0, 0])
    for Q in QS:
        F, V = O.amplitude(m, *Q)
        assert abs(V - a * b * c) < 1e-9 * V
        assert abs(F - _brute_box(Q, a, b, c)) < 1e-9 * V, Q
    # the common size scale stretches every side (as the triaxial ellipsoid, R-A12)
    F2, V2 = O.amplitude(m, 0.01, 0.02, 0.005, 1.3, 1.0)
    assert abs(V2 - 1.3 ** 3 * a * b * c) < 1e-9 * V2
    assert abs(F2 - _brute_box((0.01, 0.02, 0.005), 1.3 * a, 1.3 * b, 1.3 * c)) < 1e-9 * V2
    # Guinier along an axis: F/V = 1 - (q a)^2/24 + ...   (R_g^2 along A = a^2/12)
    q = 1e-3
    F, V = O.amplitude(m, q, 0.0, 0.0)
    assert abs((1 - F / V) / q ** 2 - a * a / 24) < 1e-3 * a * a / 24
    # which side belongs to which axis: the zero of sinc(Q_B b/2) is at Q_B = 2 pi / b
    F, V = O.amplitude(m, 0.0, 2 * math.pi / b, 0.0)
    assert abs(F) < 1e-12 * V


def test_core_shell_cylinder_is_eq1_with_piecewise_contrast():
    R, L, t, s0, s1 = 20.0, 300.0, 8.0, 3.0, 1.0
    m = W.model(model="core_shell_cylinder", size=[R, L, t, 0], sld=[s0, s1, 0])
    Vt = math.pi * (R + t) ** 2 * (L + 2 * t)
    for Q in QS:
        F, V = O.amplitude(m, *Q)
        ref = (s0 - s1) * _brute_cylinder(Q, R, L) + s1 * _brute_cylinder(Q, R + t, L + 2 * t)
        assert abs(V - Vt) < 1e-9 * Vt
        assert abs(F - ref) < 2e-9 * s0 * Vt, Q
    # equal contrasts: one homogeneous cylinder (R + t, L + 2 t); no shell: the core cylinder
    hom = W.model(model="cylinder", size=[R + t, L + 2 * t, 0, 0], sld=[s1, 0, 0])
    eq = W.model(model="core_shell_cylinder", size=[R, L, t, 0], sld=[s1, s1, 0])
    core = W.model(model="cylinder", size=[R, L, 0, 0], sld=[s0, 0, 0])
    bare = W.model(model="core_shell_cylinder", size=[R, L, 0.0, 0], sld=[s0, 0.7, 0])
    for Q in QS:
        assert abs(O.amplitude(eq, *Q)[0] - O.amplitude(hom, *Q)[0]) < 1e-12 * s1 * Vt
        assert abs(O.amplitude(bare, *Q)[0] - O.amplitude(core, *Q)[0]) < 1e-12 * s0 * Vt
    # the two polydisperse lengths: x0 scales R, x1 scales L, the shell keeps its thickness
    F, V = O.amplitude(m, 0.01, 0.0, 0.004, 1.2, 0.9)
    ref = (s0 - s1) * _brute_cylinder((0.01, 0, 0.004), 1.2 * R, 0.9 * L) + \
        s1 * _brute_cylinder((0.01, 0, 0.004), 1.2 * R + t, 0.9 * L + 2 * t)
    assert abs(F - ref) < 2e-9 * s0 * V and abs(V - math.pi * (1.2 * R + t) ** 2 * (0.9 * L + 2 * t)) < 1e-9 * V


def test_ellipsoid_of_revolution_is_eq1_integrated_and_a_special_triaxial():
    Re, Rp = 30.0, 70.0
    m = W.model(model="ellipsoid", size=[Re, Rp, 0, 0], sld=[1.0, 0, 0])
    tri = W.model(model="triaxial", size=[Re, Re, Rp, 0], sld=[1.0, 0, 0])
    sph = W.model(model="sphere", size=[Re, 0, 0, 0], sld=[1.0, 0, 0])
    V0 = 4 * math.pi / 3 * Re * Re * Rp
    for Q in QS:
        F, V = O.amplitude(m, *Q)
        assert abs(V - V0) < 1e-9 * V0
        assert abs(F - _brute_ellipsoid(Q, Re, Re, Rp)) < 2e-10 * V0, Q
        assert abs(F - O.amplitude(tri, *Q)[0]) < 1e-12 * V0
        # polar radius scaled down to the equatorial one: a sphere
        Fs, Vs = O.amplitude(m, Q[0], Q[1], Q[2], 1.0, Re / Rp)
        assert abs(Fs - O.amplitude(sph, *Q)[0]) < 1e-12 * Vs
    # Guinier along the axis and across it: R_g^2 = R^2/5 per direction
    q = 1e-3
    for Qv, Rr in (((0, 0, q), Rp), ((q, 0, 0), Re)):
        F, V = O.amplitude(m, *Qv)
        assert abs((1 - F / V) / q ** 2 - Rr * Rr / 10) < 1e-3 * Rr * Rr / 10


def test_new_models_trace_end_to_end_and_average_over_nodes():
    # fixed-node polydispersity and per-event sampling both reach the new models through the same tables
    ins = W.instrument(det_dist=3.0)
    for over in (dict(model="parallelepiped", size=[35.0, 75.0, 120.0, 0], pd_kind=["schulz", "none"], pd_rel=[0.1, 0],
                      pd_nodes=[8, 1], orient_kind="isotropic_mc"),
                 dict(model="core_shell_cylinder", size=[20.0, 300.0, 8.0, 0], sld=[3e-6, 1e-6, 0],
                      pd_kind=["schulz", "schulz"], pd_rel=[0.1, 0.05], pd_nodes=[6, 5], theta=1.0, phi=0.3),
                 dict(model="ellipsoid", size=[30.0, 70.0, 0, 0], pd_kind=["gauss_mc", "gauss_mc"], pd_rel=[0.1, 0.1],
                      orient_kind="uniform_angles_mc")):
        md = W.model(**over)
        r = O.trace_range(ins, md, 99, 0, 30000, hist=False)
        det = r["pixel"] >= 0
        assert det.sum() > 1000 and np.all(r["weight"][det] > 0) and np.all(r["weight"][det] <= r["weight_env"][det] * (1 + 1e-12))
    # node average of a separable case by hand: <F^2>/<V> of the parallelepiped over its 8 Schulz nodes
    md = W.model(model="parallelepiped", size=[35.0, 75.0, 120.0, 0], pd_kind=["schulz", "none"], pd_rel=[0.1, 0],
                 pd_nodes=[8, 1], scale=0.02)
    x, w = O.schulz_nodes(0.1, 8)
    Q = (0.02, -0.01, 0.015)
    FV = [O.amplitude(md, *Q, xi, 1.0) for xi in x]
    want = 1e8 * 0.02 * sum(wi * F * F for wi, (F, V) in zip(w, FV)) / sum(wi * V for wi, (F, V) in zip(w, FV))
    assert abs(O.intensity(md, Q) / want - 1) < 1e-13


# ---- R-M2: barbell and capped cylinder (bodies of revolution with spherical end pieces)
def _brute_revolution(Q, pieces, n=64):
    """Re integral of exp(-iQ.r) over a body of revolution about z given as [(z0, z1, rho(z))...] (PAPER.md:37,
    Eq. 1, drho = 1), by Gauss-Legendre in (z, rho, phi) piece by piece; also returns the volume."""
    F = V = 0.0
    ph, wp = _gl(2 * n, 0.0, 2 * math.pi)
    t, wt = _gl(n, 0.0, 1.0)
    for z0, z1, rho in pieces:
        z, wz = _gl(n, z0, z1)
        rmax = rho(z)                                   # (n,)
        Z, T, P = np.meshgrid(z, t, ph, indexing="ij")
        RM = rmax[:, None, None]
        RR = T * RM
        f = np.cos(Q[0] * RR * np.cos(P) + Q[1] * RR * np.sin(P) + Q[2] * Z) * RR * RM
        F += np.einsum("ijk,i,j,k->", f, wz, wt, wp)
        V += np.einsum("i,i->", math.pi * rmax ** 2, wz)
    return F, V


def _pieces(kind, R, L, Rb):
    h = math.sqrt(Rb * Rb - R * R)
    zc = 0.5 * L + h if kind == "barbell" else 0.5 * L - h
    cap = lambda z: np.sqrt(np.maximum(Rb * Rb - (np.abs(z) - zc) ** 2, 0.0))
    return [(-0.5 * L, 0.5 * L, lambda z: np.full_like(z, R)), (0.5 * L, zc + Rb, cap), (-(zc + Rb), -0.5 * L, cap)]


def test_barbell_and_capped_cylinder_are_eq1_integrated_slice_by_slice():
    for kind, R, L, Rb in (("barbell", 20.0, 200.0, 40.0), ("capped_cylinder", 20.0, 200.0, 25.0),
                           ("barbell", 30.0, 90.0, 30.0001), ("capped_cylinder", 30.0, 90.0, 60.0)):
        m = W.model(model=kind, size=[R, L, Rb, 0], sld=[1.0, 0, 0])
        for Q in (np.array(v) for v in ((0.03, 0.0, 0.0), (0.0, 0.0, 0.02), (0.013, -0.021, 0.017), (0.05, 0.04, -0.06),
                                        (1e-4, 2e-4, -1e-4))):
            F, V = O.amplitude(m, *Q)
            Fb, Vb = _brute_revolution(Q, _pieces(kind, R, L, Rb))
            assert abs(V - Vb) < 1e-9 * Vb, (kind, V, Vb)
            assert abs(F - Fb) < 2e-8 * Vb, (kind, Q, F, Fb)
    # closed-form volumes: cylinder + two sphere pieces
    R, L, Rb = 20.0, 200.0, 40.0
    h = math.sqrt(Rb * Rb - R * R)
    v_big = math.pi * (2 * Rb ** 3 / 3 + Rb * Rb * h - h ** 3 / 3)      # sphere part beyond the plane at distance h
    assert abs(O.amplitude(W.model(model="barbell", size=[R, L, Rb, 0]), 0, 0, 0)[1] - (math.pi * R * R * L + 2 * v_big)) < 1e-6
    Rc = 25.0
    hc = math.sqrt(Rc * Rc - R * R)
    v_cap = math.pi * (Rc - hc) ** 2 * (2 * Rc + hc) / 3                 # spherical cap of height Rc - hc
    assert abs(O.amplitude(W.model(model="capped_cylinder", size=[R, L, Rc, 0]), 0, 0, 0)[1] - (math.pi * R * R * L + 2 * v_cap)) < 1e-6
    # a cap radius much larger than R flattens the caps: the capped cylinder tends to the plain cylinder
    cyl = W.model(model="cylinder", size=[R, L, 0, 0], sld=[1.0, 0, 0])
    flat = W.model(model="capped_cylinder", size=[R, L, 1e5, 0], sld=[1.0, 0, 0])
    for Q in ((0.02, 0.0, 0.01), (0.0, 0.03, 0.02)):
        assert abs(O.amplitude(flat, *Q)[0] - O.amplitude(cyl, *Q)[0]) < 1e-4 * O.amplitude(cyl, 0, 0, 0)[1]
    # a barbell of zero length with R -> 0 is two touching spheres: F = 2 V_s Phi(q Rb) cos(Q_C Rb)
    two = W.model(model="barbell", size=[1e-6, 1e-9, 30.0, 0], sld=[1.0, 0, 0])
    Vs = 4 * math.pi / 3 * 30.0 ** 3
    for qc_, qa_ in ((0.02, 0.0), (0.01, 0.03), (0.0, 0.05)):
        q = math.hypot(qc_, qa_)
        u = q * 30.0
        want = 2 * Vs * 3 * (math.sin(u) - u * math.cos(u)) / u ** 3 * math.cos(qc_ * 30.0)
        assert abs(O.amplitude(two, qa_, 0.0, qc_)[0] - want) < 1e-6 * Vs


# ---- R-M3: elliptical cylinder, hollow cylinder, core-shell ellipsoid of revolution
def _brute_elliptic_cylinder(Q, a, b, L, n=48):
    r, wr = _gl(n, 0.0, 1.0)
    ph, wp = _gl(2 * n, 0.0, 2 * math.pi)
    z, wz = _gl(n, -0.5 * L, 0.5 * L)
    RR, P, Z = np.meshgrid(r, ph, z, indexing="ij")
    f = np.cos(Q[0] * a * RR * np.cos(P) + Q[1] * b * RR * np.sin(P) + Q[2] * Z) * RR * (a * b)
    return np.einsum("ijk,i,j,k->", f, wr, wp, wz)


def test_elliptical_cylinder_hollow_cylinder_core_shell_ellipsoid_are_eq1_integrated():
    a, b, L = 20.0, 35.0, 300.0
    m = W.model(model="elliptical_cylinder", size=[a, b, L, 0], sld=[1.0, 0, 0])
    circ = W.model(model="elliptical_cylinder", size=[a, a, L, 0], sld=[1.0, 0, 0])
    cyl = W.model(model="cylinder", size=[a, L, 0, 0], sld=[1.0, 0, 0])
    for Q in QS:
        F, V = O.amplitude(m, *Q)
        assert abs(V - math.pi * a * b * L) < 1e-9 * V
        assert abs(F - _brute_elliptic_cylinder(Q, a, b, L)) < 2e-9 * V, Q
        assert abs(O.amplitude(circ, *Q)[0] - O.amplitude(cyl, *Q)[0]) < 1e-12 * V     # a = b: the circular cylinder
    # which semi-axis belongs to which particle axis: Lambda's first zero (j_{1,1} = 3.8317) along A and along B
    assert abs(O.amplitude(m, 3.8317059702 / a, 0.0, 0.0)[0]) < 1e-8 * math.pi * a * b * L
    assert abs(O.amplitude(m, 0.0, 3.8317059702 / b, 0.0)[0]) < 1e-8 * math.pi * a * b * L
    # x0 scales both semi-axes, x1 the length
    F, V = O.amplitude(m, 0.01, 0.02, 0.005, 1.2, 0.8)
    assert abs(F - _brute_elliptic_cylinder((0.01, 0.02, 0.005), 1.2 * a, 1.2 * b, 0.8 * L)) < 2e-9 * V

    Ri, Lh, t = 20.0, 300.0, 8.0
    hol = W.model(model="hollow_cylinder", size=[Ri, Lh, t, 0], sld=[1.0, 0, 0])
    Vw = math.pi * ((Ri + t) ** 2 - Ri ** 2) * Lh
    for Q in QS:
        F, V = O.amplitude(hol, *Q)
        ref = _brute_cylinder(Q, Ri + t, Lh) - _brute_cylinder(Q, Ri, Lh)
        assert abs(V - Vw) < 1e-9 * Vw and abs(F - ref) < 5e-9 * math.pi * (Ri + t) ** 2 * Lh, Q
    # the same body as a core-shell cylinder whose core has the solvent's contrast and whose caps are missing:
    # for Q perpendicular to the axis the caps do not matter in the radial factor
    F0, V0 = O.amplitude(W.model(model="hollow_cylinder", size=[1e-9, Lh, t, 0], sld=[1.0, 0, 0]), 0.02, 0.01, 0.003)
    Fc, Vc = O.amplitude(W.model(model="cylinder", size=[t, Lh, 0, 0], sld=[1.0, 0, 0]), 0.02, 0.01, 0.003)
    assert abs(F0 - Fc) < 1e-9 * Vc                       # no hole: a solid cylinder of radius t

    Re, Rp, ts, s0, s1 = 30.0, 70.0, 8.0, 3.0, 1.0
    cse = W.model(model="core_shell_ellipsoid", size=[Re, Rp, ts, 0], sld=[s0, s1, 0])
    Vt = 4 * math.pi / 3 * (Re + ts) ** 2 * (Rp + ts)
    for Q in QS:
        F, V = O.amplitude(cse, *Q)
        ref = (s0 - s1) * _brute_ellipsoid(Q, Re, Re, Rp) + s1 * _brute_ellipsoid(Q, Re + ts, Re + ts, Rp + ts)
        assert abs(V - Vt) < 1e-9 * Vt and abs(F - ref) < 1e-9 * s0 * Vt, Q
    # equal contrasts: the homogeneous ellipsoid (R_e + t, R_p + t); R_e = R_p: the core-shell sphere
    hom = W.model(model="ellipsoid", size=[Re + ts, Rp + ts, 0, 0], sld=[s1, 0, 0])
    eq = W.model(model="core_shell_ellipsoid", size=[Re, Rp, ts, 0], sld=[s1, s1, 0])
    css = W.model(model="core_shell_sphere", size=[Re, ts, 0, 0], sld=[s0, s1, 0])
    rnd = W.model(model="core_shell_ellipsoid", size=[Re, Re, ts, 0], sld=[s0, s1, 0])
    for Q in QS:
        assert abs(O.amplitude(eq, *Q)[0] - O.amplitude(hom, *Q)[0]) < 1e-12 * s1 * Vt
        assert abs(O.amplitude(rnd, *Q)[0] - O.amplitude(css, *Q)[0]) < 1e-12 * s0 * Vt
