"""Pins of the oracle's RNG, form factors, structure factor and quadrature tables
against things that are NOT the oracle: published known-answer vectors, brute-force
integration of PAPER.md Eq. 1, the Ornstein-Zernike integral of the PY direct
correlation function, closed-form moments, Guinier radii, the paper's own
Q_min = 0.032 1/A pin."""
import math
import os

import numpy as np
import pytest

import sas_workloads as W
from oracle import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold_lines(name):
    with open(os.path.join(GOLD, name)) as f:
        return [l.split() for l in f if l.strip() and not l.startswith("#")]


# ------------------------------------------------------------------ Philox
def test_philox_known_answers():
    for t in _gold_lines("philox_kat.txt"):
        v = [int(x, 16) for x in t]
        assert O.philox(v[0:4], v[4:6]) == v[6:10]


def test_philox_is_a_bijection_on_counters_and_sensitive_to_every_input_word():
    base = O.philox([1, 2, 3, 4], [5, 6])
    seen = {tuple(base)}
    for i in range(4):
        c = [1, 2, 3, 4]
        c[i] ^= 1
        seen.add(tuple(O.philox(c, [5, 6])))
    for i in range(2):
        k = [5, 6]
        k[i] ^= 1
        seen.add(tuple(O.philox([1, 2, 3, 4], k)))
    assert len(seen) == 7


def test_uniform_conversion_is_exact_and_open():
    L = O.lib()
    assert L.orc_uniform(0) == 2.0 ** -33
    assert L.orc_uniform(0xFFFFFFFF) == 1.0 - 2.0 ** -33
    assert L.orc_uniform(0x80000000) == 0.5 + 2.0 ** -33


def test_uniform_stream_moments():
    # mean 1/2, variance 1/12 of the uniforms of 50k consecutive counters
    u = np.array([O.philox([i, 0, 0, 0], [20250106, 0]) for i in range(50000)], dtype=np.float64)
    u = (u + 0.5) / 2.0 ** 32
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / u.size)
    assert abs(u.var() - 1 / 12) < 0.002
    assert abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.02


# ------------------------------------------------- brute force of Eq. 1
def _gl(n, a, b):
    x, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (b - a) * x + 0.5 * (b + a), 0.5 * (b - a) * w


def _brute_ellipsoid(Q, a, b, c, n=48):
    """Re integral of exp(-iQ.r) over the ellipsoid x^2/a^2+y^2/b^2+z^2/c^2<=1 (Eq. 1
    with drho = 1), by Gauss-Legendre in stretched spherical coordinates."""
    r, wr = _gl(n, 0.0, 1.0)
    mu, wm = _gl(n, -1.0, 1.0)
    ph, wp = _gl(2 * n, 0.0, 2 * math.pi)
    R, M, P = np.meshgrid(r, mu, ph, indexing="ij")
    s = np.sqrt(1 - M * M)
    x, y, z = a * R * s * np.cos(P), b * R * s * np.sin(P), c * R * M
    f = np.cos(Q[0] * x + Q[1] * y + Q[2] * z) * (a * b * c) * R * R
    return np.einsum("ijk,i,j,k->", f, wr, wm, wp)


def _brute_cylinder(Q, R, L, n=48):
    """Same for a cylinder of radius R, length L, axis z."""
    r, wr = _gl(n, 0.0, R)
    ph, wp = _gl(2 * n, 0.0, 2 * math.pi)
    z, wz = _gl(n, -0.5 * L, 0.5 * L)
    RR, P, Z = np.meshgrid(r, ph, z, indexing="ij")
    f = np.cos(Q[0] * RR * np.cos(P) + Q[1] * RR * np.sin(P) + Q[2] * Z) * RR
    return np.einsum("ijk,i,j,k->", f, wr, wp, wz)


def test_sphere_amplitude_is_eq1_integrated():
    m = W.model(model="sphere", size=[50.0, 0, 0, 0], sld=[1.0, 0, 0])
    for q in (0.001, 0.004, 0.0099, 0.0101, 0.03, 0.0899, 0.13, 0.3):
        Q = np.array([0.3, -0.5, 0.81]) / np.linalg.norm([0.3, -0.5, 0.81]) * q
        F, V = O.amplitude(m, *Q)
        ref = _brute_ellipsoid(Q, 50.0, 50.0, 50.0)
        assert abs(F - ref) < 2e-10 * V, (q, F, ref)
        assert abs(V - 4 * math.pi / 3 * 50.0 ** 3) < 1e-9 * V


def test_sphere_closed_form_values_and_limits():
    L = O.lib()
    assert L.orc_sphere_phi(0.0) == 1.0
    # first zero of the sphere form factor: tan u = u
    assert abs(L.orc_sphere_phi(4.493409457909064)) < 1e-15
    for t in _gold_lines("worked_example_c0.txt"):
        if t[0] == "sphereP":
            q, P = float(t[1]), float(t[2])
            assert abs(L.orc_sphere_phi(q * 50.0) ** 2 - P) < 2e-12 * max(P, 1e-3)
    # series and direct branch meet at u = 0.5 (a wrong series coefficient shows here)
    lo, hi = L.orc_sphere_phi(0.5 - 1e-9), L.orc_sphere_phi(0.5 + 1e-9)
    assert abs(lo - hi) < 1e-9
    # Guinier: Phi^2 ~ exp(-u^2/5)  => R_g^2 = 3 R^2/5
    u = 1e-2
    assert abs((1 - L.orc_sphere_phi(u) ** 2) / u ** 2 - 0.2) < 1e-5
    # I(0.01) for c0 in 1/cm (scale 0.01, drho 1e-6, R 50): survey closed-form value
    I = O.intensity(W.config(0)["model"], [0.01, 0.0, 0.0])
    assert abs(I - 4.979729654907e-01) < 1e-11


def test_sphere_phi_against_mpmath_everywhere():
    import mpmath as mp
    mp.mp.dps = 40
    L = O.lib()
    for u in list(np.geomspace(1e-6, 60.0, 200)) + [0.4999999, 0.5, 0.5000001]:
        ref = 3 * (mp.sin(u) - mp.mpf(u) * mp.cos(u)) / mp.mpf(u) ** 3
        assert abs(L.orc_sphere_phi(float(u)) - float(ref)) < 3e-15 * max(1.0, u) / max(u, 1.0) ** 2 + 2e-16


def test_cylinder_amplitude_is_eq1_integrated_and_eq9_is_swapped_as_printed():
    m = W.model(model="cylinder", size=[20.0, 400.0, 0, 0], sld=[1.0, 0, 0])
    V = math.pi * 20.0 ** 2 * 400.0
    for Q in ([0.1, 0.0, 0.0], [0.0, 0.0, 0.02], [0.03, 0.04, 0.011], [0.002, 0.0, 0.001], [0.2, 0.1, 0.05]):
        F, vol = O.amplitude(m, *Q)     # particle frame: (Q_A, Q_B, Q_C), axis = C
        ref = _brute_cylinder(Q, 20.0, 400.0, n=64)
        assert abs(vol - V) < 1e-9 * V
        assert abs(F - ref) < 1e-9 * V, (Q, F / V, ref / V)
    # values quoted in SURVEY.md A4 from an independent brute force
    assert abs(O.amplitude(m, 0.1, 0, 0)[0] / V - 0.5767) < 2e-4
    assert abs(O.amplitude(m, 0, 0, 0.02)[0] / V + 0.18920) < 1e-4
    # Q parallel to the axis -> sinc(qL/2); perpendicular -> 2 J1(qR)/(qR)
    from scipy.special import j1
    assert abs(O.amplitude(m, 0, 0, 0.013)[0] / V - math.sin(2.6) / 2.6) < 1e-14
    assert abs(O.amplitude(m, 0.06, 0.08, 0)[0] / V - 2 * j1(2.0) / 2.0) < 1e-14


def test_lambda1_against_mpmath():
    import mpmath as mp
    mp.mp.dps = 40
    L = O.lib()
    assert L.orc_lambda1(0.0) == 1.0
    for x in np.concatenate([np.geomspace(1e-9, 1.0, 40), np.linspace(1.0, 65.0, 400)]):
        ref = float(2 * mp.besselj(1, x) / x)
        assert abs(L.orc_lambda1(float(x)) - ref) < 4e-16 * max(1.0, 1.0 / x ** 1.5) + 2e-16, x


def test_triaxial_ellipsoid_is_eq1_integrated_and_reduces_to_sphere():
    m = W.model(model="triaxial", size=[30.0, 50.0, 80.0, 0], sld=[2.0, 0, 0])
    V = 4 * math.pi / 3 * 30 * 50 * 80
    for Q in ([0.05, 0.0, 0.0], [0.0, 0.05, 0.0], [0.0, 0.0, 0.05], [0.02, -0.03, 0.01], [0.1, 0.1, 0.1]):
        F, vol = O.amplitude(m, *Q)
        ref = 2.0 * _brute_ellipsoid(Q, 30.0, 50.0, 80.0, n=56)
        assert abs(vol - V) < 1e-9 * V
        assert abs(F - ref) < 1e-9 * 2 * V, (Q, F, ref)
    ms = W.model(model="triaxial", size=[50.0, 50.0, 50.0, 0])
    sp = W.model(model="sphere", size=[50.0, 0, 0, 0])
    for Q in ([0.01, 0.02, 0.03], [0.1, 0, 0]):
        assert abs(O.amplitude(ms, *Q)[0] - O.amplitude(sp, *Q)[0]) < 1e-12 * abs(O.amplitude(sp, 0, 0, 0)[0])


def test_core_shell_models_piecewise_contrast_and_reductions():
    # core-shell sphere = Eq. 1 with piecewise drho: drho_c inside Rc, drho_s in the shell
    cs = W.model(model="core_shell_sphere", size=[40.0, 10.0, 0, 0], sld=[3.0, 1.0, 0])
    for q in (0.005, 0.05, 0.2):
        Q = [0.0, q, 0.0]
        core = _brute_ellipsoid(Q, 40.0, 40.0, 40.0)
        tot = _brute_ellipsoid(Q, 50.0, 50.0, 50.0)
        ref = 3.0 * core + 1.0 * (tot - core)
        F, V = O.amplitude(cs, *Q)
        assert abs(F - ref) < 1e-9 * V
        assert abs(V - 4 * math.pi / 3 * 50.0 ** 3) < 1e-9 * V
    # equal contrasts -> homogeneous sphere of radius Rc + t ; shell contrast 0 -> core only
    eq = W.model(model="core_shell_sphere", size=[40.0, 10.0, 0, 0], sld=[2.0, 2.0, 0])
    sp = W.model(model="sphere", size=[50.0, 0, 0, 0], sld=[2.0, 0, 0])
    co = W.model(model="core_shell_sphere", size=[40.0, 10.0, 0, 0], sld=[2.0, 0.0, 0])
    s4 = W.model(model="sphere", size=[40.0, 0, 0, 0], sld=[2.0, 0, 0])
    for q in (0.01, 0.07, 0.25):
        assert abs(O.amplitude(eq, q, 0, 0)[0] - O.amplitude(sp, q, 0, 0)[0]) < 1e-9
        assert abs(O.amplitude(co, q, 0, 0)[0] - O.amplitude(s4, q, 0, 0)[0]) < 1e-9
    # core-shell triaxial: piecewise contrast on nested ellipsoids (a+t, b+t, c+t)   (R-A12)
    ct = W.model(model="core_shell_triaxial", size=[30.0, 50.0, 80.0, 10.0], sld=[3.0, 1.0, 0])
    for Q in ([0.03, 0.0, 0.0], [0.01, 0.02, -0.015], [0.0, 0.0, 0.08]):
        core = _brute_ellipsoid(Q, 30.0, 50.0, 80.0, n=56)
        tot = _brute_ellipsoid(Q, 40.0, 60.0, 90.0, n=56)
        F, V = O.amplitude(ct, *Q)
        assert abs(F - (3.0 * core + (tot - core))) < 1e-9 * V * 3
        assert abs(V - 4 * math.pi / 3 * 40 * 60 * 90) < 1e-9 * V


# --------------------------------------------------------------- PY S(q)
def _py_sq_by_ornstein_zernike(q, R, phi):
    """S = 1/(1 - rho c^(q)) with the Wertheim/Thiele PY direct correlation function
    c(s) = -(alpha + beta s + gamma s^3), s = r/sigma < 1, transformed numerically."""
    sig = 2.0 * R
    alpha = (1 + 2 * phi) ** 2 / (1 - phi) ** 4
    beta = -6 * phi * (1 + phi / 2) ** 2 / (1 - phi) ** 4
    gamma = phi * alpha / 2
    s, w = _gl(200, 0.0, 1.0)
    c = -(alpha + beta * s + gamma * s ** 3)
    x = q * sig * s
    ch = 4 * math.pi * sig ** 3 * np.sum(w * s * s * c * np.sinc(x / math.pi))
    rho = 6 * phi / (math.pi * sig ** 3)
    return 1.0 / (1.0 - rho * ch)


def test_py_structure_factor():
    L = O.lib()
    # compressibility limit and dilute limit
    assert abs(L.orc_py_sq(1e-9, 40.0, 0.2) - (1 - 0.2) ** 4 / (1 + 0.4) ** 2) < 1e-12
    assert abs(L.orc_py_sq(0.05, 40.0, 1e-12) - 1.0) < 1e-10
    assert abs(L.orc_py_sq(50.0, 40.0, 0.2) - 1.0) < 1e-5
    for t in _gold_lines("py_sq_mpmath.txt"):
        assert abs(L.orc_py_sq(float(t[0]), 40.0, 0.2) - float(t[1])) < 2e-12
    # numerical Ornstein-Zernike transform: pins t1,t2,t3, both branches and the series coefficients
    for phi in (0.05, 0.2, 0.45):
        for q in list(np.geomspace(1e-4, 0.3, 60)) + [0.0124999, 0.0125, 0.0125001]:
            ref = _py_sq_by_ornstein_zernike(q, 40.0, phi)
            assert abs(L.orc_py_sq(float(q), 40.0, phi) - ref) < 2e-12 * max(1.0, ref), (phi, q)


# ------------------------------------------------------------ quadrature
def test_schulz_nodes_moments():
    for p, n in ((0.15, 32), (0.1, 16), (0.3, 20), (0.05, 8)):
        z = 1 / p ** 2 - 1
        s, w = O.schulz_nodes(p, n)
        assert np.all(s > 0) and np.all(w > 0)
        assert abs(w.sum() - 1) < 1e-14
        assert abs((w * s).sum() - 1) < 1e-13
        assert abs((w * s ** 2).sum() - (1 + p * p)) < 1e-13
        m6 = np.prod([(z + k) for k in range(1, 7)]) / (z + 1) ** 6
        assert abs((w * s ** 6).sum() - m6) < 1e-12 * m6
    s, w = O.schulz_nodes(0.15, 32)
    assert abs((w * s ** 6).sum() - 1.383165055808594) < 1e-12   # SURVEY 8(c) D value
    assert O.schulz_nodes(0.0, 32)[0].tolist() == [1.0]


def test_schulz_rule_equals_dense_integral_of_the_distribution():
    from scipy.special import gammaln
    p, Rm = 0.15, 40.0
    z = 1 / p ** 2 - 1
    m = W.config(1)["model"]
    m["sq_kind"] = "none"
    r = np.linspace(1e-3, 160.0, 400001)
    logf = (z + 1) * math.log((z + 1) / Rm) + z * np.log(r) - (z + 1) * r / Rm - gammaln(z + 1)
    f = np.exp(logf)
    L = O.lib()
    V = 4 * math.pi / 3 * r ** 3
    for q in (0.001, 0.02, 0.11, 0.3):
        phi = np.array([L.orc_sphere_phi(float(q * ri)) for ri in r[::40]])
        F2 = (1e-6 * V[::40] * phi) ** 2
        num = np.trapezoid(f[::40] * F2, r[::40])
        den = np.trapezoid(f * V, r)
        ref = 1e8 * 0.2 * num / den
        got = O.intensity(m, [q, 0, 0])
        assert abs(got - ref) < 1e-6 * ref, (q, got, ref)


def test_gauss_orientation_quadrature_against_brute_force_and_limits():
    c2 = W.config(2)["model"]
    fine = dict(c2, n_theta=64, n_phi=64)
    for Q in ([0.01, 0.0, 0.0005], [0.03, 0.04, 0.001], [0.0, 0.08, 0.003]):
        a, b = O.intensity(c2, Q), O.intensity(fine, Q)
        assert abs(a - b) < 2e-4 * b
    # independent brute force: dense trapezoid over the two tilts, same Gaussian weights
    sig = c2["sigma_theta"]
    d = np.linspace(-3 * sig, 3 * sig, 601)
    g = np.exp(-d * d / (2 * sig * sig))
    g /= g.sum()
    Q = np.array([0.03, 0.04, 0.001])
    from scipy.special import j1
    DT, DP = np.meshgrid(d, d, indexing="ij")
    cx, cy, cz = np.sin(DT) * np.cos(DP), np.sin(DP), np.cos(DT) * np.cos(DP)
    qc = Q[0] * cx + Q[1] * cy + Q[2] * cz
    qab = np.sqrt(np.maximum(Q @ Q - qc * qc, 0))
    V = math.pi * 20.0 ** 2 * 400.0
    F = 2e-6 * V * np.sinc(qc * 200.0 / math.pi) * 2 * j1(qab * 20.0) / (qab * 20.0)
    ref = 1e8 * 0.01 * np.einsum("ij,i,j->", F * F, g, g) / V
    assert abs(O.intensity(c2, Q) - ref) < 2e-3 * ref
    # sigma -> 0 and n = 1 both reduce to the fixed orientation
    fixed = dict(c2, orient_kind="fixed")
    tiny = dict(c2, sigma_theta=1e-9, sigma_phi=1e-9)
    assert abs(O.intensity(tiny, Q) - O.intensity(fixed, Q)) < 1e-9 * O.intensity(fixed, Q)


def test_orientation_angles_convention():
    # R-A7: theta from the beam axis (+z), phi azimuth from +x. A long thin rod scatters in the
    # plane perpendicular to its axis: intensity is maximal for Q perpendicular to c^.
    th, ph = math.radians(60), math.radians(60)
    rod = W.model(model="cylinder", size=[5.0, 2000.0, 0, 0], theta=th, phi=ph)
    c = np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
    perp = np.cross(c, [0, 0, 1.0])
    perp /= np.linalg.norm(perp)
    assert O.intensity(rod, 0.02 * perp) > 100 * O.intensity(rod, 0.02 * c)
    # psi spins about c^: a triaxial ellipsoid with theta = 0 and psi = 90 deg swaps a and b
    e0 = W.model(model="triaxial", size=[30.0, 50.0, 80.0, 0], psi=0.0)
    e9 = W.model(model="triaxial", size=[50.0, 30.0, 80.0, 0], psi=math.pi / 2)
    for Q in ([0.03, 0.01, 0.0], [0.0, 0.05, 0.01]):
        assert abs(O.intensity(e0, Q) - O.intensity(e9, Q)) < 1e-9 * O.intensity(e0, Q)


def test_isotropic_orientation_average_guinier_and_paper_pin():
    # Guinier radius of an isotropically averaged cylinder: Rg^2 = R^2/2 + L^2/12
    cyl = W.model(model="cylinder", size=[20.0, 100.0, 0, 0], orient_kind="isotropic_mc")
    mu, w = _gl(64, 0.0, 1.0)

    def iso(model, q):
        # average over cos(theta) of the axis relative to Q; u_or[0] = (1 - cos)/2
        return sum(wi * O.intensity(model, [0, 0, q], (0.5 * (1 - m_), 0.3, 0.7)) for m_, wi in zip(mu, w))

    q = 2e-3
    rg2 = 20.0 ** 2 / 2 + 100.0 ** 2 / 12
    assert abs((1 - iso(cyl, q) / iso(cyl, 1e-7)) / q ** 2 - rg2 / 3) < 2e-3 * rg2 / 3
    # randomly oriented cylinder R = 119 A (L = 800 A) has its lowest-Q minimum at
    # Q_min ~ 0.032 1/A (R = 3.78 / Q_min)
    mic = W.model(model="cylinder", size=[119.0, 800.0, 0, 0], orient_kind="isotropic_mc")
    mu, w = _gl(400, 0.0, 1.0)
    qs = np.linspace(0.02, 0.045, 126)
    vals = [sum(wi * O.intensity(mic, [0, 0, float(qq)], (0.5 * (1 - m_), 0.1, 0.2)) for m_, wi in zip(mu, w))
            for qq in qs]
    qmin = qs[int(np.argmin(vals))]
    assert 0.0315 <= qmin <= 0.0335, qmin


def test_isotropic_mc_draws_are_isotropic():
    # R-A3: cos(theta) = 1 - 2 u. For a thin rod along c^, <(Q^.c^)^2> over draws must be 1/3.
    e = W.model(model="triaxial", size=[30.0, 50.0, 80.0, 0], orient_kind="isotropic_mc")
    s = W.model(model="triaxial", size=[30.0, 50.0, 80.0, 0])
    # u = (0,*,*) -> cos theta = 1 -> c^ = +z: equals fixed theta = 0 with psi = phi_draw + psi_draw
    v = O.intensity(e, [0.02, 0.01, 0.03], (0.0, 0.0, 0.0))
    assert abs(v - O.intensity(s, [0.02, 0.01, 0.03])) < 1e-12 * v
    # u0 = 0.5 -> theta = 90 deg, phi = 2 pi u1
    v = O.intensity(e, [0.02, 0.01, 0.03], (0.5, 0.25, 0.0))
    s90 = dict(s, theta=math.pi / 2, phi=math.pi / 2)
    assert abs(v - O.intensity(s90, [0.02, 0.01, 0.03])) < 1e-9 * v
