"""Pins of the oracle's thin-walled hollow rectangular prism (DESIGN.md R-M5; PAPER.md:201 names "Hollow rectangular
prism thin walls" among the models expensive enough for the GPU to win at 1e8 neutrons).  The amplitude is PAPER.md
Eq. 1 with the contrast confined to the six faces: checked against (1) that surface integral done numerically with
numpy Gauss-Legendre rules, face by face (nothing of the oracle in the reference), (2) the difference of two
parallelepipeds -- a model pinned on its own in test_oracle_more_models.py -- whose sides differ by a small wall
thickness, (3) the forward value, the closed form along an axis and the first zero of the end-face term."""
import math

import numpy as np

import sas_workloads as W
from oracle import oracle as O


def _gl(n, a, b):
    x, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (b - a) * x + 0.5 * (b + a), 0.5 * (b - a) * w


def _brute_faces(Q, a, b, c, n=64):
    """Re of the integral of exp(-i Q.r) over the six faces of the box |x|<=a/2, |y|<=b/2, |z|<=c/2."""
    tot = 0.0
    sides = (a, b, c)
    for k in range(3):                                   # the pair of faces perpendicular to axis k
        i, j = [ax for ax in range(3) if ax != k]
        u, wu = _gl(n, -0.5 * sides[i], 0.5 * sides[i])
        v, wv = _gl(n, -0.5 * sides[j], 0.5 * sides[j])
        U, V = np.meshgrid(u, v, indexing="ij")
        for sgn in (-1.0, 1.0):
            phase = Q[i] * U + Q[j] * V + Q[k] * (sgn * 0.5 * sides[k])
            tot += np.einsum("ij,i,j->", np.cos(phase), wu, wv)
    return tot


QS = [np.array(v) for v in ((0.02, 0.0, 0.0), (0.0, 0.03, 0.0), (0.0, 0.0, 0.011), (0.013, -0.021, 0.017),
                            (0.07, 0.05, -0.09), (1e-4, 2e-4, -1e-4), (0.21, -0.13, 0.08))]
A, B, C_, T = 35.0, 75.0, 120.0, 2.0


def test_hollow_prism_is_eq1_over_its_faces():
    m = W.model(model="hollow_prism_thin", size=[A, B, C_, T], sld=[1.0, 0, 0])
    area = 2.0 * (A * B + B * C_ + C_ * A)
    for Q in QS:
        F, V = O.amplitude(m, *Q)
        assert abs(V - T * area) < 1e-12 * V
        assert abs(F - T * _brute_faces(Q, A, B, C_)) < 1e-9 * V, Q
    # the common size scale stretches the three sides, not the wall
    F2, V2 = O.amplitude(m, 0.01, 0.02, 0.005, 1.3, 1.0)
    assert abs(V2 - 1.3 ** 2 * T * area) < 1e-12 * V2
    assert abs(F2 - T * _brute_faces((0.01, 0.02, 0.005), 1.3 * A, 1.3 * B, 1.3 * C_)) < 1e-9 * V2
    # the contrast multiplies the amplitude
    m3 = W.model(model="hollow_prism_thin", size=[A, B, C_, T], sld=[3.0e-6, 0, 0])
    assert abs(O.amplitude(m3, *QS[3])[0] - 3.0e-6 * O.amplitude(m, *QS[3])[0]) < 1e-20


def test_hollow_prism_is_the_thin_wall_limit_of_two_parallelepipeds():
    """A wall of thickness t centred on the faces = box (a+t, b+t, c+t) minus box (a-t, b-t, c-t); to first order in
    t that is t x the surface integral (the next term is of relative order (t / side)^2)."""
    t = 0.02
    outer = W.model(model="parallelepiped", size=[A + t, B + t, C_ + t, 0], sld=[1.0, 0, 0])
    inner = W.model(model="parallelepiped", size=[A - t, B - t, C_ - t, 0], sld=[1.0, 0, 0])
    thin = W.model(model="hollow_prism_thin", size=[A, B, C_, t], sld=[1.0, 0, 0])
    for Q in QS:
        d = O.amplitude(outer, *Q)[0] - O.amplitude(inner, *Q)[0]
        F, V = O.amplitude(thin, *Q)
        assert abs(d - F) < 2e-6 * V, (Q, d, F)
    Vo, Vi = O.amplitude(outer, 0, 0, 0)[1], O.amplitude(inner, 0, 0, 0)[1]
    assert abs((Vo - Vi) - O.amplitude(thin, 0, 0, 0)[1]) < 1e-6 * (Vo - Vi)


def test_hollow_prism_closed_forms():
    m = W.model(model="hollow_prism_thin", size=[A, B, C_, T], sld=[2.0, 0, 0])
    F0, V = O.amplitude(m, 0.0, 0.0, 0.0)
    assert abs(F0 - 2.0 * V) < 1e-12 * F0                                   # forward scattering: contrast x volume
    # along A: the end faces give 2 bc cos(q a/2), the four side walls 2 (ab + ac) sinc(q a/2)
    for q in (0.003, 0.05, 0.19):
        x = 0.5 * q * A
        want = 2.0 * T * 2.0 * (B * C_ * math.cos(x) + (A * B + A * C_) * math.sin(x) / x)
        assert abs(O.amplitude(m, q, 0.0, 0.0)[0] - want) < 1e-12 * abs(F0)
    # a flat plate (c -> 0 against a, b) seen along its normal: the two large faces dominate, F ~ 2 t ab cos(q c/2)
    plate = W.model(model="hollow_prism_thin", size=[4000.0, 4000.0, 10.0, 0.5], sld=[1.0, 0, 0])
    q = math.pi / 10.0                                                       # cos(q c / 2) = 0: the faces cancel
    Fz = O.amplitude(plate, 0.0, 0.0, q)[0]
    side = 2.0 * 0.5 * 2.0 * 4000.0 * 10.0 * math.sin(q * 5.0) / (q * 5.0)   # what the four side walls leave
    assert abs(Fz - side) < 1e-9 * abs(side)
    # intensity: Eq. 4 with the wall volume (R-A2), even in Q, background added
    mi = W.model(model="hollow_prism_thin", size=[A, B, C_, T], sld=[1.5e-6, 0, 0], scale=0.02, background=0.003)
    Q = np.array([0.021, -0.017, 0.009])
    F, V = O.amplitude(mi, *Q)
    want = 1.0e8 * 0.02 * F * F / V + 0.003
    assert abs(O.intensity(mi, Q) - want) < 1e-13 * want and O.intensity(mi, -Q) == O.intensity(mi, Q)


def test_hollow_prism_random_orientation_average_falls_as_a_surface():
    """The orientation average of a thin shell decays as q^-2 (a surface), not q^-4 (a solid): the ratio of the
    averages at q and 2q over many random orientations, well above 1 / side, is ~4 within the oscillations."""
    m = O.make_model(W.model(model="hollow_prism_thin", size=[60.0, 80.0, 100.0, 1.0], sld=[1.0, 0, 0], orient_kind="isotropic_mc"))
    rng = np.random.default_rng(5)
    u = rng.random((6000, 3))

    def avg(q):
        return np.mean([O.intensity(m, (0.0, 0.0, q), tuple(ui)) for ui in u])

    lo = np.mean([avg(q) for q in np.linspace(0.28, 0.32, 5)])
    hi = np.mean([avg(q) for q in np.linspace(0.56, 0.64, 5)])
    assert 3.0 < lo / hi < 5.5, lo / hi
