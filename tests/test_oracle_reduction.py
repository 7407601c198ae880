"""Pins of the oracle's ring average (NEXT-4, DESIGN.md R-R1) against things that are not the oracle: the closed-form
solid angle of a rectangle seen from its axis, the normalisation on a synthetic image of known intensity, the ring of
a single hot pixel worked out by hand, conservation of the summed weights, and the first zero of the sphere form
factor at qR = 4.4934 on an analytic image."""
import math

import numpy as np

import sas_workloads as W
from oracle import oracle as O


def _pixel_grid(ins):
    nx, ny, Wd, H = ins["det_nx"], ins["det_ny"], ins["det_xw"], ins["det_yh"]
    X = (np.arange(nx) + 0.5) * (Wd / nx) - 0.5 * Wd
    Y = (np.arange(ny) + 0.5) * (H / ny) - 0.5 * H
    return np.meshgrid(X, Y)


def test_solid_angles_add_up_to_the_rectangle_seen_from_the_sample():
    # I == 1 per steradian per neutron on every pixel: P_pix = dOmega_pix.  Reducing P = 1 on one wide ring gives
    # I = npix / sum(dOmega), so sum(dOmega) comes out of the oracle: compare with the closed form
    # Omega = 4 atan(a b / (d sqrt(a^2 + b^2 + d^2))) of a (2a x 2b) rectangle at distance d on its axis
    ins = W.instrument(det_nx=200, det_ny=160, det_xw=0.6, det_yh=0.4, det_dist=3.0)
    ones = np.ones((160, 200))
    q, I, s, n = O.reduce_radial(ins, ones, ones, 1.0, 6.0, 0.0, 10.0, 1)
    assert n[0] == 200 * 160
    omega_sum = n[0] / I[0]
    a, b, d = 0.3, 0.2, 3.0
    omega = 4 * math.atan(a * b / (d * math.sqrt(a * a + b * b + d * d)))
    assert abs(omega_sum / omega - 1) < 2e-6            # midpoint rule on 200 x 160 pixels


def test_normalisation_ring_assignment_and_errors():
    ins = W.instrument(det_nx=64, det_ny=64)
    lam, D = 5.0, ins["det_dist"]
    # one hot pixel: its ring worked out by hand
    P = np.zeros((64, 64)); P2 = np.zeros((64, 64))
    iy, ix = 40, 51
    P[iy, ix] = 3.0; P2[iy, ix] = 9.0
    X = (ix + 0.5) * 0.5 / 64 - 0.25; Y = (iy + 0.5) * 0.5 / 64 - 0.25
    r = math.hypot(X, Y)
    qpix = 4 * math.pi / lam * math.sin(0.5 * math.atan(r / D))
    q, I, s, n = O.reduce_radial(ins, P, P2, 7.0, lam, 0.0, 0.1, 50)
    b = int(qpix / 0.1 * 50)
    assert np.count_nonzero(I) == 1 and I[b] > 0 and abs(q[b] - (b + 0.5) * 0.002) < 1e-15
    # the ring holds other pixels too: I = P / (sum of the ring's solid angles * launched), sigma = I here
    Xg, Yg = _pixel_grid(ins)
    rg = np.hypot(Xg, Yg)
    qg = 4 * math.pi / lam * np.sin(0.5 * np.arctan(rg / D))
    ring = np.floor(qg / 0.1 * 50).astype(int) == b
    dO = (0.5 / 64) ** 2 * D / (D * D + rg * rg) ** 1.5
    assert n[b] == ring.sum()
    assert abs(I[b] - 3.0 / (dO[ring].sum() * 7.0)) < 1e-12 * I[b] and abs(s[b] - I[b]) < 1e-12 * I[b]
    # a synthetic image of constant intensity c per steradian per neutron reduces to c in every populated ring
    c, launched = 2.5e-4, 1e6
    q, I, s, n = O.reduce_radial(ins, c * launched * dO, np.zeros_like(dO), launched, lam, 0.0, 0.1, 50)
    assert np.all(np.abs(I[n > 0] - c) < 1e-12 * c) and np.all(s == 0)
    # conservation: sum_b I_b * (sum dOmega)_b * launched = all weight inside the q window
    rng = np.random.Generator(np.random.PCG64(5))
    P = rng.random((64, 64)); P2 = P * P
    q, I, s, n = O.reduce_radial(ins, P, P2, 3.0, lam, 0.004, 0.07, 33)
    bins = np.floor((qg - 0.004) / (0.07 - 0.004) * 33).astype(int)
    inside = (qg >= 0.004) & (qg < 0.07)
    om = np.array([dO[inside & (bins == k)].sum() for k in range(33)])
    assert abs((I * om * 3.0).sum() - P[inside].sum()) < 1e-10 * P[inside].sum()
    assert n.sum() == inside.sum()


def test_sphere_minimum_lands_at_the_first_zero_of_phi():
    # analytic image of a sphere R = 100 A: the ring average has its first minimum where q R = 4.4934
    ins = W.instrument(det_nx=256, det_ny=256)
    lam, D, R = 6.0, ins["det_dist"], 100.0
    Xg, Yg = _pixel_grid(ins)
    rg = np.hypot(Xg, Yg)
    qg = 4 * math.pi / lam * np.sin(0.5 * np.arctan(rg / D))
    u = qg * R
    img = (3 * (np.sin(u) - u * np.cos(u)) / u ** 3) ** 2 * ((0.5 / 256) ** 2 * D / (D * D + rg * rg) ** 1.5)
    q, I, s, n = O.reduce_radial(ins, img, img * img, 1.0, lam, 0.01, 0.06, 200)
    i_min = int(np.argmin(I[:180]))
    assert abs(q[i_min] * R - 4.493409457909) < 0.03
    # and away from the minimum it reproduces Phi^2 at the bin centre
    ok = (n > 20) & (np.abs(q * R - 4.4934) > 0.6) & (q * R < 5.2)
    uu = q[ok] * R
    assert np.all(np.abs(I[ok] / (3 * (np.sin(uu) - uu * np.cos(uu)) / uu ** 3) ** 2 - 1) < 0.02)
