"""Pins of the oracle's Hayter-Penfold MSA structure factor (DESIGN.md R-S2; PAPER.md:201 names "Hayter MSA" among
the expensive models; the closure is Hayter & Penfold's, Mol. Phys. 42 (1981) 109: mean-spherical approximation for
hard spheres with a screened-Coulomb repulsion).  The oracle solves the closure through the Baxter / Hoye-Blum
factorisation; nothing here retypes those equations: the pins check that the result HAS the two properties that
define the mean-spherical solution -- g(x) = 0 inside the core and c(x) = -beta u(x) outside, both obtained by
numerical inverse Fourier transforms of S(K) -- and its limits (no charge or infinite screening: the pinned
Percus-Yevick S(q); large K: 1; K -> 0: the compressibility 1/a^2)."""
import math

import numpy as np

import sas_workloads as W
from oracle import oracle as O


def msa_model(eta, gam, k, r_eff=40.0):
    """(the closure is solved once, here: O.make_model)"""
    return O.make_model(W.model(sq_kind="hayter_msa", sq_radius_eff=r_eff, sq_volfrac=eta, sq_contact_kT=gam, sq_kappa_sigma=k))


def test_no_charge_and_strong_screening_are_percus_yevick():
    for eta in (0.05, 0.2, 0.4):
        m = msa_model(eta, 0.0, 1.7)
        for q in np.linspace(0.001, 0.3, 120):
            assert abs(O.msa_sq(m, q) / O.lib().orc_py_sq(q, 40.0, eta) - 1.0) < 1e-12
    # a repulsion screened within a thin shell changes less and less: S tends to Percus-Yevick as k grows
    qs = np.linspace(0.005, 0.3, 60)
    dist = []
    for k in (5.0, 20.0, 80.0, 320.0):
        m = msa_model(0.2, 2.0, k)
        dist.append(max(abs(O.msa_sq(m, q) - O.lib().orc_py_sq(q, 40.0, 0.2)) for q in qs))
    assert dist[0] > dist[1] > dist[2] > dist[3] and dist[3] < 0.01 and dist[0] > 0.1


def _transforms(eta, gam, k):
    """h(x) and c(x) at a few x by inverse sine transforms of S(K) on a fine K grid (S from the oracle's Baxter
    function integrated with a dense composite rule, so that K reaches 900)."""
    a, b, E, Cp, Dp = O.msa_solve(eta, gam, k)
    gx, gw = np.polynomial.legendre.leggauss(100)
    P = 12
    xs = np.concatenate([(p + 0.5 * (gx + 1)) / P for p in range(P)])
    ws = np.concatenate([0.5 * gw / P for p in range(P)])
    Q = 0.5 * a * (xs * xs - 1) + b * (xs - 1) + E * np.exp(-k * xs) - Cp
    dK = 0.04
    K = np.arange(dK / 2, 900, dK)
    S = np.empty_like(K)
    for i0 in range(0, K.size, 1500):
        Kb = K[i0:i0 + 1500, None]
        den = k * k + Kb[:, 0] ** 2
        re = 1 - 12 * eta * ((ws * Q * np.cos(Kb * xs)).sum(1) + Dp * (k * np.cos(Kb[:, 0]) - Kb[:, 0] * np.sin(Kb[:, 0])) / den)
        im = -12 * eta * ((ws * Q * np.sin(Kb * xs)).sum(1) + Dp * (k * np.sin(Kb[:, 0]) + Kb[:, 0] * np.cos(Kb[:, 0])) / den)
        S[i0:i0 + 1500] = 1 / (re * re + im * im)
    rho = 6 * eta / math.pi
    win = np.exp(-(K / 350.0) ** 2)
    hh, ch = (S - 1) / rho, (1 - 1 / S) / rho
    inv = lambda f, x: dK / (2 * math.pi ** 2 * x) * float((K * f * win * np.sin(K * x)).sum())
    return (lambda x: inv(hh, x)), (lambda x: inv(ch, x)), S, K, a


def test_the_solution_satisfies_the_mean_spherical_closure():
    for eta, gam, k in ((0.2, 5.0, 2.0), (0.3, 2.0, 1.0), (0.15, 1.0, 0.7), (0.35, 6.0, 6.0)):
        h, c, S, K, a = _transforms(eta, gam, k)
        for x in (0.25, 0.5, 0.75, 0.93):
            assert abs(h(x) + 1.0) < 2e-3, (eta, gam, k, x, h(x))          # g = 0 inside the core
        for x in (1.08, 1.3, 1.8, 2.6, 4.0):
            u = gam * math.exp(-k * (x - 1.0)) / x
            assert abs(c(x) + u) < 2e-3 * max(1.0, u), (eta, gam, k, x, c(x), -u)   # c = -beta u outside
        assert np.all(S > 0) and abs(S[-1] - 1.0) < 1e-4
        assert abs(S[0] - 1.0 / a ** 2) < 1e-3 * S[0]                        # S(0) = 1 / Qhat(0)^2, Qhat(0) = a


def test_the_oracle_function_is_that_structure_factor_and_repulsion_suppresses_small_angles():
    eta, gam, k = 0.2, 5.0, 2.0
    m = msa_model(eta, gam, k)
    _, _, S, K, _ = _transforms(eta, gam, k)
    for q in (0.004, 0.03, 0.0785, 0.2, 0.6):                                # K = 80 q up to 48 (< 64: the rule's range)
        j = int(round((80.0 * q - 0.02) / 0.04))
        assert abs(O.msa_sq(m, K[j] / 80.0) - S[j]) < 1e-10 * S[j]
    # charge pushes the particles apart: lower compressibility, higher first peak than the uncharged fluid
    assert O.msa_sq(m, 0.001) < 0.2 * O.lib().orc_py_sq(0.001, 40.0, eta)
    peak = max(O.msa_sq(m, q) for q in np.linspace(0.05, 0.11, 200))
    peak_py = max(O.lib().orc_py_sq(q, 40.0, eta) for q in np.linspace(0.05, 0.11, 200))
    assert peak > peak_py
    # through the model interface: I = 1e8 scale F^2 / V S(q)
    ms = O.make_model(W.model(size=[30.0, 0, 0, 0], sq_kind="hayter_msa", sq_radius_eff=40.0, sq_volfrac=eta, sq_contact_kT=gam,
                              sq_kappa_sigma=k))
    m0 = O.make_model(W.model(size=[30.0, 0, 0, 0]))
    Q = [0.02, 0.01, -0.015]
    q = math.sqrt(sum(v * v for v in Q))
    assert abs(O.intensity(ms, Q) - O.intensity(m0, Q) * O.msa_sq(ms, q)) < 1e-15 * O.intensity(ms, Q) + 1e-300
