"""Pins of the oracle's polymer-micelle form factor (DESIGN.md R-M4; PAPER.md:201 names the model among the
expensive ones; Pedersen & Gerstenberg, Macromolecules 29 (1996) 1363).  None of them retypes the oracle's
formula: the Gaussian-chain pieces are checked against the chain averages that define them (numerical integrals of
exp(-x |s - s'|)), the composition against brute-force Monte Carlo over explicit configurations of point
scatterers and of random-walk chains, the limits against the already pinned sphere."""
import math

import numpy as np

import sas_workloads as W
from oracle import oracle as O


def micelle(**over):
    d = dict(model="polymer_micelle", precision="fp64", size=[40.0, 15.0, 4000.0, 30.0], sld=[2.0e-6, 1.0e-6, 0.0], scale=0.01)
    d.update(over)
    return W.model(**d)


def test_debye_function_is_the_double_chain_average():
    # D(x) = int_0^1 int_0^1 exp(-x |s - s'|) ds ds', psi(x) = int_0^1 exp(-x s) ds  (Gauss-Legendre, split at s = s')
    g, w = np.polynomial.legendre.leggauss(80)
    s = 0.5 * (g + 1.0)
    ws = 0.5 * w
    for x in (1e-6, 1e-3, 9.9e-3, 1.01e-2, 0.0999, 0.1001, 0.3, 1.0, 7.0, 40.0, 300.0):
        psi = float((ws * np.exp(-x * s)).sum())
        # inner integral over s' in [0, s] in closed form is what we avoid: do it numerically on a scaled rule
        inner = np.array([float((ws * si * np.exp(-x * (si - si * s))).sum()) for si in s])    # int_0^si exp(-x (si - t)) dt
        D = 2.0 * float((ws * inner).sum())
        assert abs(O.chain_psi(x) - psi) < 2e-13 * max(1.0, psi)
        assert abs(O.debye(x) - D) < 5e-13
    assert O.debye(0.0) == 1.0 and O.chain_psi(0.0) == 1.0
    # the two are tied by D = 2 (1 - psi) / x
    for x in (0.05, 2.0, 50.0):
        assert abs(O.debye(x) - 2.0 * (1.0 - O.chain_psi(x)) / x) < 1e-14


def test_no_chains_is_the_homogeneous_sphere_and_forward_scattering_is_the_total_excess_length():
    for q in (0.0, 0.003, 0.02, 0.11, 0.3):
        m = micelle(size=[40.0, 15.0, 4000.0, 0.0])
        f2, vol = O.micelle_f2(m, q)
        F, V = O.amplitude(W.model(model="sphere", size=[40.0, 0, 0, 0], sld=[2.0e-6, 0, 0]), 0.0, 0.0, q)
        assert abs(f2 - F * F) <= 1e-15 * F * F and vol == V
    m = micelle()
    f2, vol = O.micelle_f2(m, 0.0)
    Vcore = 4.0 * math.pi / 3.0 * 40.0 ** 3
    total = 2.0e-6 * Vcore + 30.0 * 1.0e-6 * 4000.0
    assert abs(f2 - total ** 2) < 1e-14 * total ** 2
    assert abs(vol - (Vcore + 30.0 * 4000.0)) < 1e-9
    # the intensity through the model interface: 1e8 scale F^2 / V
    I = O.intensity(m, [0.0, 0.0, 1e-9])
    assert abs(I - 1e8 * 0.01 * total ** 2 / vol) < 1e-12 * I


def test_composition_against_explicit_point_scatterers_on_the_shell():
    """R_g -> 0: every chain is a point of excess length b_c at radius R, independent and uniform on the sphere.
    The orientational average of |B_s Phi(qR) + b_c sum_j exp(i q.r_j)|^2 over explicit configurations must give
    the oracle's four terms (self, chain self, chain-chain N(N-1), cross 2N) with their factors and signs."""
    rng = np.random.Generator(np.random.PCG64(2501))
    R, N, bc_sld, Vc = 30.0, 4, -3.0e-6, 9000.0          # a negative chain contrast makes the cross term negative
    m = micelle(size=[R, 1e-9, Vc, float(N)], sld=[2.0e-6, bc_sld, 0.0])
    Bs, bc = 2.0e-6 * 4.0 * math.pi / 3.0 * R ** 3, bc_sld * Vc
    n_cfg = 400000
    v = rng.normal(size=(n_cfg, N, 3))
    v /= np.linalg.norm(v, axis=2, keepdims=True)
    for q in (0.02, 0.07, 0.15):
        phase = q * R * v[:, :, 2]                          # Q along z
        u = q * R
        phi = 3.0 * (math.sin(u) - u * math.cos(u)) / u ** 3
        amp = Bs * phi + bc * np.exp(1j * phase).sum(axis=1)
        mc = float((np.abs(amp) ** 2).mean())
        err = float((np.abs(amp) ** 2).std()) / math.sqrt(n_cfg)
        f2, _ = O.micelle_f2(m, q)
        assert abs(f2 - mc) < 5 * err, (q, f2, mc, err)


def test_chain_amplitude_against_explicit_random_walks():
    """One chain, no core contrast: |F|^2 = b_c^2 D(x); and the cross term of a core with ONE chain is
    2 B_s b_c Phi psi(x) sinc(q (R + R_g)): the chain starts on the sphere of radius R + R_g and is a Gaussian random
    walk from there.  Explicit walks of 200 steps reproduce both within Monte-Carlo error."""
    rng = np.random.Generator(np.random.PCG64(6054))
    R, Rg, Vc = 25.0, 12.0, 5000.0
    n_cfg, M = 40000, 200
    sigma = math.sqrt(2.0 * Rg * Rg / M)                    # per-axis step: <(r_M - r_0)^2> = 6 R_g^2 (R_g^2 = N b^2 / 6)
    steps = rng.normal(scale=sigma, size=(n_cfg, M, 3))
    walk = np.concatenate([np.zeros((n_cfg, 1, 3)), np.cumsum(steps, axis=1)], axis=1)
    start = rng.normal(size=(n_cfg, 3))
    start *= (R + Rg) / np.linalg.norm(start, axis=1, keepdims=True)
    pts = walk + start[:, None, :]
    for q in (0.03, 0.08):
        a_chain = np.exp(1j * q * pts[:, :, 2]).mean(axis=1)            # chain amplitude per unit excess length
        m1 = micelle(size=[R, Rg, Vc, 1.0], sld=[0.0, 1.0e-6, 0.0])
        f2, _ = O.micelle_f2(m1, q)
        bc = 1.0e-6 * Vc
        mc = float((np.abs(a_chain) ** 2).mean()) * bc * bc
        err = float((np.abs(a_chain) ** 2).std()) / math.sqrt(n_cfg) * bc * bc
        assert abs(f2 - mc) < 5 * err + 0.01 * mc, (q, f2, mc)            # 1 %: discretisation of the walk (M = 200)
        m2 = micelle(size=[R, Rg, Vc, 1.0], sld=[2.0e-6, 1.0e-6, 0.0])
        Bs = 2.0e-6 * 4.0 * math.pi / 3.0 * R ** 3
        u = q * R
        phi = 3.0 * (math.sin(u) - u * math.cos(u)) / u ** 3
        full = np.abs(Bs * phi + bc * a_chain) ** 2
        f2b, _ = O.micelle_f2(m2, q)
        errb = float(full.std()) / math.sqrt(n_cfg)
        assert abs(f2b - float(full.mean())) < 5 * errb + 0.01 * abs(f2b), (q, f2b, float(full.mean()))


def test_polydisperse_core_and_event_sampling_reduce_to_the_same_monodisperse_value():
    m = micelle()
    Q = [0.03, -0.02, 0.01]
    I0 = O.intensity(m, Q)
    q = math.sqrt(sum(v * v for v in Q))
    f2, vol = O.micelle_f2(m, q)
    assert abs(I0 - 1e8 * 0.01 * f2 / vol) < 1e-13 * I0
    assert O.intensity_event(m, Q, x=(1.0, 1.0)) == I0                  # Delta = 0: the same arithmetic
    # a Schulz average over the core radius against a dense integral of the distribution
    p, n = 0.1, 40
    mp_ = micelle(pd_kind=["schulz", "none"], pd_rel=[p, 0.0], pd_nodes=[n, 1])
    Ip = O.intensity(mp_, Q)
    z = 1.0 / (p * p) - 1.0
    s = np.linspace(1e-6, 3.0, 200001)
    logf = (z + 1.0) * math.log(z + 1.0) + z * np.log(s) - (z + 1.0) * s - math.lgamma(z + 1.0)
    f = np.exp(logf)
    vals = np.array([O.micelle_f2(m, q, float(x)) for x in s[::200]])
    f2s, vols = vals[:, 0], vals[:, 1]
    fs = f[::200]
    num = np.trapezoid(fs * f2s, s[::200])
    den = np.trapezoid(fs * vols, s[::200])
    assert abs(Ip - 1e8 * 0.01 * num / den) < 2e-4 * Ip
