"""Seeded synthetic workloads c0..c4 (BASELINE.json `configs`).

This module is the ONLY thing the oracle (oracle/) and the CUDA library
(paper_2501_06054_b200/) have in common.  It holds plain descriptor values
(numbers and names) and nothing of the method's arithmetic: no RNG stream of
the tracer, no geometry, no form factors, no quadrature nodes.  Each side
turns these dictionaries into its own structures with its own code.

The paper times 70 SasView-default models on the KWS-1 instrument file
(PAPER.md:86, :153); neither is available, so these five synthetic virtual
experiments of the same shape stand in for them.
"""
from __future__ import annotations

import copy

import numpy as np

# --- instrument of config 0; the other configs override fields --------------
BASE_INSTRUMENT = dict(
    src_xw=0.010, src_yh=0.010,            # 10 x 10 mm flat source
    lambda_min=5.4, lambda_max=6.6,        # Angstrom
    lambda_dist="uniform",                 # or "triangle": velocity-selector law (DESIGN.md R-L1)
    flux=1.0,
    slit1_z=0.0, slit1_xw=0.005, slit1_yh=0.005,
    slit2_z=5.0, slit2_xw=0.005, slit2_yh=0.005,
    focus_z=5.0, focus_xw=0.005, focus_yh=0.005,   # focus rectangle = slit 2
    sample_shape="box",
    sample_z=5.01, sample_xw=0.010, sample_yh=0.010, sample_zd=0.001, sample_radius=0.005,
    mu_abs_2200=0.0, mu_inc=0.0,
    q_min=0.001, q_max=0.3,
    det_dist=5.0, det_xw=0.5, det_yh=0.5, det_nx=128, det_ny=128,
)

BASE_MODEL = dict(
    model="sphere", precision="fp64",
    scale=0.01, background=0.0,
    sld=[1.0e-6, 0.0, 0.0],
    size=[50.0, 0.0, 0.0, 0.0],
    pd_kind=["none", "none"], pd_rel=[0.0, 0.0], pd_nodes=[1, 1],
    orient_kind="fixed", theta=0.0, phi=0.0, psi=0.0,
    sigma_theta=0.0, sigma_phi=0.0, n_theta=1, n_phi=1,
    sq_kind="none", sq_radius_eff=0.0, sq_volfrac=0.0,
    sq_contact_kT=0.0, sq_kappa_sigma=0.0,     # "hayter_msa": contact potential in kT, inverse screening length x diameter
)


def instrument(**over):
    d = copy.deepcopy(BASE_INSTRUMENT)
    d.update(over)
    return d


def model(**over):
    d = copy.deepcopy(BASE_MODEL)
    d.update(over)
    return d


def config(i: int, precision: str | None = None):
    """Return dict(name, instrument, model, n_neutrons, seed) for config i in 0..3 and 5..9,
    or dict(name, instruments[], models[], n_neutrons_each, seed) for config 4."""
    if i == 0:
        return dict(name="c0_sphere_fp64", instrument=instrument(),
                    model=model(precision=precision or "fp64"),
                    n_neutrons=10**6, seed=20250106)
    if i == 1:
        return dict(
            name="c1_polysphere_py", instrument=instrument(det_nx=256, det_ny=256),
            model=model(precision=precision or "fp32", size=[40.0, 0, 0, 0], scale=0.2,
                        pd_kind=["schulz", "none"], pd_rel=[0.15, 0.0], pd_nodes=[32, 1],
                        sq_kind="hard_sphere_py", sq_radius_eff=40.0, sq_volfrac=0.2),
            n_neutrons=10**8, seed=20250107)
    if i == 2:
        deg = np.pi / 180.0
        return dict(
            name="c2_oriented_cylinder",
            instrument=instrument(lambda_min=4.5, lambda_max=5.5, det_dist=2.0, det_nx=256, det_ny=256),
            model=model(model="cylinder", precision=precision or "fp32", sld=[2.0e-6, 0, 0],
                        size=[20.0, 400.0, 0, 0], orient_kind="gauss_quad",
                        theta=0.0, phi=0.0, psi=0.0,
                        sigma_theta=10.0 * deg, sigma_phi=10.0 * deg, n_theta=24, n_phi=24),
            n_neutrons=10**9, seed=20250108)
    if i == 3:
        return dict(
            name="c3_coreshell_triaxial",
            instrument=instrument(sample_shape="cyl_y", sample_radius=0.005, sample_yh=0.010,
                                  det_nx=512, det_ny=512),
            model=model(model="core_shell_triaxial", precision=precision or "fp32",
                        sld=[3.0e-6, 1.0e-6, 0.0], size=[30.0, 50.0, 80.0, 10.0],
                        pd_kind=["schulz", "schulz"], pd_rel=[0.1, 0.1], pd_nodes=[16, 16],
                        orient_kind="isotropic_mc"),
            n_neutrons=10**9, seed=20250109)
    if i == 4:
        return batch_config(1024, 10**7, 20250110, precision or "fp32")
    if i == 5:
        # NEXT-1 (not a BASELINE.json config): the paper's own averaging on the cylinder it compares with a
        # measurement (R = 119 A, L = 800 A, 5 % polydispersity, random orientation): one Gaussian
        # size pair and one uniform-angle orientation per scattering event (DESIGN.md R-N1..R-N3)
        return dict(
            name="n1_paper_cylinder", instrument=instrument(det_nx=256, det_ny=256),
            model=model(model="cylinder", precision="fp64", size=[119.0, 800.0, 0, 0],
                        pd_kind=["gauss_mc", "gauss_mc"], pd_rel=[0.05, 0.05],
                        orient_kind="uniform_angles_mc"),
            n_neutrons=10**9, seed=20250111)
    if i == 6:
        # NEXT-2 (not a BASELINE.json config): one of the models the paper found expensive, the
        # barbell, with the paper's per-event sizes and orientation: 64 slice evaluations with a Bessel J1 each per
        # detected neutron
        return dict(
            name="n2_paper_barbell", instrument=instrument(det_nx=256, det_ny=256),
            model=model(model="barbell", precision="fp64", size=[20.0, 400.0, 40.0, 0],
                        pd_kind=["gauss_mc", "gauss_mc"], pd_rel=[0.05, 0.05], orient_kind="uniform_angles_mc"),
            n_neutrons=10**9, seed=20250112)
    if i == 7:
        # NEXT-2 (not a BASELINE.json config): the polymer micelle, another model PAPER.md:201 singles out, with the
        # paper's per-event Gaussian core radius (DESIGN.md R-M4, R-N1)
        return dict(
            name="n3_paper_micelle", instrument=instrument(det_nx=256, det_ny=256),
            model=model(model="polymer_micelle", precision="fp64", size=[40.0, 15.0, 4000.0, 30.0],
                        sld=[2.0e-6, 1.0e-6, 0.0], pd_kind=["gauss_mc", "none"], pd_rel=[0.1, 0.0]),
            n_neutrons=10**9, seed=20250113)
    if i == 8:
        # NEXT-2 (not a BASELINE.json config): "Hayter MSA", the third expensive model of PAPER.md:201 built here:
        # charged spheres, the paper's per-event Gaussian radius, S(q) from the mean-spherical closure (DESIGN.md
        # R-S2): 33 fp64 sine/cosine pairs per detected neutron (the 64-node rule folded about x = 1/2)
        return dict(
            name="n4_paper_hayter_msa", instrument=instrument(det_nx=256, det_ny=256),
            model=model(model="sphere", precision="fp64", size=[40.0, 0, 0, 0], pd_kind=["gauss_mc", "none"],
                        pd_rel=[0.1, 0.0], scale=0.2, sq_kind="hayter_msa", sq_radius_eff=45.0, sq_volfrac=0.2,
                        sq_contact_kT=5.0, sq_kappa_sigma=2.0),
            n_neutrons=10**9, seed=20250114)
    if i == 9:
        # NEXT-2 (not a BASELINE.json config): "Hollow rectangular prism thin walls", the fourth expensive model of
        # PAPER.md:201 built here (DESIGN.md R-M5), with the paper's per-event size scale and orientation
        return dict(
            name="n5_paper_hollow_prism", instrument=instrument(det_nx=256, det_ny=256),
            model=model(model="hollow_prism_thin", precision="fp64", size=[35.0, 75.0, 120.0, 2.0],
                        pd_kind=["gauss_mc", "none"], pd_rel=[0.1, 0.0], orient_kind="uniform_angles_mc"),
            n_neutrons=10**9, seed=20250115)
    raise ValueError(i)


def batch_config(n_exp: int, n_each: int, seed: int, precision: str = "fp32"):
    """Config 4: n_exp virtual experiments, even index = sphere, odd = cylinder
    (L = 20 R, isotropic random orientation per neutron).  Parameters are drawn
    from numpy's own seeded generator (not the tracer's stream): R~U[10,100] A,
    drho~U[0.5,5]e-6 1/A^2, mean wavelength~U[4,10] A with +-10 % spread,
    detector distance~U[1,10] m."""
    rng = np.random.Generator(np.random.PCG64(seed))
    pars = rng.random((n_exp, 4))
    instruments, models = [], []
    for e in range(n_exp):
        R = 10.0 + 90.0 * pars[e, 0]
        drho = (0.5 + 4.5 * pars[e, 1]) * 1.0e-6
        lam = 4.0 + 6.0 * pars[e, 2]
        dist = 1.0 + 9.0 * pars[e, 3]
        instruments.append(instrument(lambda_min=0.9 * lam, lambda_max=1.1 * lam, det_dist=dist))
        if e % 2 == 0:
            models.append(model(model="sphere", precision=precision, sld=[drho, 0, 0], size=[R, 0, 0, 0]))
        else:
            models.append(model(model="cylinder", precision=precision, sld=[drho, 0, 0],
                                size=[R, 20.0 * R, 0, 0], orient_kind="isotropic_mc"))
    return dict(name="c4_batch", instruments=instruments, models=models,
                n_neutrons_each=n_each, seed=seed)


def pencil_instrument(**over):
    """Monochromatic pencil beam (source, slits, focus 0.1 mm; d-lambda = 0) used by the
    chi^2 test against the numerically integrated I(Q) (DESIGN.md R-C17)."""
    d = instrument(src_xw=1e-4, src_yh=1e-4, slit1_xw=1e-4, slit1_yh=1e-4,
                   slit2_xw=1e-4, slit2_yh=1e-4, focus_xw=1e-4, focus_yh=1e-4,
                   lambda_min=6.0, lambda_max=6.0)
    d.update(over)
    return d
