"""ctypes front-end of the CPU oracle -- TEST INFRASTRUCTURE ONLY.

Builds oracle/sas_oracle.c with gcc (-O2 -ffp-contract=off), converts the
neutral workload dictionaries of sas_workloads.py into the oracle's own
structs, and expands the quadrature tables with numpy:

* Schulz polydispersity (DESIGN.md R-A9): generalised Gauss-Laguerre rule with
  alpha = z = 1/p^2 - 1 by Golub-Welsch -- eigen-decomposition (numpy.linalg.eigh,
  a library primitive) of the Jacobi matrix with diagonal 2i+1+alpha and
  off-diagonal sqrt(i (i+alpha)); node value x_i/(z+1) (mean 1), weight = squared
  first eigenvector component (sums to 1).
* Gaussian orientation spread (DESIGN.md R-A11): Gauss-Legendre nodes on
  [-3 sigma, 3 sigma] (numpy.polynomial.legendre.leggauss), weights
  w_i exp(-Delta_i^2 / 2 sigma^2) normalised to sum 1.

Nothing here imports, links or reads anything of paper_2501_06054_b200/.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sas_oracle.c")
_HDR = os.path.join(_HERE, "sas_oracle.h")
_LIB = os.path.join(_HERE, "liboracle.so")
MAX_NODES = 64

_SAMPLE = {"box": 0, "cyl_y": 1}
_LAMBDA = {"uniform": 0, "triangle": 1}
_MODEL = {"sphere": 0, "core_shell_sphere": 1, "cylinder": 2, "triaxial": 3,
          "core_shell_triaxial": 4, "flat": 5, "parallelepiped": 6, "core_shell_cylinder": 7, "ellipsoid": 8,
          "barbell": 9, "capped_cylinder": 10, "elliptical_cylinder": 11, "hollow_cylinder": 12,
          "core_shell_ellipsoid": 13, "polymer_micelle": 14, "hollow_prism_thin": 15}
_ORIENT = {"fixed": 0, "gauss_quad": 1, "isotropic_mc": 2, "uniform_angles_mc": 3}
_SQ = {"none": 0, "hard_sphere_py": 1, "hayter_msa": 2}


class Instrument(C.Structure):
    _fields_ = [(n, C.c_double) for n in
                ("src_xw", "src_yh", "lambda_min", "lambda_max", "flux",
                 "slit1_z", "slit1_xw", "slit1_yh", "slit2_z", "slit2_xw", "slit2_yh",
                 "focus_z", "focus_xw", "focus_yh")] + \
               [("sample_shape", C.c_int32), ("lambda_dist", C.c_int32)] + \
               [(n, C.c_double) for n in
                ("sample_z", "sample_xw", "sample_yh", "sample_zd", "sample_radius",
                 "mu_abs_2200", "mu_inc", "q_min", "q_max", "det_dist", "det_xw", "det_yh")] + \
               [("det_nx", C.c_int32), ("det_ny", C.c_int32)]


class Model(C.Structure):
    _fields_ = [("model", C.c_int32), ("orient_kind", C.c_int32), ("sq_kind", C.c_int32),
                ("pad0", C.c_int32), ("scale", C.c_double), ("background", C.c_double),
                ("sld", C.c_double * 3), ("size", C.c_double * 4),
                ("n_pd", C.c_int32 * 2),
                ("pd_x", (C.c_double * MAX_NODES) * 2), ("pd_w", (C.c_double * MAX_NODES) * 2),
                ("theta", C.c_double), ("phi", C.c_double), ("psi", C.c_double),
                ("n_or", C.c_int32 * 2),
                ("or_d", (C.c_double * MAX_NODES) * 2), ("or_w", (C.c_double * MAX_NODES) * 2),
                ("sq_radius_eff", C.c_double), ("sq_volfrac", C.c_double),
                ("pd_mc", C.c_int32 * 2), ("pd_rel", C.c_double * 2),
                ("sq_contact_kT", C.c_double), ("sq_kappa_sigma", C.c_double), ("msa", C.c_double * 5)]


class Record(C.Structure):
    _fields_ = [("status", C.c_int32), ("pixel", C.c_int32), ("weight", C.c_double),
                ("weight_env", C.c_double), ("q", C.c_double), ("Q", C.c_double * 3),
                ("lam", C.c_double), ("ell", C.c_double), ("p0", C.c_double),
                ("intensity", C.c_double), ("u", C.c_double * 12),
                ("pd_x", C.c_double * 2), ("pd_tries", C.c_int32 * 2)]


def build(force: bool = False) -> str:
    """Compile the oracle shared library if it is missing or stale."""
    stale = force or not os.path.exists(_LIB) or \
        os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if stale:
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.orc_philox4x32_10.restype = None
        L.orc_uniform.argtypes = [C.c_uint32]
        L.orc_uniform.restype = C.c_double
        for f in (L.orc_sphere_phi, L.orc_sinc, L.orc_lambda1):
            f.argtypes = [C.c_double]
            f.restype = C.c_double
        for f in (L.orc_debye, L.orc_chain_psi):
            f.argtypes = [C.c_double]
            f.restype = C.c_double
        L.orc_micelle_f2.argtypes = [C.POINTER(Model), C.c_double, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_micelle_f2.restype = C.c_double
        L.orc_msa_sq.argtypes = [C.c_double, C.POINTER(Model)]
        L.orc_msa_sq.restype = C.c_double
        L.orc_py_sq.argtypes = [C.c_double] * 3
        L.orc_py_sq.restype = C.c_double
        L.orc_intensity.argtypes = [C.POINTER(Model), C.POINTER(C.c_double), C.POINTER(C.c_double),
                                    C.POINTER(C.c_double)]
        L.orc_intensity.restype = C.c_double
        L.orc_intensity_event.argtypes = [C.POINTER(Model), C.POINTER(C.c_double), C.POINTER(C.c_double),
                                          C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_intensity_event.restype = C.c_double
        L.orc_draw_rel_size.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_int, C.c_double,
                                        C.POINTER(C.c_int32)]
        L.orc_draw_rel_size.restype = C.c_double
        L.orc_amplitude.argtypes = [C.POINTER(Model)] + [C.c_double] * 5 + [C.POINTER(C.c_double)] * 2
        L.orc_amplitude.restype = C.c_double
        L.orc_trace_one.argtypes = [C.POINTER(Instrument), C.POINTER(Model), C.c_uint64, C.c_uint64,
                                    C.c_uint32, C.POINTER(Record)]
        L.orc_trace_one.restype = None
        L.orc_trace_range.argtypes = [C.POINTER(Instrument), C.POINTER(Model), C.c_uint64, C.c_uint64,
                                      C.c_uint64, C.c_uint32] + [C.c_void_p] * 8
        L.orc_trace_range.restype = None
        L.orc_reduce_radial.argtypes = [C.POINTER(Instrument), C.c_void_p, C.c_void_p, C.c_double, C.c_double,
                                        C.c_double, C.c_double, C.c_int32] + [C.c_void_p] * 4
        L.orc_reduce_radial.restype = None
    return _lib


# ---------------------------------------------------------------- tables
def schulz_nodes(p: float, n: int):
    """n-node rule for a Schulz (gamma) distribution of unit mean and relative
    width p: returns (values s_i, weights w_i), sum w = 1, sum w s = 1."""
    if n <= 1 or p <= 0.0:
        return np.ones(1), np.ones(1)
    z = 1.0 / (p * p) - 1.0
    i = np.arange(n, dtype=np.float64)
    J = np.diag(2.0 * i + 1.0 + z)
    off = np.sqrt(i[1:] * (i[1:] + z))
    J += np.diag(off, 1) + np.diag(off, -1)
    x, v = np.linalg.eigh(J)
    w = v[0, :] ** 2
    return x / (z + 1.0), w / w.sum()


def gauss_tilts(sigma: float, n: int):
    """Tilt angles Delta_i in [-3 sigma, 3 sigma] and normalised Gaussian weights."""
    if n <= 1 or sigma <= 0.0:
        return np.zeros(1), np.ones(1)
    x, w = np.polynomial.legendre.leggauss(n)
    d = 3.0 * sigma * x
    g = w * np.exp(-(d * d) / (2.0 * sigma * sigma))
    return d, g / g.sum()


def make_instrument(d: dict) -> Instrument:
    ins = Instrument()
    for name, _ in Instrument._fields_:
        if name == "lambda_dist":
            ins.lambda_dist = _LAMBDA[d.get(name, "uniform")]
            continue
        if name == "sample_shape":
            ins.sample_shape = _SAMPLE[d[name]]
        elif name in ("det_nx", "det_ny"):
            setattr(ins, name, int(d[name]))
        else:
            setattr(ins, name, float(d[name]))
    return ins


def msa_residual(u, eta, gam, k, X, W):
    """The five equations of DESIGN.md R-S2 for u = (a, b, E, C', H'); X, W: Gauss-Legendre rule on [0, 1]."""
    a, b, E, Cp, Hp = u
    e = np.exp(-k)
    Dp = E * e - Cp                                        # Q is continuous at the contact distance
    qin = lambda x: 0.5 * a * (x * x - 1.0) + b * (x - 1.0) + E * np.exp(-k * x) - Cp
    Q = qin(X)
    I0, I1, Qt = (W * Q).sum(), (W * X * Q).sum(), (W * Q * np.exp(-k * X)).sum()
    r1 = a - (1.0 - 12.0 * eta * (I0 + Dp / k))
    r2 = b - 12.0 * eta * (I1 + Dp * (1.0 / k + 1.0 / k ** 2))
    r3 = -k * E + 12.0 * eta * Dp * ((1.0 + k) / k ** 2 + Hp)
    r4 = k * Dp * (1.0 - 12.0 * eta * (Qt + Dp * e / (2.0 * k))) + gam
    phi1 = (1.0 - e * (1.0 + k)) / k ** 2
    # T = D' phi1 / 2k + int_0^1 -(1 - y) e^{ky} [int_y^1 Q e^{-ks} ds + D' e^{-k}/2k] dy: the inner integral by the same
    # rule mapped onto [y, 1] for every outer node y (rows: outer nodes, columns: inner nodes)
    s2 = X[:, None] + (1.0 - X[:, None]) * X[None, :]
    G = ((1.0 - X[:, None]) * W[None, :] * qin(s2) * np.exp(-k * s2)).sum(axis=1) + Dp * e / (2.0 * k)
    T = Dp * phi1 / (2.0 * k) + (W * (-(1.0 - X)) * np.exp(k * X) * G).sum()
    r5 = Hp * (1.0 - 12.0 * eta * Qt) - Dp / 2.0 - 12.0 * eta * T
    return np.array([r1, r2, r3, r4, r5])


def msa_solve(eta: float, gam: float, k: float, steps: int = 20):
    """Mean-spherical closure for hard spheres (packing eta, diameter 1) with the Yukawa repulsion
    beta u(x) = gam exp(-k (x - 1)) / x, x > 1 (DESIGN.md R-S2): g(x) = 0 inside the core, c(x) = -beta u(x)
    outside, through the Baxter / Hoye-Blum factorisation.  Returns (a, b, E, C', D'): Q(x) = a (x^2 - 1)/2 +
    b (x - 1) + E exp(-k x) - C' for x < 1 and D' exp(-k (x - 1)) beyond.  Newton's method on the five equations,
    started from the Percus-Yevick solution (gam = 0) and continued in `steps` equal steps of gam, which keeps
    the branch that is connected to the uncharged fluid."""
    g, w = np.polynomial.legendre.leggauss(64)
    X, W = 0.5 * (g + 1.0), 0.5 * w
    u = np.array([(1.0 + 2.0 * eta) / (1.0 - eta) ** 2, -1.5 * eta / (1.0 - eta) ** 2, 0.0, 0.0, 0.0])
    for gs in np.linspace(0.0, gam, steps + 1):
        for _ in range(60):
            r = msa_residual(u, eta, gs, k, X, W)
            J = np.zeros((5, 5))
            for j in range(5):
                du = np.zeros(5)
                du[j] = 1e-6 * max(1.0, abs(u[j]))
                J[:, j] = (msa_residual(u + du, eta, gs, k, X, W) - msa_residual(u - du, eta, gs, k, X, W)) / (2.0 * du[j])
            st = np.linalg.solve(J, -r)
            u = u + st
            if np.abs(st).max() < 1e-15 * max(1.0, np.abs(u).max()):
                break
    if np.abs(msa_residual(u, eta, gam, k, X, W)).max() > 1e-11:
        raise ValueError("the mean-spherical closure did not converge")
    a, b, E, Cp, _ = u
    return np.array([a, b, E, Cp, E * np.exp(-k) - Cp])


def msa_sq(model_d: dict, q: float) -> float:
    m = model_d if isinstance(model_d, Model) else make_model(model_d)
    return lib().orc_msa_sq(float(q), C.byref(m))


def make_model(d: dict) -> Model:
    m = Model()
    m.model = _MODEL[d["model"]]
    m.orient_kind = _ORIENT[d["orient_kind"]]
    m.sq_kind = _SQ[d["sq_kind"]]
    m.scale = d["scale"]
    m.background = d["background"]
    for i in range(3):
        m.sld[i] = d["sld"][i]
    for i in range(4):
        m.size[i] = d["size"][i]
    for k in range(2):
        if d["pd_kind"][k] == "schulz":
            s, w = schulz_nodes(d["pd_rel"][k], d["pd_nodes"][k])
        else:
            s, w = np.ones(1), np.ones(1)
        # the paper's own size averaging (DESIGN.md R-N1): one Gaussian draw per event
        m.pd_mc[k] = 1 if d["pd_kind"][k] == "gauss_mc" else 0
        m.pd_rel[k] = float(d["pd_rel"][k])
        m.n_pd[k] = len(s)
        for i in range(len(s)):
            m.pd_x[k][i] = s[i]
            m.pd_w[k][i] = w[i]
    m.theta, m.phi, m.psi = d["theta"], d["phi"], d["psi"]
    sig = (d["sigma_theta"], d["sigma_phi"])
    nn = (d["n_theta"], d["n_phi"])
    for k in range(2):
        if d["orient_kind"] == "gauss_quad":
            dd, w = gauss_tilts(sig[k], nn[k])
        else:
            dd, w = np.zeros(1), np.ones(1)
        m.n_or[k] = len(dd)
        for i in range(len(dd)):
            m.or_d[k][i] = dd[i]
            m.or_w[k][i] = w[i]
    m.sq_radius_eff = d["sq_radius_eff"]
    m.sq_volfrac = d["sq_volfrac"]
    m.sq_contact_kT = d.get("sq_contact_kT", 0.0)
    m.sq_kappa_sigma = d.get("sq_kappa_sigma", 0.0)
    if d["sq_kind"] == "hayter_msa":
        sol = msa_solve(d["sq_volfrac"], m.sq_contact_kT, m.sq_kappa_sigma)
        for i in range(5):
            m.msa[i] = sol[i]
    if "gauss_mc" in d["pd_kind"] and (d["orient_kind"] == "gauss_quad" or "schulz" in d["pd_kind"]):
        raise ValueError("per-event sizes (gauss_mc) do not combine with fixed-node averages (DESIGN.md R-N1)")
    if d["orient_kind"] == "gauss_quad" and d["model"] != "cylinder":
        raise ValueError("gauss_quad orientation is built for the cylinder only (DESIGN.md R-A11)")
    return m


# ----------------------------------------------------------------- calls
def philox(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def intensity(model_d: dict, Q, u_or=(0.0, 0.0, 0.0), want_env=False):
    m = model_d if isinstance(model_d, Model) else make_model(model_d)
    q = (C.c_double * 3)(*[float(v) for v in Q])
    u = (C.c_double * 3)(*u_or)
    env = C.c_double()
    val = lib().orc_intensity(C.byref(m), q, u, C.byref(env))
    return (val, env.value) if want_env else val


def intensity_event(model_d: dict, Q, x=(1.0, 1.0), u_or=(0.0, 0.0, 0.0)):
    """Eq. 4 for one scattering event with relative sizes x (DESIGN.md R-N2)."""
    m = model_d if isinstance(model_d, Model) else make_model(model_d)
    q = (C.c_double * 3)(*[float(v) for v in Q])
    u = (C.c_double * 3)(*u_or)
    xx = (C.c_double * 2)(*x)
    return lib().orc_intensity_event(C.byref(m), q, u, xx, None)


def draw_rel_size(seed: int, nid: int, k: int, rel: float, exp_index: int = 0):
    """(relative size, Philox blocks used) of axis k of event (seed, nid, exp_index) (DESIGN.md R-N1)."""
    tries = C.c_int32()
    x = lib().orc_draw_rel_size(seed, nid, exp_index, k, float(rel), C.byref(tries))
    return x, tries.value


def amplitude(model_d: dict, qa, qb, qc, x0=1.0, x1=1.0):
    m = model_d if isinstance(model_d, Model) else make_model(model_d)
    vol, env = C.c_double(), C.c_double()
    F = lib().orc_amplitude(C.byref(m), qa, qb, qc, x0, x1, C.byref(vol), C.byref(env))
    return F, vol.value


def micelle_f2(model_d: dict, q: float, x0: float = 1.0):
    """(|F|^2, normalising volume) of the polymer micelle (DESIGN.md R-M4)."""
    m = model_d if isinstance(model_d, Model) else make_model(model_d)
    vol, env2 = C.c_double(), C.c_double()
    f2 = lib().orc_micelle_f2(C.byref(m), float(q), float(x0), C.byref(vol), C.byref(env2))
    return f2, vol.value


def debye(x: float) -> float:
    return lib().orc_debye(float(x))


def chain_psi(x: float) -> float:
    return lib().orc_chain_psi(float(x))


def trace_one(ins_d, model_d, seed: int, nid: int, exp_index: int = 0) -> Record:
    ins = ins_d if isinstance(ins_d, Instrument) else make_instrument(ins_d)
    m = model_d if isinstance(model_d, Model) else make_model(model_d)
    rec = Record()
    lib().orc_trace_one(C.byref(ins), C.byref(m), seed, nid, exp_index, C.byref(rec))
    return rec


def trace_range(ins_d, model_d, seed: int, first: int, n: int, exp_index: int = 0,
                dump: bool = True, hist: bool = True):
    """Trace ids [first, first+n).  Returns a dict with numpy arrays:
    pixel, weight, weight_env, q (if dump); sum_p, sum_p2, counts (if hist); counters."""
    ins = ins_d if isinstance(ins_d, Instrument) else make_instrument(ins_d)
    m = model_d if isinstance(model_d, Model) else make_model(model_d)
    out = {}
    ptr = lambda a: a.ctypes.data_as(C.c_void_p) if a is not None else None
    pixel = weight = wenv = q = sp = sp2 = cnt = None
    if dump:
        pixel = np.empty(n, np.int32)
        weight = np.empty(n, np.float64)
        wenv = np.empty(n, np.float64)
        q = np.empty(n, np.float64)
    if hist:
        npix = ins.det_nx * ins.det_ny
        sp = np.zeros(npix, np.float64)
        sp2 = np.zeros(npix, np.float64)
        cnt = np.zeros(npix, np.uint64)
    counters = np.zeros(8, np.uint64)
    lib().orc_trace_range(C.byref(ins), C.byref(m), seed, first, n, exp_index,
                          ptr(pixel), ptr(weight), ptr(wenv), ptr(q), ptr(sp), ptr(sp2), ptr(cnt),
                          ptr(counters))
    out.update(pixel=pixel, weight=weight, weight_env=wenv, q=q, sum_p=sp, sum_p2=sp2, counts=cnt,
               counters=counters)
    return out


def reduce_radial(ins_d, sum_p, sum_p2, launched, lambda_ref, q_lo, q_hi, n_bins):
    """Ring average of one detector image (DESIGN.md R-R1): returns (q, I, sigma, npix) arrays of n_bins."""
    ins = ins_d if isinstance(ins_d, Instrument) else make_instrument(ins_d)
    sp = np.ascontiguousarray(sum_p, np.float64).reshape(-1)
    sp2 = np.ascontiguousarray(sum_p2, np.float64).reshape(-1)
    assert sp.size == ins.det_nx * ins.det_ny == sp2.size and 1 <= n_bins <= 4096
    q, i, s = (np.zeros(n_bins) for _ in range(3))
    n = np.zeros(n_bins, np.uint64)
    ptr = lambda a: a.ctypes.data_as(C.c_void_p)
    lib().orc_reduce_radial(C.byref(ins), ptr(sp), ptr(sp2), float(launched), float(lambda_ref), float(q_lo),
                            float(q_hi), int(n_bins), ptr(q), ptr(i), ptr(s), ptr(n))
    return q, i, s, n

