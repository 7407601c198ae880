// fp64 geometry of one neutron between the source and the detector (DESIGN.md R-C2..R-C11).
// Written operation by operation as the design note states them; the translation unit is compiled
// with -fmad=false, so nothing here is contracted and the detector pixel is bit-identical to a
// plain IEEE evaluation of the same text.
//
// Control flow: a warp executes this for 32 slit-1 survivors at once, of which ~80 % will miss the
// detector.  The code is therefore straight-line: every lane computes every quantity (a dead lane
// carries harmless garbage) and the outcome is decided at the end from failure flags taken in the
// order the design note tests them.  Selects replace the d == 0 / swap branches of the slab test;
// for finite non-NaN inputs they yield the same values as the oracle's branches.
#pragma once
#include "sas_types.h"

namespace sas {

// one axis of the slab test: interval of t with |o + t d| <= h, intersected into [tin, tout]
__device__ __forceinline__ void slab_axis(double o, double d, double h, double& tin, double& tout, bool& miss) {
  const bool par = (d == 0.0);
  const double inv = 1.0 / d;
  const double ta = (-h - o) * inv, tb = (h - o) * inv;
  double t1 = fmin(ta, tb), t2 = fmax(ta, tb);
  t1 = par ? -INFINITY : t1;
  t2 = par ? INFINITY : t2;
  miss = miss || (par && fabs(o) > h);
  tin = fmax(tin, t1);
  tout = fmin(tout, t2);
}

// Ray (o + t d) against the sample volume centred on the origin of the sample frame (R-C5).
__device__ __forceinline__ bool intersect_sample(const ExpParams& P, double ox, double oy, double oz, double dx,
                                                 double dy, double dz, double& t_in, double& t_out,
                                                 bool lateral_free = false) {
  double tin = -INFINITY, tout = INFINITY;
  bool miss = false;
  if (P.sample_shape == 1) {  // warp-uniform
    const double a = dx * dx + dz * dz;
    const double b = ox * dx + oz * dz;
    const double c = (ox * ox + oz * oz) - P.radius2;
    const bool par = (a == 0.0);
    const double disc = b * b - a * c;
    const double sq = sqrt(disc);
    const double inv_a = 1.0 / a;
    const double t1 = (-b - sq) * inv_a, t2 = (-b + sq) * inv_a;
    miss = par ? (c > 0.0) : !(disc > 0.0);
    tin = par ? tin : t1;
    tout = par ? tout : t2;
  } else if (!lateral_free) {
    slab_axis(ox, dx, P.hx, tin, tout, miss);
  }
  // lateral_free: the host proved that the beam envelope lies strictly inside the sample's lateral faces over
  // its whole depth, so their slab intervals strictly contain the depth interval and max/min return the
  // depth roots themselves: skipping them is bit-identical (primary ray only, not the scattered one)
  if (!lateral_free) slab_axis(oy, dy, P.hy, tin, tout, miss);
  if (P.sample_shape != 1) slab_axis(oz, dz, P.hz, tin, tout, miss);
  t_in = tin;
  t_out = tout;
  return !miss;
}

struct Hit {
  int32_t pixel;
  double G;      // p0 * T * 100 ell * (q/k^2) * 2 pi (qmax - qmin): the weight is G * I(Q)
  double Qx, Qy, Qz;
  double q;      // drawn |Q| (0 if the neutron died before the draw)
};

// R-L1: wavelength from draw 4: uniform in the band, or the inverse distribution function of the symmetric
// triangle (velocity selector), operation by operation as the design note writes it (sqrt is correctly rounded)
__device__ __forceinline__ double lambda_from_u(const ExpParams& P, double u4) {
  double t = u4;
  if (P.lambda_dist == 1) t = (u4 < 0.5) ? sqrt(0.5 * u4) : 1.0 - sqrt(0.5 * (1.0 - u4));
  return P.lambda_min + t * P.dlam;
}

// Conservative classifier (stage B0): true when the neutron is CERTAIN to end as
// ST_MISS_DET.  The host proved for this instrument that every slit-1 survivor passes slit 2 and
// crosses the sample, and folded the worst-case beam divergence, beam radius at the sample, sample
// depth and detector half-diagonal (each with a 1e-6 margin, ten orders above fp64 rounding) into
// s_cut = sin(theta_cut): a neutron with sin(theta) = q lambda / 4 pi above it lands outside the
// detector's circumscribed circle whatever its azimuth.  q is formed exactly as R-C7 forms it.
__device__ __forceinline__ bool surely_misses_detector(const ExpParams& P, const uint32_t w1[4], double& q) {
  const double u4 = uniform_from_word(w1[0]), u6 = uniform_from_word(w1[2]);
  const double lambda = lambda_from_u(P, u4);
  q = P.q_min + u6 * P.dq;
  const double s_a = (q * lambda) * 0.07957747154594767;  // 1 / (4 pi)
  return (s_a > P.s_cut) && (s_a < 0.999999);
}

// The same decision from fp32 arithmetic (the warp-specialised kernel's stage B0): q lambda is formed from the
// raw words with host-folded constants, |relative error| < 6e-7 (two conversions, two FMAs, one product, four
// rounded constants), and compared with thresholds the host moved 2e-6 INTO the certain region, so
// true here implies true for the fp64 test above; a neutron this test leaves undecided simply runs the full
// geometry (which finds the same ST_MISS_DET).  For a wavelength law that is not linear in the draw (R-L1) the
// host sets cls_la = 0, cls_lb = lambda_min: a lower bound of lambda is all the first comparison needs, and the
// second one (|Q| reachable) is then proved for the whole instrument or the classifier is switched off.
__device__ __forceinline__ bool surely_misses_detector_f32(const ExpParams& P, uint32_t w_lambda, uint32_t w_q) {
  const float lam = fmaf(__uint2float_rn(w_lambda), P.cls_la, P.cls_lb);
  const float q = fmaf(__uint2float_rn(w_q), P.cls_qa, P.cls_qb);
  const float ql = q * lam;
  return (ql > P.cls_lo) && (ql < P.cls_hi);
}

// From the words of Philox blocks 0 and 1 to the detector pixel.  Returns the ST_* outcome.
// FAST is the instrument class of every BASELINE.json config with a box sample (ExpParams::geo_fast, set by the
// host): no slit can cut a stage-B ray (slits_free), the primary ray cannot touch the sample's lateral faces
// (lateral_free), box sample, no attenuation.  What is left of R-C4/R-C5/R-C11 is the depth slab alone, whose
// roots need no min/max (dz > 0 and hz > 0: (-hz - oz) inv <= (hz - oz) inv by monotonic rounding) -- the same
// values as the general code, without its runtime branches.
template <bool FAST>
__device__ __forceinline__ int trace_geometry(const ExpParams& P, const uint32_t w[4], const uint32_t w1[4], Hit& h) {
  // R-C2 source point
  const double u0 = uniform_from_word(w[0]), u1 = uniform_from_word(w[1]);
  const double u2 = uniform_from_word(w[2]), u3 = uniform_from_word(w[3]);
  const double x0 = (u0 - 0.5) * P.src_xw;
  const double y0 = (u1 - 0.5) * P.src_yh;
  // R-C3 aim at a uniform point of the focus rectangle (z0 = 0: Dz = focus_z - 0)
  const double xt = (u2 - 0.5) * P.focus_xw;
  const double yt = (u3 - 0.5) * P.focus_yh;
  const double Dx = xt - x0, Dy = yt - y0, Dz = P.focus_z - 0.0;
  const double r2 = (Dx * Dx + Dy * Dy) + Dz * Dz;
  const double r = sqrt(r2);
  const double inv_r = 1.0 / r;
  const double dx = Dx * inv_r, dy = Dy * inv_r, dz = Dz * inv_r;
  const double dOmega = ((P.focus_area * dz) * inv_r) * inv_r;
  const double p0 = (P.p0_pref * dOmega) * P.dlam_w;
  // R-C4 slits.  slits_free: stage A already applied the (bit-identical) integer slit-1 test and the host
  // proved that slit 2 cannot cut a ray aimed at the focus rectangle: nothing to compute
  bool f_s1 = false, f_s2 = false;
  if (!FAST && !P.slits_free) {
    const double inv_dz = 1.0 / dz;
    const double s1 = (P.slit1_z - 0.0) * inv_dz;
    const double xs1 = x0 + dx * s1, ys1 = y0 + dy * s1;
    f_s1 = fabs(xs1) > P.slit1_hx || fabs(ys1) > P.slit1_hy;
    const double s2s = (P.slit2_z - 0.0) * inv_dz;
    const double xs2 = x0 + dx * s2s, ys2 = y0 + dy * s2s;
    f_s2 = fabs(xs2) > P.slit2_hx || fabs(ys2) > P.slit2_hy;
  }
  // draws 4..7 (Philox block 1, drawn by the classifier stage)
  const double u4 = uniform_from_word(w1[0]), u5 = uniform_from_word(w1[1]);
  const double u6 = uniform_from_word(w1[2]), u7 = uniform_from_word(w1[3]);
  const double lambda = lambda_from_u(P, u4);
  // R-C5 sample
  double tin, tout;
  bool hit_s = true;
  if (FAST) {
    const double oz = 0.0 - P.sample_z, inv = 1.0 / dz;
    tin = (-P.hz - oz) * inv;
    tout = (P.hz - oz) * inv;
  } else {
    hit_s = intersect_sample(P, x0, y0, 0.0 - P.sample_z, dx, dy, dz, tin, tout, P.lateral_free != 0);
  }
  tin = tin < 0.0 ? 0.0 : tin;
  const bool f_ms = !hit_s || !(tout > tin);
  const double ell = tout - tin;
  // R-C6 scattering point
  const double ts = tin + u5 * ell;
  const double rsx = x0 + dx * ts, rsy = y0 + dy * ts, rsz = 0.0 + dz * ts;
  // R-C7 |Q| and azimuth
  const double q = P.q_min + u6 * P.dq;
  const double chi = 6.283185307179586 * u7;
  const double k = 6.283185307179586 / lambda;
  const double inv_k = lambda / 6.283185307179586;
  const double qk = q * inv_k;
  const double s = 0.5 * qk;
  const bool f_un = s >= 1.0;
  const double ss2 = 2.0 * (s * s);
  const double c2 = 1.0 - ss2;
  const double s2 = 2.0 * (s * sqrt(1.0 - s * s));
  // R-C8 outgoing direction
  const double n = sqrt(dz * dz + dx * dx);
  const double inv_n = 1.0 / n;
  const double e1x = dz * inv_n, e1z = -(dx * inv_n);
  const double e2x = dy * e1z, e2y = dz * e1x - dx * e1z, e2z = -(dy * e1x);
  double sc, cc;
  sincos_cw(chi, sc, cc);  // chi in (0, 2 pi)
  const double tx = cc * e1x + sc * e2x, ty = sc * e2y, tz = cc * e1z + sc * e2z;
  const double dpx = c2 * dx + s2 * tx, dpy = c2 * dy + s2 * ty, dpz = c2 * dz + s2 * tz;
  h.Qx = k * (ss2 * dx - s2 * tx);
  h.Qy = k * (ss2 * dy - s2 * ty);
  h.Qz = k * (ss2 * dz - s2 * tz);
  // R-C9 detector
  const double inv_dpz = 1.0 / dpz;
  const double td = (P.det_z - rsz) * inv_dpz;
  const double X = rsx + dpx * td, Y = rsy + dpy * td;
  const double fx = (X + P.det_hw) * P.det_sx;
  const double fy = (Y + P.det_hh) * P.det_sy;
  const bool f_md = !(dpz > 0.0) || !(fx >= 0.0 && fx < P.det_nxd && fy >= 0.0 && fy < P.det_nyd);
  // outcome, in the order of the design note
  int st = ST_DETECTED;
  st = f_md ? ST_MISS_DET : st;
  st = f_un ? ST_UNREACHABLE : st;
  st = f_ms ? ST_MISS_SAMPLE : st;
  st = f_s2 ? ST_SLIT2 : st;
  st = f_s1 ? ST_SLIT1 : st;
  h.q = (f_s1 || f_s2 || f_ms) ? 0.0 : q;
  h.pixel = -1;
  if (st == ST_DETECTED) {
    h.pixel = (int)floor(fy) * P.det_nx + (int)floor(fx);
    // R-C11 attenuation and the geometric part of the weight
    double T = 1.0;
    if (!FAST && P.has_mu) {
      const double mu = (P.mu_abs_2200 * lambda) / 1.7982 + P.mu_inc;
      double tin2, tout2, ell_out = 0.0;
      if (intersect_sample(P, rsx, rsy, rsz - P.sample_z, dpx, dpy, dpz, tin2, tout2) && tout2 > 0.0) ell_out = tout2;
      T = exp(-(mu * (u5 * ell + ell_out)));
    }
    const double geo = (FAST ? p0 : p0 * T) * (100.0 * ell);  // p0 * 1.0 is p0
    h.G = (geo * (qk * inv_k)) * P.qnorm;
  }
  return st;
}

}  // namespace sas
