// fp64 geometry of one neutron between the source and the detector (DESIGN.md R-C2..R-C11).
// Written operation by operation as the design note states them; the translation unit is compiled
// with -fmad=false, so nothing here is contracted and the detector pixel is bit-identical to a
// plain IEEE evaluation of the same text.
#pragma once
#include "sas_types.h"

namespace sas {

// Ray (o + t d) against the sample volume centred on the origin of the sample frame (R-C5).
__device__ __forceinline__ bool intersect_sample(const ExpParams& P, double ox, double oy, double oz, double dx,
                                                 double dy, double dz, double& t_in, double& t_out) {
  double tin = -INFINITY, tout = INFINITY;
  bool cyl = P.sample_shape == 1;
  if (cyl) {
    const double a = dx * dx + dz * dz;
    const double b = ox * dx + oz * dz;
    const double c = (ox * ox + oz * oz) - P.radius2;
    if (a == 0.0) {
      if (c > 0.0) return false;
    } else {
      const double disc = b * b - a * c;
      if (!(disc > 0.0)) return false;
      const double sq = sqrt(disc);
      const double inv_a = 1.0 / a;
      tin = (-b - sq) * inv_a;
      tout = (-b + sq) * inv_a;
    }
  } else {
    // x slab
    if (dx == 0.0) {
      if (fabs(ox) > P.hx) return false;
    } else {
      const double inv = 1.0 / dx;
      double t1 = (-P.hx - ox) * inv, t2 = (P.hx - ox) * inv;
      if (t1 > t2) { const double t = t1; t1 = t2; t2 = t; }
      if (t1 > tin) tin = t1;
      if (t2 < tout) tout = t2;
    }
  }
  // y slab (box and cylinder height)
  if (dy == 0.0) {
    if (fabs(oy) > P.hy) return false;
  } else {
    const double inv = 1.0 / dy;
    double t1 = (-P.hy - oy) * inv, t2 = (P.hy - oy) * inv;
    if (t1 > t2) { const double t = t1; t1 = t2; t2 = t; }
    if (t1 > tin) tin = t1;
    if (t2 < tout) tout = t2;
  }
  if (!cyl) {
    if (dz == 0.0) {
      if (fabs(oz) > P.hz) return false;
    } else {
      const double inv = 1.0 / dz;
      double t1 = (-P.hz - oz) * inv, t2 = (P.hz - oz) * inv;
      if (t1 > t2) { const double t = t1; t1 = t2; t2 = t; }
      if (t1 > tin) tin = t1;
      if (t2 < tout) tout = t2;
    }
  }
  t_in = tin;
  t_out = tout;
  return true;
}

struct Hit {
  int32_t pixel;
  double G;      // p0 * T * 100 ell * (q/k^2) * 2 pi (qmax - qmin): the weight is G * I(Q)
  double Qx, Qy, Qz;
  double q;      // drawn |Q| (0 if the neutron died before the draw)
};

// From the four words of Philox block 0 to the detector pixel.  Returns the ST_* outcome.
__device__ __forceinline__ int trace_geometry(const ExpParams& P, const PhiloxKeys& keys, uint32_t id_lo,
                                              uint32_t id_hi, uint32_t exp_word, const uint32_t w[4], Hit& h) {
  h.q = 0.0;
  h.pixel = -1;
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
  // R-C4 slits
  const double inv_dz = 1.0 / dz;
  {
    const double s = (P.slit1_z - 0.0) * inv_dz;
    const double xs = x0 + dx * s, ys = y0 + dy * s;
    if (fabs(xs) > P.slit1_hx || fabs(ys) > P.slit1_hy) return ST_SLIT1;
  }
  {
    const double s = (P.slit2_z - 0.0) * inv_dz;
    const double xs = x0 + dx * s, ys = y0 + dy * s;
    if (fabs(xs) > P.slit2_hx || fabs(ys) > P.slit2_hy) return ST_SLIT2;
  }
  // draws 4..7
  uint32_t w1[4];
  philox4x32_10(keys, id_lo, id_hi, 1u, exp_word, w1);
  const double u4 = uniform_from_word(w1[0]), u5 = uniform_from_word(w1[1]);
  const double u6 = uniform_from_word(w1[2]), u7 = uniform_from_word(w1[3]);
  const double lambda = P.lambda_min + u4 * P.dlam;
  // R-C5 sample
  double tin, tout;
  if (!intersect_sample(P, x0, y0, 0.0 - P.sample_z, dx, dy, dz, tin, tout)) return ST_MISS_SAMPLE;
  if (tin < 0.0) tin = 0.0;
  if (!(tout > tin)) return ST_MISS_SAMPLE;
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
  h.q = q;
  if (s >= 1.0) return ST_UNREACHABLE;
  const double ss2 = 2.0 * (s * s);
  const double c2 = 1.0 - ss2;
  const double s2 = 2.0 * (s * sqrt(1.0 - s * s));
  // R-C8 outgoing direction
  const double n = sqrt(dz * dz + dx * dx);
  const double inv_n = 1.0 / n;
  const double e1x = dz * inv_n, e1z = -(dx * inv_n);
  const double e2x = dy * e1z, e2y = dz * e1x - dx * e1z, e2z = -(dy * e1x);
  double sc, cc;
  sincos(chi, &sc, &cc);
  const double tx = cc * e1x + sc * e2x, ty = sc * e2y, tz = cc * e1z + sc * e2z;
  const double dpx = c2 * dx + s2 * tx, dpy = c2 * dy + s2 * ty, dpz = c2 * dz + s2 * tz;
  h.Qx = k * (ss2 * dx - s2 * tx);
  h.Qy = k * (ss2 * dy - s2 * ty);
  h.Qz = k * (ss2 * dz - s2 * tz);
  // R-C9 detector
  if (!(dpz > 0.0)) return ST_MISS_DET;
  const double inv_dpz = 1.0 / dpz;
  const double td = (P.det_z - rsz) * inv_dpz;
  const double X = rsx + dpx * td, Y = rsy + dpy * td;
  const double fx = (X + P.det_hw) * P.det_sx;
  const double fy = (Y + P.det_hh) * P.det_sy;
  if (!(fx >= 0.0 && fx < P.det_nxd && fy >= 0.0 && fy < P.det_nyd)) return ST_MISS_DET;
  h.pixel = (int)floor(fy) * P.det_nx + (int)floor(fx);
  // R-C11 attenuation and the geometric part of the weight
  double T = 1.0;
  if (P.has_mu) {
    const double mu = (P.mu_abs_2200 * lambda) / 1.7982 + P.mu_inc;
    double tin2, tout2, ell_out = 0.0;
    if (intersect_sample(P, rsx, rsy, rsz - P.sample_z, dpx, dpy, dpz, tin2, tout2) && tout2 > 0.0) ell_out = tout2;
    T = exp(-(mu * (u5 * ell + ell_out)));
  }
  const double geo = (p0 * T) * (100.0 * ell);
  h.G = (geo * (qk * inv_k)) * P.qnorm;
  return ST_DETECTED;
}

}  // namespace sas
