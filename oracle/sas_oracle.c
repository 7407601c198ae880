/*
 * sas_oracle.c -- TEST INFRASTRUCTURE ONLY (see sas_oracle.h).
 *
 * The oracle of the SANS Monte-Carlo hot path: one neutron at a time, fp64,
 * in the order and notation of DESIGN.md section 3 ("readings" R-A*, R-B,
 * R-C*), which restate PAPER.md where the paper speaks and fix a reading where
 * it is silent.  No blocking, fusion or reordering.  Every expression is
 * written so that, compiled with -ffp-contract=off, each operation is rounded
 * once, left to right.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors,
 * closed forms of the sphere, brute-force Eq. 1 integrals for cylinder and
 * ellipsoid, mpmath values of PY S(q) and 2J1(x)/x, weight conservation of the
 * flat model, pencil-beam chi^2 against the numerically integrated I(Q),
 * Guinier radii, model reductions; NEXT-1 (tests/test_oracle_paper_sampling.py):
 * normal / truncated-normal laws of the per-event sizes, raw-Philox draw layout,
 * numpy integrals of F^2/V, isotropic vs printed orientation law; NEXT-2
 * (tests/test_oracle_more_models.py): Eq. 1 integrated over the box, the
 * core-shell cylinder and the ellipsoid of revolution.  "parity unpinned": whole detector images
 * of configs c1-c4 have no external pin beyond those pieces (DESIGN.md s.3.D).
 */
#define _GNU_SOURCE
#include "sas_oracle.h"

#include <math.h>
#include <string.h>

static const double TWO_PI = 6.283185307179586;
static const double FOUR_PI_3 = 4.1887902047863905; /* 4 pi / 3 */
static const double PI_ = 3.141592653589793;

/* ------------------------------------------------------------------ R-B */
/* Philox4x32-10: multipliers 0xD2511F53, 0xCD9E8D57; Weyl key increments
 * 0x9E3779B9, 0xBB67AE85; ten rounds (Salmon, Moraes, Dror, Shaw, SC'11). */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* u = (w + 0.5) * 2^-32, exact in fp64, in (0,1). */
double orc_uniform(uint32_t word) { return ((double)word + 0.5) * 2.3283064365386963e-10; }

/* draw block `block` of neutron `id` of experiment `exp`: ctr=(id_lo,id_hi,block,exp) */
static void draw_block(uint64_t seed, uint64_t id, uint32_t block, uint32_t exp_index, double u4[4]) {
  uint32_t ctr[4] = {(uint32_t)(id & 0xFFFFFFFFu), (uint32_t)(id >> 32), block, exp_index};
  uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
  uint32_t w[4];
  orc_philox4x32_10(ctr, key, w);
  for (int i = 0; i < 4; ++i) u4[i] = orc_uniform(w[i]);
}

/* -------------------------------------------------------------- R-C12 */
/* Phi(u) = 3 (sin u - u cos u) / u^3 : sphere amplitude, PAPER.md:37 (Eq. 1
 * integrated over a sphere).  Even series below u = 0.5 where the direct form
 * cancels. */
double orc_sphere_phi(double u) {
  if (fabs(u) < 0.5) {
    double u2 = u * u;
    double s = 1.0 / 31135104000.0;
    s = s * u2 - 1.0 / 172972800.0;
    s = s * u2 + 1.0 / 1330560.0;
    s = s * u2 - 1.0 / 15120.0;
    s = s * u2 + 1.0 / 280.0;
    s = s * u2 - 1.0 / 10.0;
    s = s * u2 + 1.0;
    return s;
  }
  return (3.0 * (sin(u) - u * cos(u))) / ((u * u) * u);
}

double orc_sinc(double x) {
  if (x == 0.0) return 1.0;
  return sin(x) / x;
}

/* Lambda(x) = 2 J1(x) / x, the disc factor of the cylinder. */
double orc_lambda1(double x) {
  if (x == 0.0) return 1.0;
  return (2.0 * j1(x)) / x;
}

/* -------------------------------------------------------------- R-C13 */
/* Percus-Yevick hard-sphere structure factor (Table II F.11). */
double orc_py_sq(double q, double r_eff, double volfrac) {
  double phi = volfrac;
  double x = 2.0 * (q * r_eff);
  double om = 1.0 - phi;
  double om4 = (om * om) * (om * om);
  double alpha = ((1.0 + 2.0 * phi) * (1.0 + 2.0 * phi)) / om4;
  double beta = (-6.0 * phi) * ((1.0 + 0.5 * phi) * (1.0 + 0.5 * phi)) / om4;
  double gamma = (phi * alpha) * 0.5;
  double t1, t2, t3;
  if (x < 1.0) {
    static const double a1[8] = {1.0 / 3.0, -1.0 / 30.0, 1.0 / 840.0, -1.0 / 45360.0,
                                 1.0 / 3991680.0, -1.0 / 518918400.0, 1.0 / 93405312000.0,
                                 -1.0 / 22230464256000.0};
    static const double a2[8] = {1.0 / 4.0, -1.0 / 36.0, 1.0 / 960.0, -1.0 / 50400.0,
                                 1.0 / 4354560.0, -1.0 / 558835200.0, 1.0 / 99632332800.0,
                                 -1.0 / 23538138624000.0};
    static const double a3[8] = {1.0 / 6.0, -1.0 / 48.0, 1.0 / 1200.0, -1.0 / 60480.0,
                                 1.0 / 5080320.0, -1.0 / 638668800.0, 1.0 / 112086374400.0,
                                 -1.0 / 26153487360000.0};
    double x2 = x * x;
    t1 = a1[7]; t2 = a2[7]; t3 = a3[7];
    for (int i = 6; i >= 0; --i) {
      t1 = t1 * x2 + a1[i];
      t2 = t2 * x2 + a2[i];
      t3 = t3 * x2 + a3[i];
    }
  } else {
    double s = sin(x), c = cos(x);
    double x2 = x * x, x3 = x2 * x, x4 = x2 * x2, x6 = x3 * x3;
    t1 = (s - x * c) / x3;
    t2 = ((2.0 * x) * s + (2.0 - x2) * c - 2.0) / x4;
    t3 = (-(x4 * c) + 4.0 * (((3.0 * x2 - 6.0) * c + (x3 - 6.0 * x) * s) + 6.0)) / x6;
  }
  return 1.0 / (1.0 + (24.0 * phi) * ((alpha * t1 + beta * t2) + gamma * t3));
}

/* n-node Gauss-Legendre rule on [-1, 1] (nodes ascending, weights summing to 2): Newton iteration on the
 * Legendre polynomial P_n from the Chebyshev-like starting points, the textbook construction. */
static void gl_rule(int n, double* xs, double* ws) {
  for (int i = 0; i < n; ++i) {
    double x = cos(PI_ * ((double)i + 0.75) / ((double)n + 0.5));
    double dp = 1.0;
    for (int it = 0; it < 100; ++it) {
      double p0 = 1.0, p1 = x;
      for (int k = 2; k <= n; ++k) {
        double pk = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
        p0 = p1; p1 = pk;
      }
      dp = n * (x * p1 - p0) / (x * x - 1.0);
      double dx = p1 / dp;
      x -= dx;
      if (fabs(dx) < 1e-16) break;
    }
    xs[n - 1 - i] = x;
    ws[n - 1 - i] = 2.0 / ((1.0 - x * x) * dp * dp);
  }
}
#define ORC_GL_N 32
static double gl_x[ORC_GL_N], gl_w[ORC_GL_N];
static int gl_ready = 0;
static void gl_init(void) {
  if (gl_ready) return;
  gl_rule(ORC_GL_N, gl_x, gl_w);
  gl_ready = 1;
}

/* R-S2: Hayter-Penfold MSA structure factor from the Baxter function the caller solved for (sas_oracle.h).
 * With x in units of the diameter and K = q sigma:
 *   Qhat(K) = 1 - 12 eta [ int_0^1 Q_in(x) e^{iKx} dx + D' e^{iK} / (k - iK) ],   S = 1 / |Qhat|^2. */
double orc_msa_sq(double q, const orc_model* m) {
  static double x64[64], w64[64];
  static int ready = 0;
  if (!ready) { gl_rule(64, x64, w64); ready = 1; }
  double K = q * (2.0 * m->sq_radius_eff), eta = m->sq_volfrac, k = m->sq_kappa_sigma;
  double a = m->msa[0], b = m->msa[1], E = m->msa[2], Cp = m->msa[3], Dp = m->msa[4];
  double re = 0.0, im = 0.0;
  for (int j = 0; j < 64; ++j) {
    double x = 0.5 * (x64[j] + 1.0), w = 0.5 * w64[j];
    double Qin = ((0.5 * a) * (x * x - 1.0) + b * (x - 1.0)) + (E * exp(-k * x) - Cp);
    re += (w * Qin) * cos(K * x);
    im += (w * Qin) * sin(K * x);
  }
  double den = k * k + K * K;
  re += Dp * (k * cos(K) - K * sin(K)) / den;   /* Re, Im of e^{iK} / (k - iK) = e^{iK} (k + iK) / (k^2 + K^2) */
  im += Dp * (k * sin(K) + K * cos(K)) / den;
  re = 1.0 - (12.0 * eta) * re;
  im = -(12.0 * eta) * im;
  return 1.0 / (re * re + im * im);
}

/* R-M2: end piece of a body of revolution about C: the part z in [L/2, zc + Rb] of the sphere of radius Rb
 * centred on the axis at zc.  Eq. 1 slice by slice: a slice at height z is a disc of radius rho(z) whose
 * in-plane integral is pi rho^2 Lambda(Q_AB rho); the two end pieces at +-z add up to 2 cos(Q_C z).
 * Returns the integral for ONE end piece without the factor 2; *vcap its volume. */
static double end_piece(double qab, double qc, double L, double Rb, double zc, double* vcap) {
  gl_init();
  double z0 = 0.5 * L, z1 = zc + Rb;
  double half = 0.5 * (z1 - z0), mid = 0.5 * (z1 + z0);
  double sum = 0.0;
  for (int i = 0; i < ORC_GL_N; ++i) {
    double z = mid + half * gl_x[i];
    double dz = z - zc;
    double rho2 = Rb * Rb - dz * dz;
    if (rho2 < 0.0) rho2 = 0.0;
    double rho = sqrt(rho2);
    sum += gl_w[i] * (((PI_ * rho2) * orc_lambda1(qab * rho)) * cos(qc * z));
  }
  double a = z1 - zc, b = z0 - zc;
  *vcap = PI_ * ((Rb * Rb) * (z1 - z0) - (((a * a) * a) - ((b * b) * b)) / 3.0);
  return half * sum;
}

/* ------------------------------------------------------ R-C12 amplitudes */
/* One particle, sizes scaled by the polydispersity node values x0, x1
 * (R-A12).  qa,qb,qc: projections of Q on the particle axes (PAPER.md:76-82,
 * Eq. 6-7).  Returns F = integral of Delta-rho exp(-iQr) (real for these
 * centro-symmetric shapes); *vol = normalising volume V_m
 * (PAPER.md:49); *env = F with every shape factor set to 1. */
double orc_amplitude(const orc_model* m, double qa, double qb, double qc, double x0, double x1,
                     double* vol, double* env) {
  double q = sqrt((qa * qa + qb * qb) + qc * qc);
  switch (m->model) {
    case ORC_SPHERE: {
      double R = m->size[0] * x0;
      double V = FOUR_PI_3 * ((R * R) * R);
      *vol = V;
      *env = m->sld[0] * V;
      return (m->sld[0] * V) * orc_sphere_phi(q * R);
    }
    case ORC_CORE_SHELL_SPHERE: {
      double Rc = m->size[0] * x0;
      double t = m->size[1] * x1;
      double Rt = Rc + t;
      double Vc = FOUR_PI_3 * ((Rc * Rc) * Rc);
      double Vt = FOUR_PI_3 * ((Rt * Rt) * Rt);
      double fc = (m->sld[0] - m->sld[1]) * Vc;
      double ft = m->sld[1] * Vt;
      *vol = Vt;
      *env = fabs(fc) + fabs(ft);
      return fc * orc_sphere_phi(q * Rc) + ft * orc_sphere_phi(q * Rt);
    }
    case ORC_CYLINDER: {
      /* Eq. 9 with the projections as Eq. 1 gives them (R-A4):
       * F = 2 drho V sinc(Q_C L/2) J1(Q_AB R)/(Q_AB R), V = pi R^2 L. */
      double R = m->size[0] * x0;
      double L = m->size[1] * x1;
      double V = (PI_ * (R * R)) * L;
      double qab = sqrt(qa * qa + qb * qb);
      *vol = V;
      *env = m->sld[0] * V;
      return ((m->sld[0] * V) * orc_sinc(qc * (0.5 * L))) * orc_lambda1(qab * R);
    }
    case ORC_TRIAXIAL: {
      double a = m->size[0] * x0, b = m->size[1] * x0, c = m->size[2] * x0;
      double V = FOUR_PI_3 * ((a * b) * c);
      double u = sqrt(((a * qa) * (a * qa) + (b * qb) * (b * qb)) + (c * qc) * (c * qc));
      *vol = V;
      *env = m->sld[0] * V;
      return (m->sld[0] * V) * orc_sphere_phi(u);
    }
    case ORC_CORE_SHELL_TRIAXIAL: {
      double a = m->size[0] * x0, b = m->size[1] * x0, c = m->size[2] * x0;
      double t = m->size[3] * x1;
      double at = a + t, bt = b + t, ct = c + t;
      double Vc = FOUR_PI_3 * ((a * b) * c);
      double Vt = FOUR_PI_3 * ((at * bt) * ct);
      double uc = sqrt(((a * qa) * (a * qa) + (b * qb) * (b * qb)) + (c * qc) * (c * qc));
      double ut = sqrt(((at * qa) * (at * qa) + (bt * qb) * (bt * qb)) + (ct * qc) * (ct * qc));
      double fc = (m->sld[0] - m->sld[1]) * Vc;
      double ft = m->sld[1] * Vt;
      *vol = Vt;
      *env = fabs(fc) + fabs(ft);
      return fc * orc_sphere_phi(uc) + ft * orc_sphere_phi(ut);
    }
    case ORC_PARALLELEPIPED: {
      /* Eq. 1 over the box |x|<=a/2, |y|<=b/2, |z|<=c/2 along A, B, C: the three 1-D integrals are
       * a sinc(Q_A a/2) etc.  One common size scale x0 (as the triaxial ellipsoid, R-A12). */
      double a = m->size[0] * x0, b = m->size[1] * x0, c = m->size[2] * x0;
      double V = (a * b) * c;
      *vol = V;
      *env = m->sld[0] * V;
      return (m->sld[0] * V) * ((orc_sinc(qa * (0.5 * a)) * orc_sinc(qb * (0.5 * b))) * orc_sinc(qc * (0.5 * c)));
    }
    case ORC_HOLLOW_PRISM_THIN: {
      /* R-M5: rectangular prism a x b x c along A, B, C whose contrast sits in walls of thickness t -> 0 on its six
       * faces (first order in t): Eq. 1 becomes a surface integral, F = sld t * sum over the faces of
       * int exp(i Q.r) dS.  The two faces at x = +-a/2 give 2 cos(Q_A a/2) * [b sinc(Q_B b/2)] [c sinc(Q_C c/2)],
       * and so on cyclically.  Normalising volume = wall volume t * 2 (ab + bc + ca).  x0 scales a, b, c. */
      double a = m->size[0] * x0, b = m->size[1] * x0, c = m->size[2] * x0, t = m->size[3];
      double sa = orc_sinc(qa * (0.5 * a)), sb = orc_sinc(qb * (0.5 * b)), sc = orc_sinc(qc * (0.5 * c));
      double ca = cos(qa * (0.5 * a)), cb = cos(qb * (0.5 * b)), cc = cos(qc * (0.5 * c));
      double faces = (((b * c) * ca) * (sb * sc) + ((a * c) * cb) * (sa * sc)) + ((a * b) * cc) * (sa * sb);
      double V = t * (2.0 * ((a * b + b * c) + c * a));
      *vol = V;
      *env = m->sld[0] * V;
      return (m->sld[0] * t) * (2.0 * faces);
    }
    case ORC_CORE_SHELL_CYLINDER: {
      /* core cylinder (R, L) of contrast sld[0] inside a cylinder (R+t, L+2t) of contrast sld[1]:
       * Eq. 1 with a piecewise contrast = (sld0-sld1) x core + sld1 x whole; x0 scales R, x1 scales L */
      double R = m->size[0] * x0, L = m->size[1] * x1, t = m->size[2];
      double Rt = R + t, Lt = L + 2.0 * t;
      double Vc = (PI_ * (R * R)) * L;
      double Vt = (PI_ * (Rt * Rt)) * Lt;
      double qab = sqrt(qa * qa + qb * qb);
      double fc = (m->sld[0] - m->sld[1]) * Vc;
      double ft = m->sld[1] * Vt;
      *vol = Vt;
      *env = fabs(fc) + fabs(ft);
      return (fc * orc_sinc(qc * (0.5 * L))) * orc_lambda1(qab * R) +
             (ft * orc_sinc(qc * (0.5 * Lt))) * orc_lambda1(qab * Rt);
    }
    case ORC_ELLIPSOID: {
      /* ellipsoid of revolution about C: the sphere amplitude at u = sqrt(R_e^2 Q_AB^2 + R_p^2 Q_C^2);
       * x0 scales the equatorial, x1 the polar radius */
      double Re = m->size[0] * x0, Rp = m->size[1] * x1;
      double V = FOUR_PI_3 * ((Re * Re) * Rp);
      double u = sqrt((Re * Re) * (qa * qa + qb * qb) + (Rp * qc) * (Rp * qc));
      *vol = V;
      *env = m->sld[0] * V;
      return (m->sld[0] * V) * orc_sphere_phi(u);
    }
    case ORC_ELLIPTICAL_CYLINDER: {
      /* Eq. 1 over {x^2/a^2 + y^2/b^2 <= 1, |z| <= L/2}: the elliptic disc is a unit disc stretched by (a, b), so its
       * in-plane integral is pi a b Lambda(sqrt((a Q_A)^2 + (b Q_B)^2)); x0 scales a and b, x1 scales L */
      double a = m->size[0] * x0, b = m->size[1] * x0, L = m->size[2] * x1;
      double V = (PI_ * (a * b)) * L;
      double u = sqrt((a * qa) * (a * qa) + (b * qb) * (b * qb));
      *vol = V;
      *env = m->sld[0] * V;
      return ((m->sld[0] * V) * orc_sinc(qc * (0.5 * L))) * orc_lambda1(u);
    }
    case ORC_HOLLOW_CYLINDER: {
      /* tube = cylinder of radius R + t minus the hollow core of radius R, same length; normalised by the volume of
       * the wall; x0 scales the core radius, x1 the length, the wall keeps its thickness */
      double Ri = m->size[0] * x0, L = m->size[1] * x1, t = m->size[2];
      double Ro = Ri + t;
      double Vo = (PI_ * (Ro * Ro)) * L, Vi = (PI_ * (Ri * Ri)) * L;
      double qab = sqrt(qa * qa + qb * qb);
      double sl = orc_sinc(qc * (0.5 * L));
      *vol = Vo - Vi;
      *env = m->sld[0] * (Vo + Vi);
      return m->sld[0] * ((Vo * sl) * orc_lambda1(qab * Ro) - (Vi * sl) * orc_lambda1(qab * Ri));
    }
    case ORC_CORE_SHELL_ELLIPSOID: {
      /* core ellipsoid of revolution (R_e, R_p) of contrast sld[0] inside the ellipsoid (R_e + t, R_p + t) of
       * contrast sld[1]; x0 scales R_e, x1 scales R_p */
      double Re = m->size[0] * x0, Rp = m->size[1] * x1, t = m->size[2];
      double Ret = Re + t, Rpt = Rp + t;
      double Vc = FOUR_PI_3 * ((Re * Re) * Rp), Vt = FOUR_PI_3 * ((Ret * Ret) * Rpt);
      double qab2 = qa * qa + qb * qb;
      double uc = sqrt((Re * Re) * qab2 + (Rp * qc) * (Rp * qc));
      double ut = sqrt((Ret * Ret) * qab2 + (Rpt * qc) * (Rpt * qc));
      double fc = (m->sld[0] - m->sld[1]) * Vc, ft = m->sld[1] * Vt;
      *vol = Vt;
      *env = fabs(fc) + fabs(ft);
      return fc * orc_sphere_phi(uc) + ft * orc_sphere_phi(ut);
    }
    case ORC_BARBELL:
    case ORC_CAPPED_CYLINDER: {
      /* R-M2: cylinder (R, L) along C plus two spherical end pieces of radius Rb >= R; x0 scales R, x1 scales L */
      double R = m->size[0] * x0, L = m->size[1] * x1, Rb = m->size[2];
      double h2 = Rb * Rb - R * R;
      double h = sqrt(h2 > 0.0 ? h2 : 0.0);
      double zc = m->model == ORC_BARBELL ? 0.5 * L + h : 0.5 * L - h;
      double qab = sqrt(qa * qa + qb * qb);
      double vcap;
      double cap = end_piece(qab, qc, L, Rb, zc, &vcap);
      double Vcyl = (PI_ * (R * R)) * L;
      double V = Vcyl + 2.0 * vcap;
      *vol = V;
      *env = m->sld[0] * V;
      return m->sld[0] * ((Vcyl * orc_sinc(qc * (0.5 * L))) * orc_lambda1(qab * R) + 2.0 * cap);
    }
    default:
      *vol = 1.0;
      *env = 1.0;
      return 1.0;
  }
}

/* R-M4: Gaussian chain of gyration radius R_g, x = (q R_g)^2.  The chain is a continuous random walk of contour
 * length 1 whose points s, s' are separated by a Gaussian of variance proportional to |s - s'|:
 * <exp(i q (r_s - r_s'))> = exp(-x |s - s'|).  Debye function = double average over s, s' in [0, 1];
 * psi = single average over s of exp(-x s) (amplitude seen from the attached end).  Series below x = 0.1, where
 * the closed forms cancel (2 ulp / x^2): D = sum_k 2 (-x)^k / (k + 2)!, psi = sum_k (-x)^k / (k + 1)!. */
double orc_debye(double x) {
  if (x < 0.1) {
    double sum = 0.0, term = 1.0;             /* term = (-x)^k / (k + 2)! * 2, starting at k = 0: 2 / 2! = 1 */
    for (int k = 0; k < 12; ++k) {
      sum += term;
      term *= -x / (double)(k + 3);
    }
    return sum;
  }
  return 2.0 * ((exp(-x) - 1.0) + x) / (x * x);
}
double orc_chain_psi(double x) {
  if (x < 0.1) {
    double sum = 0.0, term = 1.0;             /* term = (-x)^k / (k + 1)! */
    for (int k = 0; k < 12; ++k) {
      sum += term;
      term *= -x / (double)(k + 2);
    }
    return sum;
  }
  return (1.0 - exp(-x)) / x;
}

/* R-M4 (Pedersen & Gerstenberg 1996): core of radius R = size[0] x0 and excess scattering length
 * B_s = sld[0] V_core; N = size[3] chains of gyration radius R_g = size[1], volume V_c = size[2] and excess
 * scattering length b_c = sld[1] V_c each, starting at radius R + d R_g with d = 1, mutually independent and
 * uniformly distributed over the surface:
 *   |F|^2 = B_s^2 Phi(qR)^2 + N b_c^2 D(x) + N (N - 1) b_c^2 [psi(x) sinc(q(R + R_g))]^2
 *           + 2 N B_s b_c Phi(qR) psi(x) sinc(q(R + R_g)),        x = (q R_g)^2.
 * Normalising volume: V_core + N V_c. */
double orc_micelle_f2(const orc_model* m, double q, double x0, double* vol, double* env2) {
  double R = m->size[0] * x0, Rg = m->size[1], Vc = m->size[2], N = m->size[3];
  double Vcore = FOUR_PI_3 * ((R * R) * R);
  double Bs = m->sld[0] * Vcore, bc = m->sld[1] * Vc;
  double x = (q * Rg) * (q * Rg);
  double phi = orc_sphere_phi(q * R);
  double ps = orc_chain_psi(x) * orc_sinc(q * (R + Rg));
  double self_core = (Bs * Bs) * (phi * phi);
  double self_chain = (N * (bc * bc)) * orc_debye(x);
  double chain_chain = ((N * (N - 1.0)) * (bc * bc)) * (ps * ps);
  double cross = ((2.0 * N) * (Bs * bc)) * (phi * ps);
  *vol = Vcore + N * Vc;
  double e = fabs(Bs) + N * fabs(bc);
  *env2 = e * e;
  return ((self_core + self_chain) + chain_chain) + cross;
}

/* particle frame from (theta, phi, psi): R-A7 */
static void frame_from_angles(double st, double ct, double sp, double cp, double ss, double cs,
                              double A[3], double B[3], double C[3]) {
  double a0[3] = {ct * cp, ct * sp, -st};
  double b0[3] = {-sp, cp, 0.0};
  C[0] = st * cp; C[1] = st * sp; C[2] = ct;
  for (int i = 0; i < 3; ++i) {
    A[i] = cs * a0[i] + ss * b0[i];
    B[i] = cs * b0[i] - ss * a0[i];
  }
}

static double dot3(const double a[3], const double b[3]) { return (a[0] * b[0] + a[1] * b[1]) + a[2] * b[2]; }

/* particle axes of one event: fixed angles, or drawn per event (R-A3 isotropic; R-N3 the paper's printed
 * uniform angles) */
static void particle_frame(const orc_model* m, const double u_or[3], double A[3], double B[3], double C[3]) {
  if (m->orient_kind == ORC_ORIENT_ISOTROPIC_MC) {
    /* R-A3: isotropic = cos(theta) uniform, phi and psi uniform */
    double ct = 1.0 - 2.0 * u_or[0];
    double st = sqrt(1.0 - ct * ct);
    double ph = TWO_PI * u_or[1];
    double ps = TWO_PI * u_or[2];
    frame_from_angles(st, ct, sin(ph), cos(ph), sin(ps), cos(ps), A, B, C);
  } else if (m->orient_kind == ORC_ORIENT_UNIFORM_ANGLES_MC) {
    /* R-N3: theta ~ U[0, pi], phi ~ U[0, 2 pi], psi ~ U[0, 2 pi] exactly as printed */
    double th = PI_ * u_or[0];
    double ph = TWO_PI * u_or[1];
    double ps = TWO_PI * u_or[2];
    frame_from_angles(sin(th), cos(th), sin(ph), cos(ph), sin(ps), cos(ps), A, B, C);
  } else {
    frame_from_angles(sin(m->theta), cos(m->theta), sin(m->phi), cos(m->phi), sin(m->psi),
                      cos(m->psi), A, B, C);
  }
}

/* I(Q) = 1e8 scale <F^2>/<V> S(q) + background  (Eq. 2-4;
 * R-A2, R-A6).  Averages are fixed-node sums (R-A1, R-A9, R-A11). */
double orc_intensity(const orc_model* m, const double Q[3], const double u_or[3], double* env_out) {
  if (m->model == ORC_FLAT) {
    if (env_out) *env_out = m->scale + m->background;
    return m->scale + m->background;
  }
  double A[3], B[3], C[3];
  particle_frame(m, u_or, A, B, C);
  double qA = dot3(Q, A), qB = dot3(Q, B), qC = dot3(Q, C);
  double q2 = dot3(Q, Q);
  double qm = sqrt(q2);

  int n_th = 1, n_ph = 1;
  if (m->orient_kind == ORC_ORIENT_GAUSS_QUAD) { n_th = m->n_or[0]; n_ph = m->n_or[1]; }

  double SF2 = 0.0, SE2 = 0.0, SV = 0.0;
  for (int a = 0; a < m->n_pd[0]; ++a)
    for (int b = 0; b < m->n_pd[1]; ++b) {
      double V, E;
      if (m->model == ORC_POLYMER_MICELLE) (void)orc_micelle_f2(m, 0.0, m->pd_x[0][a], &V, &E);
      else (void)orc_amplitude(m, 0.0, 0.0, 0.0, m->pd_x[0][a], m->pd_x[1][b], &V, &E);
      SV += (m->pd_w[0][a] * m->pd_w[1][b]) * V;
    }
  for (int i = 0; i < n_th; ++i)
    for (int j = 0; j < n_ph; ++j) {
      double qa = qA, qb = qB, qc = qC, w_or = 1.0;
      if (m->orient_kind == ORC_ORIENT_GAUSS_QUAD) {
        /* R-A11: axis tilted by (dtheta_i, dphi_j) about the mean axis, in the
         * mean particle frame: c_ij = (sin dth cos dph, sin dph, cos dth cos dph) */
        double dth = m->or_d[0][i], dph = m->or_d[1][j];
        double lx = sin(dth) * cos(dph), ly = sin(dph), lz = cos(dth) * cos(dph);
        qc = (qA * lx + qB * ly) + qC * lz;
        double r2 = q2 - qc * qc;
        qa = sqrt(r2 > 0.0 ? r2 : 0.0); /* uniaxial models only: Q_AB (Eq. 7) */
        qb = 0.0;
        w_or = m->or_w[0][i] * m->or_w[1][j];
      }
      for (int a = 0; a < m->n_pd[0]; ++a)
        for (int b = 0; b < m->n_pd[1]; ++b) {
          double V, E, F2, E2;
          if (m->model == ORC_POLYMER_MICELLE) {
            F2 = orc_micelle_f2(m, qm, m->pd_x[0][a], &V, &E2);   /* isotropic: |Q| only */
          } else {
            double F = orc_amplitude(m, qa, qb, qc, m->pd_x[0][a], m->pd_x[1][b], &V, &E);
            F2 = F * F;
            E2 = E * E;
          }
          double w = w_or * (m->pd_w[0][a] * m->pd_w[1][b]);
          SF2 += w * F2;
          SE2 += w * E2;
        }
    }
  double S = 1.0;
  if (m->sq_kind == ORC_SQ_HARD_SPHERE_PY) S = orc_py_sq(qm, m->sq_radius_eff, m->sq_volfrac);
  if (m->sq_kind == ORC_SQ_HAYTER_MSA) S = orc_msa_sq(qm, m);
  if (env_out) *env_out = ((1.0e8 * m->scale) * (SE2 / SV)) * S + m->background;
  return ((1.0e8 * m->scale) * (SF2 / SV)) * S + m->background;
}

/* R-N2: the paper's per-event model, Eq. 4 literally: M = A A* / V with the sizes of THIS scattering
 * event, I = 1e8 scale M S(q) + background.  x[k] = relative size of axis k. */
double orc_intensity_event(const orc_model* m, const double Q[3], const double u_or[3], const double x[2],
                           double* env_out) {
  if (m->model == ORC_FLAT) {
    if (env_out) *env_out = m->scale + m->background;
    return m->scale + m->background;
  }
  double A[3], B[3], C[3];
  particle_frame(m, u_or, A, B, C);
  double qA = dot3(Q, A), qB = dot3(Q, B), qC = dot3(Q, C);
  double qm = sqrt(dot3(Q, Q));
  double V, E, F2, E2;
  if (m->model == ORC_POLYMER_MICELLE) {
    F2 = orc_micelle_f2(m, qm, x[0], &V, &E2);
  } else {
    double F = orc_amplitude(m, qA, qB, qC, x[0], x[1], &V, &E);
    F2 = F * F;
    E2 = E * E;
  }
  double S = 1.0;
  if (m->sq_kind == ORC_SQ_HARD_SPHERE_PY) S = orc_py_sq(qm, m->sq_radius_eff, m->sq_volfrac);
  if (m->sq_kind == ORC_SQ_HAYTER_MSA) S = orc_msa_sq(qm, m);
  if (env_out) *env_out = ((1.0e8 * m->scale) * (E2 / V)) * S + m->background;
  return ((1.0e8 * m->scale) * (F2 / V)) * S + m->background;
}

/* R-N1 (Eq. 8): r = mean (1 + rel z), z standard normal by Box-Muller from the two
 * uniforms (words 2k, 2k+1) of Philox block 3 + t, t = 0, 1, ...: "radii and distances are always checked
 * to be positively defined, else a new iteration of the random choice is performed".  After 8 blocks
 * the mean is taken (probability Phi(-1/rel)^8). */
double orc_draw_rel_size(uint64_t seed, uint64_t id, uint32_t exp_index, int k, double rel, int32_t* tries) {
  for (int t = 0; t < 8; ++t) {
    double u4[4];
    draw_block(seed, id, 3u + (uint32_t)t, exp_index, u4);
    double z = sqrt(-2.0 * log(u4[2 * k])) * cos(TWO_PI * u4[2 * k + 1]);
    double x = 1.0 + rel * z;
    if (tries) *tries = t + 1;
    if (x > 0.0) return x;
  }
  return 1.0;
}

/* ------------------------------------------------------------- R-C5 */
/* Ray (o + t d) against the sample volume centred at the origin of the sample
 * frame.  Box: slab test per axis (x, y, z).  Cylinder: axis along y, radius
 * sample_radius, height sample_yh.  Returns 0 on a miss. */
static int intersect_sample(const orc_instrument* ins, const double o[3], const double d[3],
                            double* t_in, double* t_out) {
  double tin = -INFINITY, tout = INFINITY;
  double h[3] = {0.5 * ins->sample_xw, 0.5 * ins->sample_yh, 0.5 * ins->sample_zd};
  int first_axis = 0, last_axis = 2, step = 1;
  if (ins->sample_shape == ORC_SAMPLE_CYL_Y) {
    double a = d[0] * d[0] + d[2] * d[2];
    double b = o[0] * d[0] + o[2] * d[2];
    double c = (o[0] * o[0] + o[2] * o[2]) - ins->sample_radius * ins->sample_radius;
    if (a == 0.0) {
      if (c > 0.0) return 0;
    } else {
      double disc = b * b - a * c;
      if (!(disc > 0.0)) return 0;
      double sq = sqrt(disc);
      double inv_a = 1.0 / a;
      tin = (-b - sq) * inv_a;
      tout = (-b + sq) * inv_a;
    }
    first_axis = 1; last_axis = 1; /* only the y slab remains */
  }
  for (int ax = first_axis; ax <= last_axis; ax += step) {
    if (d[ax] == 0.0) {
      if (fabs(o[ax]) > h[ax]) return 0;
    } else {
      double inv = 1.0 / d[ax];
      double t1 = (-h[ax] - o[ax]) * inv;
      double t2 = (h[ax] - o[ax]) * inv;
      if (t1 > t2) { double tmp = t1; t1 = t2; t2 = tmp; }
      if (t1 > tin) tin = t1;
      if (t2 < tout) tout = t2;
    }
  }
  *t_in = tin;
  *t_out = tout;
  return 1;
}

/* ---------------------------------------------------- R-C2 .. R-C11 */
void orc_trace_one(const orc_instrument* ins, const orc_model* m, uint64_t seed, uint64_t id,
                   uint32_t exp_index, orc_record* rec) {
  memset(rec, 0, sizeof(*rec));
  rec->pixel = -1;
  double* u = rec->u;
  draw_block(seed, id, 0, exp_index, u + 0);

  /* R-C2 source point (flat = uniform), z0 = 0 */
  double x0 = (u[0] - 0.5) * ins->src_xw;
  double y0 = (u[1] - 0.5) * ins->src_yh;
  double z0 = 0.0;
  /* R-C3 direction towards a uniform point of the focus rectangle */
  double xt = (u[2] - 0.5) * ins->focus_xw;
  double yt = (u[3] - 0.5) * ins->focus_yh;
  double zt = ins->focus_z;
  double Dx = xt - x0, Dy = yt - y0, Dz = zt - z0;
  double r2 = (Dx * Dx + Dy * Dy) + Dz * Dz;
  double r = sqrt(r2);
  double inv_r = 1.0 / r;
  double d[3] = {Dx * inv_r, Dy * inv_r, Dz * inv_r};
  double dOmega = (((ins->focus_xw * ins->focus_yh) * d[2]) * inv_r) * inv_r;
  double dlam = ins->lambda_max - ins->lambda_min;
  double dlam_w = dlam > 0.0 ? dlam : 1.0;
  double p0 = ((ins->flux * ((ins->src_xw * ins->src_yh) * 1.0e4)) * dOmega) * dlam_w;
  rec->p0 = p0;

  /* R-C4 slits: straight lines, absorb outside the aperture (edges inclusive) */
  double inv_dz = 1.0 / d[2];
  {
    double s = (ins->slit1_z - z0) * inv_dz;
    double xs = x0 + d[0] * s, ys = y0 + d[1] * s;
    if (fabs(xs) > 0.5 * ins->slit1_xw || fabs(ys) > 0.5 * ins->slit1_yh) { rec->status = ORC_SLIT1; return; }
  }
  {
    double s = (ins->slit2_z - z0) * inv_dz;
    double xs = x0 + d[0] * s, ys = y0 + d[1] * s;
    if (fabs(xs) > 0.5 * ins->slit2_xw || fabs(ys) > 0.5 * ins->slit2_yh) { rec->status = ORC_SLIT2; return; }
  }

  draw_block(seed, id, 1, exp_index, u + 4);
  /* R-L1: position t in [0, 1] of the wavelength inside the band: t = u4 (uniform), or the inverse distribution
   * function of the symmetric triangle, 2 t^2 below the centre and 1 - 2 (1 - t)^2 above it */
  double t_lam = u[4];
  if (ins->lambda_dist == ORC_LAMBDA_TRIANGLE)
    t_lam = (u[4] < 0.5) ? sqrt(0.5 * u[4]) : 1.0 - sqrt(0.5 * (1.0 - u[4]));
  double lambda = ins->lambda_min + t_lam * dlam;
  rec->lambda = lambda;

  /* R-C5 sample intersection in the sample frame (origin at (0,0,sample_z)) */
  double o[3] = {x0, y0, z0 - ins->sample_z};
  double tin, tout;
  if (!intersect_sample(ins, o, d, &tin, &tout)) { rec->status = ORC_MISS_SAMPLE; return; }
  if (tin < 0.0) tin = 0.0;
  if (!(tout > tin)) { rec->status = ORC_MISS_SAMPLE; return; }
  double ell = tout - tin;
  rec->ell = ell;

  /* R-C6 forced single scattering, uniform along the chord */
  double ts = tin + u[5] * ell;
  double rs[3] = {x0 + d[0] * ts, y0 + d[1] * ts, z0 + d[2] * ts};

  /* R-C7 choose |Q| and azimuth */
  double q = ins->q_min + u[6] * (ins->q_max - ins->q_min);
  double chi = TWO_PI * u[7];
  double k = TWO_PI / lambda;
  double inv_k = lambda / TWO_PI;
  double qk = q * inv_k;
  double s = 0.5 * qk; /* sin(theta), |Q| = 2 k sin(theta) */
  rec->q = q;
  if (s >= 1.0) { rec->status = ORC_UNREACHABLE; return; }
  double ss2 = 2.0 * (s * s);              /* 1 - cos(2 theta) */
  double c2 = 1.0 - ss2;                   /* cos(2 theta) */
  double s2 = 2.0 * (s * sqrt(1.0 - s * s)); /* sin(2 theta) */

  /* R-C8 outgoing direction: rotate d by 2 theta at azimuth chi */
  double n = sqrt(d[2] * d[2] + d[0] * d[0]);
  double inv_n = 1.0 / n;
  double e1x = d[2] * inv_n, e1z = -(d[0] * inv_n);       /* e1 = y^ x d^, normalised; e1y = 0 */
  double e2x = d[1] * e1z, e2y = d[2] * e1x - d[0] * e1z, e2z = -(d[1] * e1x); /* e2 = d^ x e1 */
  double sc = sin(chi), cc = cos(chi);
  double tx = cc * e1x + sc * e2x, ty = sc * e2y, tz = cc * e1z + sc * e2z;
  double dp[3] = {c2 * d[0] + s2 * tx, c2 * d[1] + s2 * ty, c2 * d[2] + s2 * tz};
  double Q[3] = {k * (ss2 * d[0] - s2 * tx), k * (ss2 * d[1] - s2 * ty), k * (ss2 * d[2] - s2 * tz)};
  rec->Q[0] = Q[0]; rec->Q[1] = Q[1]; rec->Q[2] = Q[2];

  /* R-C9 detector plane at sample_z + det_dist */
  if (!(dp[2] > 0.0)) { rec->status = ORC_MISS_DET; return; }
  double inv_dpz = 1.0 / dp[2];
  double td = ((ins->sample_z + ins->det_dist) - rs[2]) * inv_dpz;
  double X = rs[0] + dp[0] * td, Y = rs[1] + dp[1] * td;
  double fx = (X + 0.5 * ins->det_xw) * ((double)ins->det_nx / ins->det_xw);
  double fy = (Y + 0.5 * ins->det_yh) * ((double)ins->det_ny / ins->det_yh);
  if (!(fx >= 0.0 && fx < (double)ins->det_nx && fy >= 0.0 && fy < (double)ins->det_ny)) {
    rec->status = ORC_MISS_DET; return;
  }
  int ix = (int)floor(fx), iy = (int)floor(fy);
  rec->pixel = iy * ins->det_nx + ix;

  /* orientation uniforms (draws 8,9,10) only for per-neutron random orientation */
  if ((m->orient_kind == ORC_ORIENT_ISOTROPIC_MC || m->orient_kind == ORC_ORIENT_UNIFORM_ANGLES_MC) &&
      m->model != ORC_FLAT)
    draw_block(seed, id, 2, exp_index, u + 8);

  /* R-C11 attenuation along the path inside the sample */
  double T = 1.0;
  if (ins->mu_abs_2200 != 0.0 || ins->mu_inc != 0.0) {
    double mu = (ins->mu_abs_2200 * lambda) / 1.7982 + ins->mu_inc;
    double o2[3] = {rs[0], rs[1], rs[2] - ins->sample_z};
    double tin2, tout2, ell_out = 0.0;
    if (intersect_sample(ins, o2, dp, &tin2, &tout2) && tout2 > 0.0) ell_out = tout2;
    T = exp(-(mu * (u[5] * ell + ell_out)));
  }

  double env, I;
  rec->pd_x[0] = rec->pd_x[1] = 1.0;
  if ((m->pd_mc[0] || m->pd_mc[1]) && m->model != ORC_FLAT) {
    /* the paper's own size averaging: one size per scattering event (R-N1, R-N2) */
    for (int kk = 0; kk < 2; ++kk)
      if (m->pd_mc[kk]) rec->pd_x[kk] = orc_draw_rel_size(seed, id, exp_index, kk, m->pd_rel[kk], &rec->pd_tries[kk]);
    I = orc_intensity_event(m, Q, u + 8, rec->pd_x, &env);
  } else {
    I = orc_intensity(m, Q, u + 8, &env);
  }
  rec->intensity = I;
  double jac = qk * inv_k;                            /* q / k^2 */
  double qnorm = TWO_PI * (ins->q_max - ins->q_min);  /* 1 / pdf(q, chi) */
  double geo = (p0 * T) * (100.0 * ell);              /* ell in cm: I is per cm */
  rec->weight = ((geo * I) * jac) * qnorm;
  rec->weight_env = ((geo * env) * jac) * qnorm;
  rec->status = ORC_DETECTED;
}

void orc_trace_range(const orc_instrument* ins, const orc_model* m, uint64_t seed, uint64_t first,
                     uint64_t n, uint32_t exp_index, int32_t* pixel, double* weight, double* weight_env,
                     double* q, double* sum_p, double* sum_p2, uint64_t* counts, uint64_t counters[8]) {
  orc_record rec;
  for (uint64_t i = 0; i < n; ++i) {
    orc_trace_one(ins, m, seed, first + i, exp_index, &rec);
    if (pixel) pixel[i] = rec.pixel;
    if (weight) weight[i] = rec.status == ORC_DETECTED ? rec.weight : 0.0;
    if (weight_env) weight_env[i] = rec.status == ORC_DETECTED ? rec.weight_env : 0.0;
    if (q) q[i] = rec.q;
    if (counters) {
      counters[0] += 1;
      switch (rec.status) {
        case ORC_SLIT1: counters[1] += 1; break;
        case ORC_SLIT2: counters[2] += 1; break;
        case ORC_MISS_SAMPLE: counters[3] += 1; break;
        case ORC_UNREACHABLE: counters[4] += 1; break;
        case ORC_MISS_DET: counters[5] += 1; break;
        default: counters[6] += 1; break;
      }
    }
    if (rec.status == ORC_DETECTED) {
      /* R-C14 accumulate in id order */
      if (counts) counts[rec.pixel] += 1;
      if (sum_p) sum_p[rec.pixel] += rec.weight;
      if (sum_p2) sum_p2[rec.pixel] += rec.weight * rec.weight;
    }
  }
}

/* ------------------------------------------------------------- R-R1 */
void orc_reduce_radial(const orc_instrument* ins, const double* sum_p, const double* sum_p2, double launched,
                       double lambda_ref, double q_lo, double q_hi, int32_t n_bins, double* q_out, double* i_out,
                       double* sigma_out, uint64_t* npix_out) {
  double k = TWO_PI / lambda_ref;
  double D = ins->det_dist;
  double px = ins->det_xw / (double)ins->det_nx, py = ins->det_yh / (double)ins->det_ny;
  double a_pix = px * py;
  double scale = (double)n_bins / (q_hi - q_lo);
  for (int b = 0; b < n_bins; ++b) {
    q_out[b] = q_lo + ((double)b + 0.5) * ((q_hi - q_lo) / (double)n_bins);
    i_out[b] = 0.0; sigma_out[b] = 0.0; npix_out[b] = 0;
  }
  /* i_out, sigma_out hold sum P and sum P2 until the end; the solid angles go to a scratch sum per ring */
  double omega[4096];
  if (n_bins > 4096) return;
  for (int b = 0; b < n_bins; ++b) omega[b] = 0.0;
  for (int iy = 0; iy < ins->det_ny; ++iy)
    for (int ix = 0; ix < ins->det_nx; ++ix) {
      double X = ((double)ix + 0.5) * px - 0.5 * ins->det_xw;
      double Y = ((double)iy + 0.5) * py - 0.5 * ins->det_yh;
      double r2 = X * X + Y * Y;
      double two_theta = atan2(sqrt(r2), D);
      double q = (2.0 * k) * sin(0.5 * two_theta);
      if (!(q >= q_lo && q < q_hi)) continue;
      int b = (int)floor((q - q_lo) * scale);
      if (b < 0 || b >= n_bins) continue;
      double d2 = D * D + r2;
      double dOmega = (a_pix * D) / (d2 * sqrt(d2));
      int pix = iy * ins->det_nx + ix;
      i_out[b] += sum_p[pix];
      sigma_out[b] += sum_p2[pix];
      omega[b] += dOmega;
      npix_out[b] += 1;
    }
  for (int b = 0; b < n_bins; ++b) {
    if (npix_out[b] == 0) continue;
    double norm = omega[b] * launched;
    i_out[b] = i_out[b] / norm;
    sigma_out[b] = sqrt(sigma_out[b]) / norm;
  }
}

