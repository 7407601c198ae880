// SAS model intensity I(Q) = 1e8 scale <F^2>/<V> S(q) + background for one detected neutron
// (PAPER.md:37-49 Eq. 1-4, :76-84 Eq. 6-7, :161-163 Eq. 9; DESIGN.md R-A2, R-A9, R-A11, R-A12, R-C12).
// Real = float or double.  The quadrature node tables live in shared memory, one broadcast load per
// node per warp; all Q-independent factors (volumes, contrasts, weights, <V>) were folded into the
// tables by the host (sas_api.cu: build_tables).
#pragma once
#include "sas_types.h"

#ifndef SAS_CYL_UNROLL
#define SAS_CYL_UNROLL 4
#endif

namespace sas {

// 32-node Gauss-Legendre rule on [-1, 1] for the end pieces of the barbell and the capped cylinder (R-M2):
// nodes then weights (summing to 1), uploaded once by the host from its own Jacobi-matrix rule (sas_api.cu)
constexpr int GL_N = 32;
__constant__ double c_gl[2 * GL_N];

constexpr int CYL_UNROLL = SAS_CYL_UNROLL;  // nodes of the phi-tilt loop in flight

template <typename Real>
struct Tables {  // views into the shared-memory table block
  const Real* ta;   // [n_a][TA_W]
  const Real* tb;   // [n_b][TB_W]
  const Real* tab;  // [n_a*n_b][TAB_W]
  const Real* tth;  // [n_th][TOR_W]
  const Real* tph;  // [(n_ph + 1) / 2][2 TOR_W]: pairs of nodes (cyl_quad_row)
};

template <typename Real>
__device__ __forceinline__ Tables<Real> table_views(const Real* base, const ExpParams& P) {
  Tables<Real> t;
  t.ta = base;
  t.tb = t.ta + P.n_a * TA_W;
  t.tab = t.tb + P.n_b * TB_W;
  t.tth = t.tab + P.n_a * P.n_b * TAB_W;
  t.tph = t.tth + P.n_th * TOR_W;
  return t;
}

template <typename Real>
__device__ __forceinline__ Real sq(Real x) { return x * x; }

// One row of the Gaussian-tilt quadrature of a monodisperse cylinder (R-A11): sum over the phi tilts of
// w_j [sinc(Q.c_ij L/2) Lambda(R sqrt(q^2 - (Q.c_ij)^2))]^2 for one theta tilt (Ai = Q.(tilted axis, phi = 0)).
// LC > 0: Lambda is the short polynomial of class LC in t = x^2 / h - 1 (device_math.cuh), t in one FMA.
// The phi-tilt table holds its nodes in pairs, [sin0, sin1, cos0, cos1, w0, w1, 0, 0] per pair (an odd count is
// padded with a node of weight 0): the fp32 row below takes a pair per step in packed arithmetic.
template <typename Real> __device__ __forceinline__ Real tph_sin(const Real* tph, int j) { return tph[(j >> 1) * (2 * TOR_W) + (j & 1)]; }
template <typename Real> __device__ __forceinline__ Real tph_cos(const Real* tph, int j) { return tph[(j >> 1) * (2 * TOR_W) + 2 + (j & 1)]; }
template <typename Real> __device__ __forceinline__ Real tph_w(const Real* tph, int j) { return tph[(j >> 1) * (2 * TOR_W) + 4 + (j & 1)]; }

// fp32: two phi tilts per step (FFMA2 / FMUL2 / FADD2, device_math.cuh); the two partial sums are added at the end
template <int LC>
__device__ __forceinline__ float cyl_quad_row(const float* tph, int n_ph, float Ai, float qB, float hL0, float R20, float q2) {
  const float k = R20 * (float)lambda_class_scale(LC);
  const float nk = -k, tq = fmaf(q2, k, -1.0f);
  float2 row = f2(0.0f);
  const int n_pairs = (n_ph + 1) >> 1;
#pragma unroll CYL_UNROLL / 2
  for (int p = 0; p < n_pairs; ++p) {
    const float4 sc = *reinterpret_cast<const float4*>(tph + p * (2 * TOR_W));
    const float2 w = *reinterpret_cast<const float2*>(tph + p * (2 * TOR_W) + 4);
    const float2 qc = fma2(make_float2(sc.z, sc.w), f2(Ai), mul2(f2(qB), make_float2(sc.x, sc.y)));  // Q . c_ij
    float2 f;
    if (LC > 0) {
      f = mul2(sinc_abs_r2(qc, hL0), lambda1_class2<LC>(fma2(mul2(qc, qc), f2(nk), f2(tq))));
    } else {
      float2 r2 = fma2(mul2(qc, qc), f2(-1.0f), f2(q2));
      r2.x = r2.x > 0.0f ? r2.x : 0.0f;
      r2.y = r2.y > 0.0f ? r2.y : 0.0f;
      f = mul2(sinc_abs_r2(qc, hL0), make_float2(lambda1_x2(r2.x * R20), lambda1_x2(r2.y * R20)));
    }
    row = fma2(w, mul2(f, f), row);
  }
  return row.x + row.y;
}

template <typename Real, int LC>
__device__ __forceinline__ Real cyl_quad_row(const Real* tph, int n_ph, Real Ai, Real qB, Real hL0, Real R20, Real q2) {
  if constexpr (sizeof(Real) == 4) return cyl_quad_row<LC>(tph, n_ph, Ai, qB, hL0, R20, q2);
  const Real k = R20 * (Real)lambda_class_scale(LC);
  const Real nk = -k, tq = fma_r(q2, k, (Real)-1);
  Real row = 0;
#pragma unroll CYL_UNROLL
  for (int j = 0; j < n_ph; ++j) {
    const Real sph = tph_sin(tph, j), cph = tph_cos(tph, j), wph = tph_w(tph, j);
    const Real qc = fma_r(cph, Ai, qB * sph);  // Q . c_ij
    Real f;
    if (LC > 0) {
      f = sinc_abs_r(qc, hL0) * lambda1_class<LC>(fma_r(qc * qc, nk, tq));
    } else {
      Real r2 = fma_r(-qc, qc, q2);
      r2 = r2 > (Real)0 ? r2 : (Real)0;
      f = sinc_abs_r(qc, hL0) * lambda1_x2(r2 * R20);
    }
    row = fma_r(wph, f * f, row);
  }
  return row;
}

// Particle axes A, B, C in the global frame (R-A7): the fixed / mean frame of the experiment, or one random
// orientation per scattering event from draws 8, 9, 10 (Philox block 2): isotropic (R-A3) or the paper's
// printed uniform angles (R-N3).  LIBM: CUDA's fp64 sincos, else the 1e-13 fp64 kernels.
template <bool LIBM, int V>
__device__ __forceinline__ void particle_frame(const ExpParams& P, const PhiloxKeys& keys, uint32_t id_lo, uint32_t id_hi,
                                               uint32_t exp_word, double A[3], double B[3], double C[3]) {
  if (V != V_CYL_QUAD && P.orient_kind >= 2) {
    uint32_t w2[4];
    philox4x32_10(keys, id_lo, id_hi, 2u, exp_word, w2);
    const double u8 = uniform_from_word(w2[0]), u9 = uniform_from_word(w2[1]), u10 = uniform_from_word(w2[2]);
    double ct, st, sp, cp, ss, cs;
    if (P.orient_kind == 3) {  // theta = pi u8
      if (LIBM) sincospi_cw(u8, st, ct); else sincos_2pi(0.5 * u8, st, ct);
    } else {                   // cos(theta) = 1 - 2 u8
      ct = 1.0 - 2.0 * u8;
      st = sqrt(1.0 - ct * ct);
    }
    if (LIBM) {
      // sincospi reduces exactly and has no large-argument path: within 1e-15 of sin/cos(TWO_PI u) as R-A3 writes it
      sincospi_cw(2.0 * u9, sp, cp);
      sincospi_cw(2.0 * u10, ss, cs);
    } else {
      sincos_2pi(u9, sp, cp);
      sincos_2pi(u10, ss, cs);
    }
    const double a0[3] = {ct * cp, ct * sp, -st};
    const double b0[3] = {-sp, cp, 0.0};
    C[0] = st * cp; C[1] = st * sp; C[2] = ct;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      A[i] = fma(cs, a0[i], ss * b0[i]);
      B[i] = fma(cs, b0[i], -(ss * a0[i]));
    }
  } else {
#pragma unroll
    for (int i = 0; i < 3; ++i) { A[i] = P.frame[i]; B[i] = P.frame[3 + i]; C[i] = P.frame[6 + i]; }
  }
}

// R-N1 (Eq. 8): relative size of polydisperse length k of this scattering event,
// 1 + rel z with z standard normal by Box-Muller from words 2k, 2k+1 of Philox block 3 + t; the draw is
// repeated (t = 1, 2, ...) while the size is not positive; after 8 blocks the mean is taken.
__device__ __forceinline__ double draw_rel_size(const PhiloxKeys& keys, uint32_t id_lo, uint32_t id_hi, uint32_t exp_word,
                                                int k, double rel) {
  for (uint32_t t = 0; t < 8u; ++t) {
    uint32_t w[4];
    philox4x32_10(keys, id_lo, id_hi, 3u + t, exp_word, w);
    const double ua = uniform_from_word(k ? w[2] : w[0]), ub = uniform_from_word(k ? w[3] : w[1]);
    double sb, cb;
    sincos_cw(6.283185307179586 * ub, sb, cb);
    const double x = 1.0 + rel * (sqrt(-2.0 * log(ua)) * cb);
    if (x > 0.0) return x;
  }
  return 1.0;
}

// Amplitude F and normalising volume of ONE particle with relative sizes x0, x1 (R-A12 says which lengths
// they scale), straight from the descriptor's numbers in fp64: Eq. 1 integrated over the body (R-C12; the
// NEXT-2 bodies: box -> three sincs, core-shell cylinder -> two sinc x Lambda terms, ellipsoid of revolution
// -> Phi at sqrt(Re^2 Q_AB^2 + Rp^2 Q_C^2)).
template <int V>
__device__ __forceinline__ double particle_amplitude(const ExpParams& P, double q, double qA, double qB, double qC,
                                                     double x0, double x1, double& Vol) {
  const double FOUR_PI_3 = 4.1887902047863905, PI_D = 3.141592653589793;
  const double s0 = P.ev_sld[0], s1 = P.ev_sld[1];
  double F = 1.0;
  Vol = 1.0;
  if (V == V_SPHERE) {
    const double R = P.msize[0] * x0;
    Vol = FOUR_PI_3 * ((R * R) * R);
    F = (s0 * Vol) * sphere_phi(q * R);
  } else if (V == V_CS_SPHERE) {
    const double Rc = P.msize[0] * x0, Rt = Rc + P.msize[1] * x1;
    const double Vc = FOUR_PI_3 * ((Rc * Rc) * Rc);
    Vol = FOUR_PI_3 * ((Rt * Rt) * Rt);
    F = fma((s0 - s1) * Vc, sphere_phi(q * Rc), (s1 * Vol) * sphere_phi(q * Rt));
  } else if (V == V_CYL) {
    const double R = P.msize[0] * x0, L = P.msize[1] * x1;
    Vol = (PI_D * (R * R)) * L;
    F = ((s0 * Vol) * sinc_r(qC * (0.5 * L))) * lambda1_r(sqrt(fma(qA, qA, qB * qB)) * R);
  } else if (V == V_TRIAX) {
    const double a = P.msize[0] * x0, b = P.msize[1] * x0, c = P.msize[2] * x0;
    Vol = FOUR_PI_3 * ((a * b) * c);
    const double ua = a * qA, ub = b * qB, uc = c * qC;
    F = (s0 * Vol) * sphere_phi(sqrt(fma(ua, ua, fma(ub, ub, uc * uc))));
  } else if (V == V_CS_TRIAX) {
    const double a = P.msize[0] * x0, b = P.msize[1] * x0, c = P.msize[2] * x0, t = P.msize[3] * x1;
    const double at = a + t, bt = b + t, ct = c + t;
    const double Vc = FOUR_PI_3 * ((a * b) * c);
    Vol = FOUR_PI_3 * ((at * bt) * ct);
    const double ua = a * qA, ub = b * qB, uc = c * qC, va = at * qA, vb = bt * qB, vc = ct * qC;
    F = fma((s0 - s1) * Vc, sphere_phi(sqrt(fma(ua, ua, fma(ub, ub, uc * uc)))),
            (s1 * Vol) * sphere_phi(sqrt(fma(va, va, fma(vb, vb, vc * vc)))));
  } else if (V == V_PARA) {
    const double a = P.msize[0] * x0, b = P.msize[1] * x0, c = P.msize[2] * x0;
    Vol = (a * b) * c;
    F = (s0 * Vol) * ((sinc_r(qA * (0.5 * a)) * sinc_r(qB * (0.5 * b))) * sinc_r(qC * (0.5 * c)));
  } else if (V == V_HOLLOW_PRISM) {
    // R-M5: contrast in thin walls on the six faces: F = 2 sld t [bc cos(qA a/2) sinc_b sinc_c + cyclic]
    const double a = P.msize[0] * x0, b = P.msize[1] * x0, c = P.msize[2] * x0, t = P.msize[3];
    double sa, ca, sb, cb, sc, cc;
    const double xa = qA * (0.5 * a), xb = qB * (0.5 * b), xc = qC * (0.5 * c);
    sincos_d(xa, sa, ca);
    sincos_d(xb, sb, cb);
    sincos_d(xc, sc, cc);
    sa = xa == 0.0 ? 1.0 : sa / xa;
    sb = xb == 0.0 ? 1.0 : sb / xb;
    sc = xc == 0.0 ? 1.0 : sc / xc;
    const double faces = fma((b * c) * ca, sb * sc, fma((a * c) * cb, sa * sc, ((a * b) * cc) * (sa * sb)));
    Vol = t * (2.0 * fma(a, b, fma(b, c, c * a)));
    F = (s0 * t) * (2.0 * faces);
  } else if (V == V_CS_CYL) {
    const double R = P.msize[0] * x0, L = P.msize[1] * x1, t = P.msize[2];
    const double Rt = R + t, Lt = L + 2.0 * t;
    const double Vc = (PI_D * (R * R)) * L;
    Vol = (PI_D * (Rt * Rt)) * Lt;
    const double qab = sqrt(fma(qA, qA, qB * qB));
    F = fma(((s0 - s1) * Vc) * sinc_r(qC * (0.5 * L)), lambda1_r(qab * R),
            ((s1 * Vol) * sinc_r(qC * (0.5 * Lt))) * lambda1_r(qab * Rt));
  } else if (V == V_ELL_CYL) {
    const double a = P.msize[0] * x0, b = P.msize[1] * x0, L = P.msize[2] * x1;
    Vol = (PI_D * (a * b)) * L;
    const double ua = a * qA, ub = b * qB;
    F = ((s0 * Vol) * sinc_r(qC * (0.5 * L))) * lambda1_r(sqrt(fma(ua, ua, ub * ub)));
  } else if (V == V_HOLLOW_CYL) {
    const double Ri = P.msize[0] * x0, L = P.msize[1] * x1, Ro = Ri + P.msize[2];
    const double Vo = (PI_D * (Ro * Ro)) * L, Vi = (PI_D * (Ri * Ri)) * L;
    const double qab = sqrt(fma(qA, qA, qB * qB));
    Vol = Vo - Vi;
    F = (s0 * sinc_r(qC * (0.5 * L))) * fma(Vo, lambda1_r(qab * Ro), -(Vi * lambda1_r(qab * Ri)));
  } else if (V == V_CS_ELL) {
    const double Re = P.msize[0] * x0, Rp = P.msize[1] * x1, Ret = Re + P.msize[2], Rpt = Rp + P.msize[2];
    const double Vc = FOUR_PI_3 * ((Re * Re) * Rp);
    Vol = FOUR_PI_3 * ((Ret * Ret) * Rpt);
    const double qab2 = fma(qA, qA, qB * qB), uc = Rp * qC, ut = Rpt * qC;
    F = fma((s0 - s1) * Vc, sphere_phi(sqrt(fma(Re * Re, qab2, uc * uc))),
            (s1 * Vol) * sphere_phi(sqrt(fma(Ret * Ret, qab2, ut * ut))));
  } else if (V == V_BARBELL || V == V_CAPPED) {
    // R-M2: cylinder (R, L) along C plus two sphere pieces z in [L/2, zc + Rb]; Eq. 1 slice by slice: a slice is a
    // disc pi rho^2 Lambda(Q_AB rho), the two pieces at +-z give 2 cos(Q_C z)
    const double R = P.msize[0] * x0, L = P.msize[1] * x1, Rb = P.msize[2];
    const double h = sqrt(fmax(Rb * Rb - R * R, 0.0));
    const double zc = V == V_BARBELL ? 0.5 * L + h : 0.5 * L - h;
    const double z0 = 0.5 * L, z1 = zc + Rb;
    const double half = 0.5 * (z1 - z0), mid = 0.5 * (z1 + z0);
    const double qab2 = fma(qA, qA, qB * qB), qab = sqrt(qab2);
    double sum = 0.0;
#pragma unroll 1
    for (int i = 0; i < GL_N; ++i) {
      const double z = fma(half, c_gl[i], mid);
      const double dz = z - zc;
      const double rho2 = fmax(Rb * Rb - dz * dz, 0.0);
      double sz, cz;
      sincos_d(qC * z, sz, cz);
      sum = fma(c_gl[GL_N + i], ((PI_D * rho2) * lambda1_sq(qab2 * rho2)) * cz, sum);
    }
    const double pz = z1 - zc, qz = z0 - zc;
    const double Vcyl = (PI_D * (R * R)) * L;
    Vol = Vcyl + 2.0 * (PI_D * ((Rb * Rb) * (z1 - z0) - (((pz * pz) * pz) - ((qz * qz) * qz)) / 3.0));
    // the weights sum to 1: the rule's (z1 - z0)/2 x 2 becomes (z1 - z0); two end pieces
    F = s0 * fma((Vcyl * sinc_r(qC * (0.5 * L))), lambda1_r(qab * R), 2.0 * ((z1 - z0) * sum));
  } else if (V == V_ELL) {
    const double Re = P.msize[0] * x0, Rp = P.msize[1] * x1;
    Vol = FOUR_PI_3 * ((Re * Re) * Rp);
    const double uc = Rp * qC;
    F = (s0 * Vol) * sphere_phi(sqrt(fma(Re * Re, fma(qA, qA, qB * qB), uc * uc)));
  }
  return F;
}

// R-M4, polymer micelle (Pedersen & Gerstenberg 1996): x = (q R_g)^2; Debye function D = 2 (e^-x - 1 + x) / x^2 and
// end-attached chain amplitude psi = (1 - e^-x) / x through expm1 (no cancellation at small x: with
// e = expm1(-x), psi = -e / x and D = 2 (e + x) / x^2 = 2 (1 - psi) / x, the latter by its series below x = 0.1).
__device__ __forceinline__ void chain_terms(double x, double& D, double& psi) {
  if (x < 0.1) {
    // sum_k (-x)^k / (k + 1)! and sum_k 2 (-x)^k / (k + 2)!, twelve terms: below 1e-19 at x = 0.1
    double sp = 0.0, sd = 0.0, tp = 1.0, td = 1.0;
#pragma unroll
    for (int k = 0; k < 12; ++k) {
      sp += tp; sd += td;
      tp *= -x / (double)(k + 2);
      td *= -x / (double)(k + 3);
    }
    psi = sp; D = sd;
    return;
  }
  const double e = expm1(-x);
  psi = -e / x;
  D = (2.0 * (e + x)) / (x * x);
}
// |F|^2 of one micelle with core radius msize[0] x0 (not a perfect square: the chains' self term is the Debye
// function) and its normalising volume V_core + N V_chain
__device__ __forceinline__ double micelle_f2(const ExpParams& P, double q, double x0, double& Vol) {
  const double FOUR_PI_3 = 4.1887902047863905;
  const double R = P.msize[0] * x0, Rg = P.msize[1], Vc = P.msize[2], N = P.msize[3];
  const double Vcore = FOUR_PI_3 * ((R * R) * R);
  const double Bs = P.ev_sld[0] * Vcore, bc = P.ev_sld[1] * Vc;
  const double qg = q * Rg;
  double D, psi;
  chain_terms(qg * qg, D, psi);
  const double phi = sphere_phi(q * R);
  const double ps = psi * sinc_r(q * (R + Rg));
  Vol = fma(N, Vc, Vcore);
  const double bb = bc * bc;
  return fma((2.0 * N) * (Bs * bc), phi * ps, fma((N * (N - 1.0)) * bb, ps * ps, fma(N * bb, D, (Bs * Bs) * (phi * phi))));
}
// |F|^2 and volume of any variant
template <int V>
__device__ __forceinline__ double particle_f2(const ExpParams& P, double q, double qA, double qB, double qC, double x0,
                                              double x1, double& Vol) {
  if (V == V_MICELLE) return micelle_f2(P, q, x0, Vol);
  const double F = particle_amplitude<V>(P, q, qA, qB, qC, x0, x1, Vol);
  return F * F;
}

// R-S2, Hayter-Penfold MSA: S = 1 / |Qhat(K)|^2, K = 2 q R_eff, Qhat = 1 - 12 eta [int_0^1 Q e^{iKx} dx + D' e^{iK}/(k - iK)];
// the core integral is the 64-node Gauss-Legendre sum sum_j c_j e^{iK x_j}, c_j = 12 eta w_j Q(x_j).  The nodes of
// the rule lie in pairs 1/2 +- y_j, so the sum is regrouped exactly as
//   e^{iK/2} sum_{j<32} [ (c_j+ + c_j-) cos(K y_j) + i (c_j+ - c_j-) sin(K y_j) ]:
// 32 sine/cosine pairs per detected neutron instead of 64, arguments half as large; sin K and cos K of the tail term
// follow from the same sin, cos of K/2.  The host tabulates y_j and the two coefficient rows in fp64 (global memory:
// 800 B that every detected neutron of the experiment reads).  Out of line: one call per detected neutron, and the
// kernels of the other structure factors must not carry its registers.
constexpr int MSA_N = 64;      // nodes of the rule
constexpr int MSA_H = MSA_N / 2;  // node pairs = table rows
// Offered for the globular models (sphere family, ellipsoids, micelle) only: an out-of-line call in a kernel costs
// that kernel's every workload 1-3 % through register allocation (measured on the per-event cylinder and the
// barbell), and a sphere-sphere structure factor has no meaning for rods and plates anyway (the host refuses it).
__host__ __device__ constexpr bool msa_offered(int V) {
  return V == V_SPHERE || V == V_CS_SPHERE || V == V_TRIAX || V == V_CS_TRIAX || V == V_ELL || V == V_CS_ELL || V == V_MICELLE;
}
__device__ __noinline__ double msa_sq(const double* __restrict__ t, double q) {
  const double eD = t[3 * MSA_H], k = t[3 * MSA_H + 1], K = q * t[3 * MSA_H + 2];
  double ec = 0.0, os = 0.0;
#pragma unroll 4
  for (int j = 0; j < MSA_H; ++j) {
    double s, c;
    sincos_cw(K * t[j], s, c);
    ec = fma(t[MSA_H + j], c, ec);
    os = fma(t[2 * MSA_H + j], s, os);
  }
  double sh, ch;
  sincos_cw(0.5 * K, sh, ch);
  double re = fma(ch, ec, -(sh * os)), im = fma(sh, ec, ch * os);   // e^{iK/2} (ec + i os)
  const double sK = 2.0 * (sh * ch), cK = (ch - sh) * (ch + sh);
  const double den = fma(k, k, K * K);
  re = 1.0 - fma(eD, fma(k, cK, -(K * sK)) / den, re);
  im = -fma(eD, fma(k, sK, K * cK) / den, im);
  return 1.0 / fma(re, re, im * im);
}

// R-N2: the paper's per-event model, Eq. 4 with the sizes of THIS scattering event:
// I = 1e8 scale F(r)^2 / V(r) S(q) + background, one fp64 evaluation per detected neutron.
// (compiled into kernels of its own, trace_kernel<double, V, true>: in the same kernel as the fixed-node
// path it cost that path 3-6 % through register allocation and code layout)
template <int V>
__device__ __forceinline__ double eval_intensity_event(const ExpParams& P, const PhiloxKeys& keys, uint32_t id_lo,
                                                       uint32_t id_hi, uint32_t exp_word, double Qx, double Qy, double Qz) {
  if (V == V_FLAT) return P.flat_I;
  const double x0 = P.pd_mc[0] ? draw_rel_size(keys, id_lo, id_hi, exp_word, 0, P.pd_rel[0]) : 1.0;
  const double x1 = P.pd_mc[1] ? draw_rel_size(keys, id_lo, id_hi, exp_word, 1, P.pd_rel[1]) : 1.0;
  const double q = sqrt(fma(Qx, Qx, fma(Qy, Qy, Qz * Qz)));
  double qA = 0, qB = 0, qC = 0;
  if (V >= 2 && V != V_MICELLE) {
    double A[3], B[3], C[3];
    particle_frame<true, V>(P, keys, id_lo, id_hi, exp_word, A, B, C);
    qA = fma(Qx, A[0], fma(Qy, A[1], Qz * A[2]));
    qB = fma(Qx, B[0], fma(Qy, B[1], Qz * B[2]));
    qC = fma(Qx, C[0], fma(Qy, C[1], Qz * C[2]));
  }
  double Vol;
  const double F2 = particle_f2<V>(P, q, qA, qB, qC, x0, x1, Vol);
  double S = 1.0;
  if (P.sq_kind == 1) S = py_sq<double>(q, P.py);
  if constexpr (msa_offered(V)) if (P.sq_kind == 2) S = msa_sq(P.msa_tab, q);
  return fma((P.ev_scale * (F2 / Vol)), S, P.background);
}

// Fixed-node average of the NEXT-2 models: the plain double sum over the (a, b) nodes of F^2, in fp64
// (tables: node value and weight only).  <V> is in P.norm.
template <typename Real, int V>
__device__ __forceinline__ double eval_intensity_generic(const ExpParams& P, const Real* tab_base, const PhiloxKeys& keys,
                                                         uint32_t id_lo, uint32_t id_hi, uint32_t exp_word, double Qx,
                                                         double Qy, double Qz) {
  const Real* ta = tab_base;
  const Real* tb = ta + P.n_a * TA_W;
  const double q = sqrt(fma(Qx, Qx, fma(Qy, Qy, Qz * Qz)));
  double qA = 0, qB = 0, qC = 0;
  if (V != V_MICELLE) {   // the micelle is isotropic: |Q| only
    double A[3], B[3], C[3];
    particle_frame<true, V>(P, keys, id_lo, id_hi, exp_word, A, B, C);
    qA = fma(Qx, A[0], fma(Qy, A[1], Qz * A[2]));
    qB = fma(Qx, B[0], fma(Qy, B[1], Qz * B[2]));
    qC = fma(Qx, C[0], fma(Qy, C[1], Qz * C[2]));
  }
  double acc = 0.0;
  for (int a = 0; a < P.n_a; ++a) {
    double inner = 0.0;
    for (int b = 0; b < P.n_b; ++b) {
      double Vol;
      const double F2 = particle_f2<V>(P, q, qA, qB, qC, (double)ta[a * TA_W], (double)tb[b * TB_W], Vol);
      inner = fma((double)tb[b * TB_W + 2], F2, inner);
    }
    acc = fma((double)ta[a * TA_W + 2], inner, acc);
  }
  double S = 1.0;
  if (P.sq_kind == 1) S = py_sq<double>(q, P.py);
  if constexpr (msa_offered(V)) if (P.sq_kind == 2) S = msa_sq(P.msa_tab, q);
  return fma(P.norm * acc, S, P.background);
}

// fp64 node loop of the polydisperse sphere: w (drho V)^2 Phi(u)^2 = [16 pi^2 drho^2 w] (sin u - u cos u)^2 / q^6,
// u = q R: the bracket is the node's fourth table entry and 1 / q^6 multiplies the sum once, so the loop has no
// division; sin u - u cos u is formed without cancellation at any u (device_math.cuh: sin_minus_ucos).  u < 1e6
// (sas_set_model).  Out of line: inlined, its registers cost the one-evaluation kernels (c0, c4) 2 %.
__device__ __forceinline__ void lds_f64x2(uint32_t addr, double& x, double& y) {
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "r"(addr));
}
// (ta: shared-window address of the node table {R, -, w (drho V)^2, 16 pi^2 drho^2 w} in doubles)
__device__ __noinline__ double sphere_nodes_fp64(uint32_t ta, int n_a, double qd, double q2d) {
  const double iq2 = 1.0 / q2d;
  double direct = 0.0;
#pragma unroll 4
  for (int a = 0; a < n_a; ++a) {
    double R, unused, w_small, w_direct;
    lds_f64x2(ta + 32u * (uint32_t)a, R, unused);
    lds_f64x2(ta + 32u * (uint32_t)a + 16u, w_small, w_direct);
    const double d = sin_minus_ucos(qd * R);
    direct = fma(w_direct, d * d, direct);
  }
  return direct * ((iq2 * iq2) * iq2);
}

// Model table meaning (host: fill_model).  Lengths that multiply a projection of Q are stored as a
// (hi, lo) pair: in the fp32 path hi = float(L), lo = float(L - hi); in the fp64 path hi = L, lo = 0.
//  sphere              ta = {R_hi, R_lo, w_a (drho V_a)^2}
//  core-shell sphere   ta = {Rc_hi, Rc_lo, (drho_c-drho_s) Vc_a, w_a}; tb = {-, w_b};
//                      tab = {Rt_hi, Rt_lo, drho_s Vt_ab}
//  cylinder            ta = {R_hi, R_lo, w_a (drho pi R_a^2)^2}; tb = {L_b/2 hi, lo, w_b L_b^2}
//  triaxial            ta = {x_hi, x_lo, w_a (drho V_a)^2}
//  core-shell triaxial ta = {x_hi, x_lo, (drho_c-drho_s) Vc_a, w_a}; tb = {t_b, w_b, t_b^2};
//                      tab = {drho_s Vt_ab, 2 x_a t_b}
// V is the kernel variant (sas_types.h): the model, with the cylinder split into its Gaussian tilt
// quadrature and its fixed / per-neutron random orientation forms.  One kernel is compiled per variant so
// that a launch carries the code of its own model only (instruction-cache footprint).
template <typename Real, int V>
__device__ __forceinline__ Real eval_intensity(const ExpParams& P, const Real* tab_base, const PhiloxKeys& keys,
                                               uint32_t id_lo, uint32_t id_hi, uint32_t exp_word, double Qx,
                                               double Qy, double Qz) {
  if (V == V_FLAT) return (Real)P.flat_I;
  if (V >= V_PARA) return (Real)eval_intensity_generic<Real, V>(P, tab_base, keys, id_lo, id_hi, exp_word, Qx, Qy, Qz);
  const Tables<Real> T = table_views(tab_base, P);
  constexpr int model = (V == V_CYL_QUAD) ? 2 : (V >= V_PARA ? 5 : V);
  // |Q| and the projections of Q on the particle axes (Eq. 6) in fp64: they feed the phases
  const double q2d = fma(Qx, Qx, fma(Qy, Qy, Qz * Qz));
  const double qd = sqrt(q2d);
  double qAd = 0, qBd = 0, qCd = 0;
  if (model >= 2) {
    double A[3], B[3], C[3];
    particle_frame<sizeof(Real) == 8, V>(P, keys, id_lo, id_hi, exp_word, A, B, C);
    qAd = fma(Qx, A[0], fma(Qy, A[1], Qz * A[2]));
    qBd = fma(Qx, B[0], fma(Qy, B[1], Qz * B[2]));
    qCd = fma(Qx, C[0], fma(Qy, C[1], Qz * C[2]));
  }
  const Real q = (Real)qd, q2 = (Real)q2d;

  Real acc = 0;
  switch (model) {
    case 0: {  // sphere
      if (sizeof(Real) == 8 && P.n_a > 1) {
        acc = (Real)sphere_nodes_fp64((uint32_t)__cvta_generic_to_shared(T.ta), P.n_a, qd, q2d);
      } else if (sizeof(Real) == 4 && P.n_a > 1) {
        // fp32 node loop: w (drho V)^2 Phi(u)^2 = [16 pi^2 drho^2 w] (sin u - u cos u)^2 / q^6: the bracket is the
        // node's fourth table entry, 1 / q^6 multiplies the sum once (no reciprocal and no u^-3 per node)
        // (scalar on purpose: a packed loop, two nodes per FFMA2, is 2.4 % slower here -- a packed operation needs both
        // FMA pipes at once and the producers' IMAD.WIDE stream holds the heavy one 63 % of the time)
        const Proj<float> qp = make_proj<float>(qd);
        float direct = 0.0f;
        for (int a = 0; a < P.n_a; ++a) {
          const float* r = reinterpret_cast<const float*>(T.ta) + a * TA_W;
          const Phase<float> ph = phase_mul(qp, r[0], r[1]);
          const float d = sin_minus_ucos_abs(ph.hi, ph.lo);
          direct = fmaf(r[3], d * d, direct);
        }
        const double iq2 = 1.0 / q2d;
        acc = (Real)((double)direct * ((iq2 * iq2) * iq2));
      } else {
        const Proj<Real> qp = make_proj<Real>(qd);
        for (int a = 0; a < P.n_a; ++a) {
          const Real* r = T.ta + a * TA_W;
          const Real ph = sphere_phi_abs_ph(phase_mul(qp, r[0], r[1]));
          acc = fma_r(r[2], ph * ph, acc);
        }
      }
    } break;
    case 1: {  // core-shell sphere
      const Proj<Real> qp = make_proj<Real>(qd);
      for (int a = 0; a < P.n_a; ++a) {
        const Real* ra = T.ta + a * TA_W;
        const Real fc = ra[2] * sphere_phi_ph(phase_mul(qp, ra[0], ra[1]));
        Real inner = 0;
        for (int b = 0; b < P.n_b; ++b) {
          const Real* pr = T.tab + (a * P.n_b + b) * TAB_W;
          const Real F = fma_r(pr[2], sphere_phi_ph(phase_mul(qp, pr[0], pr[1])), fc);
          inner = fma_r(T.tb[b * TB_W + 1], F * F, inner);
        }
        acc = fma_r(ra[3], inner, acc);
      }
    } break;
    case 2: {  // cylinder: separable in (R, L) for a given axis direction
      if (V == V_CYL_QUAD) {
        // Gaussian tilt quadrature (R-A11): n_th x n_ph axis directions about the mean axis, plain Real.
        // Lambda is evaluated from x^2 = R^2 (q^2 - qc^2): no square root below x = 8.
        const Real qA = (Real)qAd, qB = (Real)qBd, qC = (Real)qCd;
        const bool mono = (P.n_a == 1) && (P.n_b == 1);
        const Real hL0 = T.tb[0], cL0 = T.tb[2], R20 = T.ta[3], cR0 = T.ta[2];
        for (int i = 0; i < P.n_th; ++i) {
          const Real sth = T.tth[i * TOR_W + 0], cth = T.tth[i * TOR_W + 1], wth = T.tth[i * TOR_W + 2];
          const Real Ai = fma_r(qA, sth, qC * cth);
          Real row = 0;
          if (mono) {
            // lam_class: the host bounded x^2 = (q R)^2 for this experiment, so Lambda is one short
            // polynomial without a range test (0: no bound below 64)
            switch (P.lam_small) {
              case 4: row = cyl_quad_row<Real, 4>(T.tph, P.n_ph, Ai, qB, hL0, R20, q2); break;
              case 3: row = cyl_quad_row<Real, 3>(T.tph, P.n_ph, Ai, qB, hL0, R20, q2); break;
              case 2: row = cyl_quad_row<Real, 2>(T.tph, P.n_ph, Ai, qB, hL0, R20, q2); break;
              case 1: row = cyl_quad_row<Real, 1>(T.tph, P.n_ph, Ai, qB, hL0, R20, q2); break;
              default: row = cyl_quad_row<Real, 0>(T.tph, P.n_ph, Ai, qB, hL0, R20, q2); break;
            }
            row *= cL0 * cR0;
          } else {
            for (int j = 0; j < P.n_ph; ++j) {
              const Real sph = tph_sin(T.tph, j), cph = tph_cos(T.tph, j), wph = tph_w(T.tph, j);
              const Real qc = fma_r(cph, Ai, qB * sph);
              Real r2 = fma_r(-qc, qc, q2);
              r2 = r2 > (Real)0 ? r2 : (Real)0;
              Real SL = 0, SR = 0;
              for (int b = 0; b < P.n_b; ++b) {
                const Real sc = sinc_r(qc * T.tb[b * TB_W + 0]);
                SL = fma_r(T.tb[b * TB_W + 2], sc * sc, SL);
              }
              for (int a = 0; a < P.n_a; ++a) {
                const Real la = lambda1_x2(r2 * T.ta[a * TA_W + 3]);
                SR = fma_r(T.ta[a * TA_W + 2], la * la, SR);
              }
              row = fma_r(wph, SL * SR, row);
            }
          }
          acc = fma_r(wth, row, acc);
        }
      } else {
        const Proj<Real> qcp = make_proj<Real>(qCd);
        const Proj<Real> qabp = make_proj<Real>(sqrt(fma(qAd, qAd, qBd * qBd)));
        Real SL = 0, SR = 0;
        for (int b = 0; b < P.n_b; ++b) {
          const Real* r = T.tb + b * TB_W;
          const Real sc = sinc_ph(phase_mul(qcp, r[0], r[1]));
          SL = fma_r(r[2], sc * sc, SL);
        }
        for (int a = 0; a < P.n_a; ++a) {
          const Real* r = T.ta + a * TA_W;
          const Real la = lambda1_ph(phase_mul(qabp, r[0], r[1]));
          SR = fma_r(r[2], la * la, SR);
        }
        acc = SL * SR;
      }
    } break;
    case 3: {  // triaxial ellipsoid: common size scale x_a (R-A12)
      const double ua = P.msize[0] * qAd, ub = P.msize[1] * qBd, uc = P.msize[2] * qCd;
      const Proj<Real> U0 = make_proj<Real>(sqrt(fma(ua, ua, fma(ub, ub, uc * uc))));
      for (int a = 0; a < P.n_a; ++a) {
        const Real* r = T.ta + a * TA_W;
        const Real ph = sphere_phi_abs_ph(phase_mul(U0, r[0], r[1]));
        acc = fma_r(r[2], ph * ph, acc);
      }
    } break;
    case 4: {  // core-shell triaxial ellipsoid
      const double ma = P.msize[0], mb = P.msize[1], mc = P.msize[2];
      const double qa2 = qAd * qAd, qb2 = qBd * qBd, qc2 = qCd * qCd;
      const double U02d = fma(ma * ma, qa2, fma(mb * mb, qb2, (mc * mc) * qc2));
      const Proj<Real> U0 = make_proj<Real>(sqrt(U02d));
      const Real U02 = (Real)U02d;
      const Real Wm = (Real)fma(ma, qa2, fma(mb, qb2, mc * qc2));
      const Real qq2 = (Real)((qa2 + qb2) + qc2);
      for (int a = 0; a < P.n_a; ++a) {
        const Real* ra = T.ta + a * TA_W;
        const Real fc = ra[2] * sphere_phi_ph(phase_mul(U0, ra[0], ra[1]));
        const Real xa = ra[0] + ra[1];
        const Real xa2U = (xa * xa) * U02;
        Real inner = 0;
        int b = 0;
        if constexpr (sizeof(Real) == 4) {
          // fp32: two shell nodes per step in packed arithmetic (device_math.cuh); the unified kernel's node loop is
          // short of issue slots, not of FMA-pipe time
          const float* tab = reinterpret_cast<const float*>(T.tab) + a * P.n_b * TAB_W;
          const float* tb = reinterpret_cast<const float*>(T.tb);
          float2 inner2 = f2(0.0f);
          for (; b + 1 < P.n_b; b += 2) {
            const float2 p0 = *reinterpret_cast<const float2*>(tab + b * TAB_W);
            const float2 p1 = *reinterpret_cast<const float2*>(tab + (b + 1) * TAB_W);
            const float4 r0 = *reinterpret_cast<const float4*>(tb + b * TB_W);
            const float4 r1 = *reinterpret_cast<const float4*>(tb + (b + 1) * TB_W);
            const float2 ut2 = fma2(make_float2(r0.z, r1.z), f2((float)qq2), fma2(make_float2(p0.y, p1.y), f2((float)Wm), f2((float)xa2U)));
            const float2 phi = sphere_phi2(make_float2(sqrt_fast(ut2.x), sqrt_fast(ut2.y)));
            const float2 F = fma2(make_float2(p0.x, p1.x), phi, f2((float)fc));
            inner2 = fma2(make_float2(r0.y, r1.y), mul2(F, F), inner2);
          }
          inner = (Real)(inner2.x + inner2.y);
        }
        for (; b < P.n_b; ++b) {
          const Real* pr = T.tab + (a * P.n_b + b) * TAB_W;
          const Real* rb = T.tb + b * TB_W;
          // u_t^2 = sum ((x a_k + t) Q_k)^2 = x^2 U0^2 + 2 x t W + t^2 q^2
          const Real ut2 = fma_r(rb[2], qq2, fma_r(pr[1], Wm, xa2U));
          const Real F = fma_r(pr[0], sphere_phi(sqrt_r(ut2)), fc);
          inner = fma_r(rb[1], F * F, inner);
        }
        acc = fma_r(ra[3], inner, acc);
      }
    } break;
    default: break;
  }
  Real S = 1;
  if (P.sq_kind == 1) S = py_sq<Real>(q, P.py);
  if constexpr (msa_offered(V)) if (P.sq_kind == 2) S = (Real)msa_sq(P.msa_tab, qd);
  return fma_r((Real)P.norm * acc, S, (Real)P.background);
}

}  // namespace sas
