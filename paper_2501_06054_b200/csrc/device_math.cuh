// Device math of the CUDA tracer: Philox4x32-10, sin/cos, sphere Phi, sinc, Lambda = 2J1(x)/x and
// Percus-Yevick S(q) in fp32 and fp64.  The translation unit is compiled with -fmad=false so that
// the fp64 geometry keeps one rounding per written operation (DESIGN.md R-C0); everything here that
// wants a fused multiply-add says so with fmaf()/fma().
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "coeffs_generated.h"
#include "j1_f64_generated.h"

namespace sas {

// ---------------------------------------------------------------- Philox4x32-10 (DESIGN.md R-B)
struct PhiloxKeys {  // the ten round keys are the same for every neutron of a launch
  uint32_t k0[10], k1[10];
};

__host__ __device__ inline void philox_make_keys(uint64_t seed, PhiloxKeys& pk) {
  uint32_t a = (uint32_t)seed, b = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) {
    pk.k0[r] = a;
    pk.k1[r] = b;
    a += 0x9E3779B9u;
    b += 0xBB67AE85u;
  }
}

// 32 x 32 -> 64-bit product as ONE instruction (IMAD.WIDE.U32: 4 clocks of the heavy FMA pipe, one issue slot).
// Written as mul.wide.u32 because ptxas otherwise may split a __umulhi/mul.lo pair into IMAD.HI + IMAD: the
// same pipe time but twice the issue slots (seen in the SASS of the round-2 kernels; pipe rates: profiles/r2_microbench.md).
__device__ __forceinline__ void mul_wide(uint32_t a, uint32_t b, uint32_t& hi, uint32_t& lo) {
  unsigned long long p;
  asm("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(a), "r"(b));
  lo = (uint32_t)p;
  hi = (uint32_t)(p >> 32);
}

__device__ __forceinline__ void philox4x32_10(const PhiloxKeys& pk, uint32_t c0, uint32_t c1, uint32_t c2,
                                              uint32_t c3, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0, lo0, hi1, lo1;
    mul_wide(0xD2511F53u, c0, hi0, lo0);
    mul_wide(0xCD9E8D57u, c2, hi1, lo1);
    uint32_t n0 = hi1 ^ c1 ^ pk.k0[r];
    uint32_t n2 = hi0 ^ c3 ^ pk.k1[r];
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// u = (w + 0.5) 2^-32, exact, in one FMA: the double 2^52 + w is assembled from its words (no I2F), and
// (2^52 + w) 2^-32 + (2^-33 - 2^20) = (w + 0.5) 2^-32 has 33 significant bits, so the single rounding of the
// FMA returns it exactly -- the same double as the oracle's ((double)w + 0.5) * 2^-32.
__device__ __forceinline__ double uniform_from_word(uint32_t w) {
  return fma(__hiloint2double(0x43300000, (int)w), 2.3283064365386963e-10, 1.1641532182693481e-10 - 1048576.0);
}

// ---------------------------------------------------------------- polynomial helpers
template <int N>
__device__ __forceinline__ float horner(const float (&c)[N], float t) {
  float r = c[N - 1];
#pragma unroll
  for (int i = N - 2; i >= 0; --i) r = fmaf(r, t, c[i]);
  return r;
}

// ---------------------------------------------------------------- packed fp32 pairs (sm_100: FFMA2 / FMUL2 / FADD2)
// One instruction works on two fp32 values per lane (a 64-bit register pair) at two clocks per warp instruction:
// the FMA pipes do the same work per clock as with FFMA, but in half the issue slots, which is what the fp32 node
// loops are short of.  Each component is rounded exactly as the scalar operation rounds it.
__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
template <int N>
__device__ __forceinline__ float2 horner2(const float (&c)[N], float2 t) {
  float2 r = f2(c[N - 1]);
#pragma unroll
  for (int i = N - 2; i >= 0; --i) r = fma2(r, t, f2(c[i]));
  return r;
}

// ---------------------------------------------------------------- sin/cos
// fp32: two-step Cody-Waite reduction by pi/2 with FMAs (48 bits of pi/2), kernels on [-pi/4, pi/4].
// Valid for |x| < ~1e5 (k exact in fp32); the tracer's arguments are q*size < ~1e3.
// k = nearest integer to x*inv_period is taken from the mantissa of x*inv_period + 1.5*2^23 (no
// FRND/F2I on the XU pipe); |x*inv_period| < 2^22.
#define SAS_ROUND_MAGIC 12582912.0f
__device__ __forceinline__ void sincos_core(float x, float lo, float& s, float& c) {
  const float t = fmaf(x, 0.636619772f, SAS_ROUND_MAGIC);
  const int kb = __float_as_int(t);
  const float kf = t - SAS_ROUND_MAGIC;
  float r = fmaf(kf, -1.57079625129699707031e+00f, x);  // exact: the product has <= 32 significant bits
  r = fmaf(kf, -7.54978941586159635335e-08f, r);
  r += lo;  // the third Cody-Waite term, k * 5.4e-15, is below 1e-11 rad for |x| < 1e3
  const float z = r * r;
  const float SP[SAS_SIN_POLY_N] = SAS_SIN_POLY;
  const float CP[SAS_COS_POLY_N] = SAS_COS_POLY;
  const float ps = fmaf(r * z, horner(SP, z), r);
  const float pc = fmaf(z, horner(CP, z), 1.0f);
  const bool odd = (kb & 1) != 0;
  const float ss = odd ? pc : ps;
  const float cc = odd ? ps : pc;
  s = __int_as_float(__float_as_int(ss) ^ ((kb << 30) & 0x80000000));        // k mod 4 in {2,3}: -sin
  c = __int_as_float(__float_as_int(cc) ^ (((kb + 1) << 30) & 0x80000000));  // k mod 4 in {1,2}: -cos
}
__device__ __forceinline__ void sincos_r(float x, float& s, float& c) { sincos_core(x, 0.0f, s, c); }

// fp64 sin and cos for the tracer's arguments (azimuth 2 pi u, form-factor phases q x size): three-step
// Cody-Waite reduction by pi/2 with FMAs (pi/2 in three 33-bit pieces: n P1 is exact for |n| < 2^20), Taylor
// kernels on [-pi/4, pi/4] up to r^15 / r^16 (truncation below 6e-17 relative).  About one ulp, i.e. within the
// two ulps that separate any two good libraries (DESIGN.md R-C10); straight-line, no large-argument path, its
// constants in constant memory (an fp64 literal costs two moves per use).  |x| > 1e6 goes to the library.
__constant__ double c_sincos[20] = {
    0x1.45f306dc9c883p-1,                                     // 2 / pi
    0x1.921fb544p+0, 0x1.0b4611a6p-34, 0x1.3198a2ep-69,       // pi/2 = P1 + P2 + P3 + 8.5e-32 (33 bits each)
    -1.0 / 6.0, 1.0 / 120.0, -1.0 / 5040.0, 1.0 / 362880.0, -1.0 / 39916800.0, 1.0 / 6227020800.0,
    -1.0 / 1307674368000.0, 0.0,                              // sin: r + r^3 (S1 + z (S2 + ...)), z = r^2
    -0.5, 1.0 / 24.0, -1.0 / 720.0, 1.0 / 40320.0, -1.0 / 3628800.0, 1.0 / 479001600.0, -1.0 / 87178291200.0,
    1.0 / 20922789888000.0};                                  // cos: 1 + z (C1 + z (C2 + ...))
__device__ __forceinline__ void sincos_cw(double x, double& s, double& c) {
  const double t = fma(x, c_sincos[0], 6755399441055744.0);  // 1.5 * 2^52: nearest integer in the low word
  const int k = __double2loint(t);
  const double nf = t - 6755399441055744.0;
  double r = fma(-nf, c_sincos[1], x);
  r = fma(-nf, c_sincos[2], r);
  r = fma(-nf, c_sincos[3], r);
  const double z = r * r;
  double ps = fma(z, c_sincos[10], c_sincos[9]);
  ps = fma(ps, z, c_sincos[8]);
  ps = fma(ps, z, c_sincos[7]);
  ps = fma(ps, z, c_sincos[6]);
  ps = fma(ps, z, c_sincos[5]);
  ps = fma(ps, z, c_sincos[4]);
  ps = fma(r * z, ps, r);
  double pc = fma(z, c_sincos[19], c_sincos[18]);
  pc = fma(pc, z, c_sincos[17]);
  pc = fma(pc, z, c_sincos[16]);
  pc = fma(pc, z, c_sincos[15]);
  pc = fma(pc, z, c_sincos[14]);
  pc = fma(pc, z, c_sincos[13]);
  pc = fma(pc, z, c_sincos[12]);
  pc = fma(pc, z, 1.0);
  const double ss = (k & 1) ? pc : ps;
  const double cc = (k & 1) ? ps : pc;
  s = (k & 2) ? -ss : ss;
  c = ((k + 1) & 2) ? -cc : cc;
}
// sin u - u cos u, u >= 0, without the cancellation of the direct form at small u: the reduction gives u = k pi/2 + r,
// sin r = r + r z S(z), cos r = 1 + z C(z) (z = r^2); for k = 0 (u < pi/4) sin u - u cos u = r z (S - C) exactly in
// the polynomials, elsewhere the direct form is well conditioned.  No branch, no series (R-C12's series of Phi serves
// the same purpose in the oracle).
__device__ __forceinline__ double sin_minus_ucos(double u) {
  const double t = fma(u, c_sincos[0], 6755399441055744.0);
  const int k = __double2loint(t);
  const double nf = t - 6755399441055744.0;
  double r = fma(-nf, c_sincos[1], u);
  r = fma(-nf, c_sincos[2], r);
  r = fma(-nf, c_sincos[3], r);
  const double z = r * r;
  double S = fma(z, c_sincos[10], c_sincos[9]);
  S = fma(S, z, c_sincos[8]);
  S = fma(S, z, c_sincos[7]);
  S = fma(S, z, c_sincos[6]);
  S = fma(S, z, c_sincos[5]);
  S = fma(S, z, c_sincos[4]);
  double C = fma(z, c_sincos[19], c_sincos[18]);
  C = fma(C, z, c_sincos[17]);
  C = fma(C, z, c_sincos[16]);
  C = fma(C, z, c_sincos[15]);
  C = fma(C, z, c_sincos[14]);
  C = fma(C, z, c_sincos[13]);
  C = fma(C, z, c_sincos[12]);
  const double rz = r * z;
  const double ps = fma(rz, S, r), pc = fma(C, z, 1.0);
  const double ss = (k & 1) ? pc : ps;
  const double cc = (k & 1) ? ps : pc;
  const double sn = (k & 2) ? -ss : ss;
  const double cs = ((k + 1) & 2) ? -cc : cc;
  return (k == 0) ? rz * (S - C) : fma(-u, cs, sn);
}
__device__ __forceinline__ void sincos_d(double x, double& s, double& c) {
  if (fabs(x) > 1.0e6) { sincos(x, &s, &c); return; }
  sincos_cw(x, s, c);
}
__device__ __forceinline__ void sincos_r(double x, double& s, double& c) { sincos_d(x, s, c); }
// sin and cos of pi x for |x| < 2^51: x = k/2 + r exactly (|r| <= 1/4), then the same Taylor kernels on pi r
// (pi r carries one rounding of r pi_hi plus the r pi_lo correction: about one ulp)
__device__ __forceinline__ void sincospi_cw(double x, double& s, double& c) {
  const double t = fma(x, 2.0, 6755399441055744.0);
  const int k = __double2loint(t);
  const double nf = t - 6755399441055744.0;
  const double rr = fma(nf, -0.5, x);
  const double r = fma(rr, 0x1.921fb54442d18p+1, rr * 0x1.1a62633145c07p-53);
  const double z = r * r;
  double ps = fma(z, c_sincos[10], c_sincos[9]);
  ps = fma(ps, z, c_sincos[8]);
  ps = fma(ps, z, c_sincos[7]);
  ps = fma(ps, z, c_sincos[6]);
  ps = fma(ps, z, c_sincos[5]);
  ps = fma(ps, z, c_sincos[4]);
  ps = fma(r * z, ps, r);
  double pc = fma(z, c_sincos[19], c_sincos[18]);
  pc = fma(pc, z, c_sincos[17]);
  pc = fma(pc, z, c_sincos[16]);
  pc = fma(pc, z, c_sincos[15]);
  pc = fma(pc, z, c_sincos[14]);
  pc = fma(pc, z, c_sincos[13]);
  pc = fma(pc, z, c_sincos[12]);
  pc = fma(pc, z, 1.0);
  const double ss = (k & 1) ? pc : ps;
  const double cc = (k & 1) ? ps : pc;
  s = (k & 2) ? -ss : ss;
  c = ((k + 1) & 2) ? -cc : cc;
}

// fp32 reciprocal / square root: one MUFU each (~1 ulp), no IEEE fix-up path
__device__ __forceinline__ float rcp_fast(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sqrt_fast(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rsqrt_fast(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rcp_r(float x) { return rcp_fast(x); }
__device__ __forceinline__ double rcp_r(double x) { return 1.0 / x; }
__device__ __forceinline__ float sqrt_r(float x) { return sqrt_fast(x); }
__device__ __forceinline__ double sqrt_r(double x) { return sqrt(x); }
__device__ __forceinline__ float fma_r(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_r(double a, double b, double c) { return fma(a, b, c); }

// ---------------------------------------------------------------- phases in extended precision
// A form-factor phase is (projection of Q) x (particle length) and reaches hundreds of radians
// (q L/2 for a 2000 A rod).  In the fp32 model path the projection is carried as an unevaluated sum
// of two floats (hi + lo, from the fp64 value) and so is the length (split by the host), the product
// is formed with FMAs and the lo part joins after the Cody-Waite reduction: the reduced argument
// is good to ~1e-7 rad whatever the magnitude.  In the fp64 path both are plain doubles.
template <typename Real> struct Proj;
template <> struct Proj<double> { double v; };
template <> struct Proj<float> { float hi, lo; };
template <typename Real> struct Phase;
template <> struct Phase<double> { double v; };
template <> struct Phase<float> { float hi, lo; };

template <typename Real> __device__ __forceinline__ Proj<Real> make_proj(double v);
template <> __device__ __forceinline__ Proj<double> make_proj<double>(double v) { return {v}; }
template <> __device__ __forceinline__ Proj<float> make_proj<float>(double v) {
  const float hi = (float)v;
  return {hi, (float)(v - (double)hi)};
}
__device__ __forceinline__ Phase<double> phase_mul(Proj<double> p, double l_hi, double) { return {p.v * l_hi}; }
__device__ __forceinline__ Phase<float> phase_mul(Proj<float> p, float l_hi, float l_lo) {
  const float h = p.hi * l_hi;
  float e = fmaf(p.hi, l_hi, -h);
  e = fmaf(p.hi, l_lo, e);
  e = fmaf(p.lo, l_hi, e);
  return {h, e};
}
__device__ __forceinline__ double ph_val(Phase<double> p) { return p.v; }
__device__ __forceinline__ float ph_val(Phase<float> p) { return p.hi; }

__device__ __forceinline__ void sincos_ph(Phase<double> p, double& s, double& c) { sincos_d(p.v, s, c); }
__device__ __forceinline__ void sincos_ph(Phase<float> p, float& s, float& c) { sincos_core(p.hi, p.lo, s, c); }

// sin/cos of 2 pi u, u in (0,1), fp64, ~1e-13: exact reduction by quarter turns, Taylor kernels.
// Used by the fp32 model path for the per-neutron random orientation (the fp64 path calls sincos()).
__device__ __forceinline__ void sincos_2pi(double u, double& s, double& c) {
  const double kf = rint(4.0 * u);
  const double r = 6.283185307179586 * (u - 0.25 * kf);  // |r| <= pi/4
  const int k = (int)kf;
  const double z = r * r;
  double ps = fma(z, 1.0 / 6227020800.0, -1.0 / 39916800.0);
  ps = fma(ps, z, 1.0 / 362880.0);
  ps = fma(ps, z, -1.0 / 5040.0);
  ps = fma(ps, z, 1.0 / 120.0);
  ps = fma(ps, z, -1.0 / 6.0);
  ps = fma(r * z, ps, r);
  double pc = fma(z, -1.0 / 479001600.0, 1.0 / 3628800.0);
  pc = fma(pc, z, -1.0 / 40320.0);
  pc = fma(pc, z, 1.0 / 720.0);
  pc = fma(pc, z, -1.0 / 24.0);
  pc = fma(pc, z, 0.5);
  pc = fma(-z, pc, 1.0);
  const double ss = (k & 1) ? pc : ps;
  const double cc = (k & 1) ? ps : pc;
  s = (k & 2) ? -ss : ss;
  c = ((k + 1) & 2) ? -cc : cc;
}

// ---------------------------------------------------------------- sphere Phi(u) = 3 (sin u - u cos u)/u^3
// PAPER.md:37 (Eq. 1 over a sphere).  Even series below the threshold where the direct form cancels.
// fp32: reduction of u by pi (u = k pi + r, |r| <= pi/2), then sin u - u cos u = (-1)^k (sin r - u cos r)
// with sin r = r + r z S(z), cos r = 1 + z C(z), z = r^2.  For k = 0 (u < pi/2, where the direct form
// cancels) the same two polynomials give Phi without cancellation: sin r - r cos r = r^3 (S - C), so
// Phi = 3 (S(z) - C(z)).  SIGNED = false drops (-1)^k for callers that only use Phi^2.
template <bool SIGNED>
__device__ __forceinline__ float sphere_phi_core(float u, float lo) {
  const float t = fmaf(u, 0.318309886f, SAS_ROUND_MAGIC);
  const int kb = __float_as_int(t);
  const float kf = t - SAS_ROUND_MAGIC;
  float r = fmaf(kf, -3.14159250259399414062e+00f, u);
  r = fmaf(kf, -1.50995788317231927067e-07f, r);
  r += lo;  // the third Cody-Waite term, k * 1.1e-14, is below 1e-11 rad for |x| < 1e3
  const float z = r * r;
  const float SP[SAS_SINPI_POLY_N] = SAS_SINPI_POLY;
  const float CP[SAS_COSPI_POLY_N] = SAS_COSPI_POLY;
  const float S = horner(SP, z), C = horner(CP, z);
  const float sr = fmaf(r * z, S, r);
  const float cr = fmaf(z, C, 1.0f);
  const float inv = rcp_fast(u);
  float dir = fmaf(-u, cr, sr) * ((inv * inv) * inv);
  if (SIGNED) dir = __int_as_float(__float_as_int(dir) ^ (kb << 31));
  const float sel = (kb == __float_as_int(SAS_ROUND_MAGIC)) ? (S - C) : dir;
  return 3.0f * sel;
}
// sin u - u cos u in fp32 (the numerator of Phi without its 1/u^3): same reduction and polynomials as
// sphere_phi_core; r z (S - C) when u reduces with k = 0 (no cancellation), the direct form elsewhere.  Sign dropped
// (callers square it).
__device__ __forceinline__ float sin_minus_ucos_abs(float u, float lo) {
  const float t = fmaf(u, 0.318309886f, SAS_ROUND_MAGIC);
  const int kb = __float_as_int(t);
  const float kf = t - SAS_ROUND_MAGIC;
  float r = fmaf(kf, -3.14159250259399414062e+00f, u);
  r = fmaf(kf, -1.50995788317231927067e-07f, r);
  r += lo;
  const float z = r * r;
  const float SP[SAS_SINPI_POLY_N] = SAS_SINPI_POLY;
  const float CP[SAS_COSPI_POLY_N] = SAS_COSPI_POLY;
  const float S = horner(SP, z), C = horner(CP, z);
  const float rz = r * z;
  const float sr = fmaf(rz, S, r);
  const float cr = fmaf(z, C, 1.0f);
  return (kb == __float_as_int(SAS_ROUND_MAGIC)) ? rz * (S - C) : fmaf(-u, cr, sr);
}
// signed Phi of two arguments at once (packed arithmetic; the operations of sphere_phi_core<true>(u, 0) component
// by component)
__device__ __forceinline__ float2 sphere_phi2(float2 u) {
  const float2 t = fma2(u, f2(0.318309886f), f2(SAS_ROUND_MAGIC));
  const float2 kf = add2(t, f2(-SAS_ROUND_MAGIC));
  float2 r = fma2(kf, f2(-3.14159250259399414062e+00f), u);
  r = fma2(kf, f2(-1.50995788317231927067e-07f), r);
  const float2 z = mul2(r, r);
  const float SP[SAS_SINPI_POLY_N] = SAS_SINPI_POLY;
  const float CP[SAS_COSPI_POLY_N] = SAS_COSPI_POLY;
  const float2 S = horner2(SP, z), C = horner2(CP, z);
  const float2 sr = fma2(mul2(r, z), S, r);
  const float2 cr = fma2(z, C, f2(1.0f));
  const float2 inv = make_float2(rcp_fast(u.x), rcp_fast(u.y));
  const float2 dir = mul2(fma2(make_float2(-u.x, -u.y), cr, sr), mul2(mul2(inv, inv), inv));
  const float2 ser = add2(S, make_float2(-C.x, -C.y));
  const int kx = __float_as_int(t.x), ky = __float_as_int(t.y);
  const float sx = kx == __float_as_int(SAS_ROUND_MAGIC) ? ser.x : __int_as_float(__float_as_int(dir.x) ^ (kx << 31));
  const float sy = ky == __float_as_int(SAS_ROUND_MAGIC) ? ser.y : __int_as_float(__float_as_int(dir.y) ^ (ky << 31));
  return mul2(f2(3.0f), make_float2(sx, sy));
}
__device__ __forceinline__ float sphere_phi(float u) { return sphere_phi_core<true>(u, 0.0f); }
__device__ __forceinline__ double sphere_phi(double u) {
  if (u < 1.0e-8) return 1.0;   // Phi = 1 - u^2/10 + ...: 1 to the last bit
  return (3.0 * sin_minus_ucos(u)) / ((u * u) * u);
}

// ---------------------------------------------------------------- sinc
// sin(x) alone: reduction by pi, one odd polynomial on [-pi/2, pi/2], sign from the parity of k.
__device__ __forceinline__ float sin_reduced_pi(float x, float lo) {
  const float t = fmaf(x, 0.318309886f, SAS_ROUND_MAGIC);
  const int kb = __float_as_int(t);
  const float kf = t - SAS_ROUND_MAGIC;
  float r = fmaf(kf, -3.14159250259399414062e+00f, x);
  r = fmaf(kf, -1.50995788317231927067e-07f, r);
  r += lo;  // the third Cody-Waite term, k * 1.1e-14, is below 1e-11 rad for |x| < 1e3
  const float z = r * r;
  const float SP[SAS_SINPI_POLY_N] = SAS_SINPI_POLY;
  const float ps = fmaf(r * z, horner(SP, z), r);
  return __int_as_float(__float_as_int(ps) ^ (kb << 31));
}
// sin(x)/x: for tiny x the polynomial returns x itself, so the quotient is 1 to rounding; only the
// exact x = 0 gives 0 * inf = NaN, replaced by 1 with one select (no branch in the node loops)
__device__ __forceinline__ float sinc_from(float s, float x) {
  const float r = s * rcp_fast(x);
  return (r != r) ? 1.0f : r;
}
__device__ __forceinline__ float sinc_r(float x) {
  const float t = fmaf(x, 0.318309886f, SAS_ROUND_MAGIC);
  const int kb = __float_as_int(t);
  const float kf = t - SAS_ROUND_MAGIC;
  float r = fmaf(kf, -3.14159250259399414062e+00f, x);
  r = fmaf(kf, -1.50995788317231927067e-07f, r);
  const float z = r * r;
  const float SP[SAS_SINPI_POLY_N] = SAS_SINPI_POLY;
  const float ps = fmaf(r * z, horner(SP, z), r);
  return sinc_from(__int_as_float(__float_as_int(ps) ^ (kb << 31)), x);
}
__device__ __forceinline__ double sinc_r(double x) {
  if (x == 0.0) return 1.0;
  double s, c;
  sincos_d(x, s, c);
  return s / x;
}
// |sinc(q h)| for callers that square it: no sign, and the phase is biased by 1e-30 so that q h = 0 gives
// sin(1e-30) / 1e-30 = 1 instead of 0/0 (the bias is far below one ulp of any other phase)
__device__ __forceinline__ float sinc_abs_r(float q, float h) {
  const float x = fmaf(q, h, 1e-30f);
  const float t = fmaf(x, 0.318309886f, SAS_ROUND_MAGIC);
  const float kf = t - SAS_ROUND_MAGIC;
  float r = fmaf(kf, -3.14159250259399414062e+00f, x);
  r = fmaf(kf, -1.50995788317231927067e-07f, r);
  const float z = r * r;
  const float SP[SAS_SINPI_POLY_N] = SAS_SINPI_POLY;
  return fmaf(r * z, horner(SP, z), r) * rcp_fast(x);
}
__device__ __forceinline__ double sinc_abs_r(double q, double h) { return sinc_r(q * h); }
// two phases at once: the same operations as sinc_abs_r(float, float), component by component
__device__ __forceinline__ float2 sinc_abs_r2(float2 q, float h) {
  const float2 x = fma2(q, f2(h), f2(1e-30f));
  const float2 t = fma2(x, f2(0.318309886f), f2(SAS_ROUND_MAGIC));
  const float2 kf = add2(t, f2(-SAS_ROUND_MAGIC));
  float2 r = fma2(kf, f2(-3.14159250259399414062e+00f), x);
  r = fma2(kf, f2(-1.50995788317231927067e-07f), r);
  const float2 z = mul2(r, r);
  const float SP[SAS_SINPI_POLY_N] = SAS_SINPI_POLY;
  const float2 p = fma2(mul2(r, z), horner2(SP, z), r);
  return mul2(p, make_float2(rcp_fast(x.x), rcp_fast(x.y)));
}

// ---------------------------------------------------------------- Lambda(x) = 2 J1(x)/x, x >= 0
// x <= 8: one polynomial in x^2 (no square root needed); x > 8: Hankel form
//   J1 = sqrt(2/(pi x)) (P cos(x - 3pi/4) - Q sin(x - 3pi/4)).
__device__ __forceinline__ float lambda1_asym(float x, float xlo) {
  const float AP[SAS_J1_ASY_P_N] = SAS_J1_ASY_P;
  const float AQ[SAS_J1_ASY_Q_N] = SAS_J1_ASY_Q;
  const float inv = rcp_fast(x);
  const float t = fmaf(128.0f * inv, inv, -1.0f);
  const float P = horner(AP, t);
  const float Q = horner(AQ, t) * inv;
  float s, c;
  Phase<float> ph = {x, xlo};
  sincos_ph(ph, s, c);
  // cos(x-3pi/4) = (s - c)/sqrt2 ; sin(x-3pi/4) = -(s + c)/sqrt2
  const float j1v = (0.797884583f * 0.707106769f) * rsqrt_fast(x) * fmaf(P, s - c, Q * (s + c));
  return 2.0f * j1v * inv;
}
// argument given as x^2 (plus a first-order correction 2 x x_lo folded in by the caller)
__device__ __forceinline__ float lambda1_x2(float x2) {
  if (x2 <= 64.0f) {
    const float LA[SAS_LAMBDA_A_N] = SAS_LAMBDA_A;
    return horner(LA, fmaf(x2, 0.03125f, -1.0f));
  }
  return lambda1_asym(sqrt_fast(x2), 0.0f);
}
// caller guarantees x^2 <= 64 (the host checked q_max * R_max for the experiment)
__device__ __forceinline__ float lambda1_x2_small(float x2) {
  const float LA[SAS_LAMBDA_A_N] = SAS_LAMBDA_A;
  return horner(LA, fmaf(x2, 0.03125f, -1.0f));
}
// Lambda by class: the caller forms t = x^2 * lambda_class_scale(LC) - 1 and guarantees x^2 within the
// class range (1: 64, 2: 36, 3: 25, 4: 16); shorter ranges take shorter polynomials
__host__ __device__ constexpr double lambda_class_scale(int lc) {
  return lc == 4 ? 1.0 / 8.0 : lc == 3 ? 1.0 / 12.5 : lc == 2 ? 1.0 / 18.0 : 1.0 / 32.0;
}
template <int LC>
__device__ __forceinline__ float lambda1_class(float t) {
  if (LC == 4) { const float c[SAS_LAMBDA_16_N] = SAS_LAMBDA_16; return horner(c, t); }
  if (LC == 3) { const float c[SAS_LAMBDA_25_N] = SAS_LAMBDA_25; return horner(c, t); }
  if (LC == 2) { const float c[SAS_LAMBDA_36_N] = SAS_LAMBDA_36; return horner(c, t); }
  const float c[SAS_LAMBDA_A_N] = SAS_LAMBDA_A;
  return horner(c, t);
}
template <int LC>
__device__ __forceinline__ float2 lambda1_class2(float2 t) {
  if (LC == 4) { const float c[SAS_LAMBDA_16_N] = SAS_LAMBDA_16; return horner2(c, t); }
  if (LC == 3) { const float c[SAS_LAMBDA_25_N] = SAS_LAMBDA_25; return horner2(c, t); }
  if (LC == 2) { const float c[SAS_LAMBDA_36_N] = SAS_LAMBDA_36; return horner2(c, t); }
  const float c[SAS_LAMBDA_A_N] = SAS_LAMBDA_A;
  return horner2(c, t);
}
template <int LC>
__device__ __forceinline__ double lambda1_class(double t);
__device__ __forceinline__ double lambda1_x2_small(double x2);
__device__ __forceinline__ float lambda1_r(float x) { return lambda1_x2(x * x); }
// fp64 Lambda(x) = 2 J1(x)/x, x >= 0, of the tracer's own (gen_j1_f64.py): a Chebyshev series in x^2 up to x = 12, the
// Hankel form with Chebyshev series for P and x Q beyond; about 3e-16 absolute.  Coefficients in constant memory,
// Clenshaw recurrence (the power basis of a degree-14 fit loses five digits).  x > 1e6 goes to the library.
template <int N>
__device__ __forceinline__ double clenshaw(const double (&c)[N], double t) {
  const double t2 = t + t;
  double b1 = c[N - 1], b2 = 0.0;
#pragma unroll
  for (int k = N - 2; k >= 1; --k) {
    const double b0 = fma(t2, b1, c[k] - b2);
    b2 = b1;
    b1 = b0;
  }
  return fma(t, b1, c[0] - b2);
}
__device__ __forceinline__ double lambda1_r(double x) {
  if (x <= SAS_J1_XA) return clenshaw(c_j1a, fma(x * x, SAS_J1_A_SCALE, -1.0));
  if (x > 1.0e6) return (2.0 * j1(x)) / x;
  const double inv = 1.0 / x;
  const double t = fma(SAS_J1_B_SCALE * inv, inv, -1.0);
  const double P = clenshaw(c_j1p, t), Q = clenshaw(c_j1q, t) * inv;
  double s, c;
  sincos_cw(x, s, c);
  // J1 = sqrt(2/(pi x)) (P cos(x - 3pi/4) - Q sin(x - 3pi/4)) = sqrt(1/(pi x)) (P (s - c) + Q (s + c))
  const double j = (0.5641895835477563 * sqrt(inv)) * fma(P, s - c, Q * (s + c));
  return (2.0 * j) * inv;
}
// Lambda of a squared argument: the series range needs no square root (the barbell's slice loop has x^2 =
// Q_AB^2 rho^2 at hand and paid an fp64 sqrt per slice for x)
__device__ __forceinline__ double lambda1_sq(double x2) {
  if (x2 <= SAS_J1_XA * SAS_J1_XA) return clenshaw(c_j1a, fma(x2, SAS_J1_A_SCALE, -1.0));
  return lambda1_r(sqrt(x2));
}
__device__ __forceinline__ double lambda1_x2(double x2) { return lambda1_r(sqrt(x2)); }
__device__ __forceinline__ double lambda1_x2_small(double x2) { return lambda1_r(sqrt(x2)); }
template <int LC>
__device__ __forceinline__ double lambda1_class(double t) {
  return lambda1_r(sqrt(fmax((t + 1.0) / lambda_class_scale(LC), 0.0)));
}

// ---------------------------------------------------------------- the same functions of a Phase
__device__ __forceinline__ float sphere_phi_ph(Phase<float> p) { return sphere_phi_core<true>(p.hi, p.lo); }
// |Phi| up to sign, for models that square a single term
__device__ __forceinline__ float sphere_phi_abs_ph(Phase<float> p) { return sphere_phi_core<false>(p.hi, p.lo); }
__device__ __forceinline__ double sphere_phi_abs_ph(Phase<double> p) { return sphere_phi(p.v); }
__device__ __forceinline__ double sphere_phi_ph(Phase<double> p) { return sphere_phi(p.v); }

__device__ __forceinline__ float sinc_ph(Phase<float> p) { return sinc_from(sin_reduced_pi(p.hi, p.lo), p.hi); }
__device__ __forceinline__ double sinc_ph(Phase<double> p) { return sinc_r(p.v); }

__device__ __forceinline__ float lambda1_ph(Phase<float> p) {
  const float x = p.hi;
  if (x <= 8.0f) {
    const float LA[SAS_LAMBDA_A_N] = SAS_LAMBDA_A;
    return horner(LA, fmaf(x * x, 0.03125f, fmaf(x * p.lo, 0.0625f, -1.0f)));
  }
  return lambda1_asym(x, p.lo);
}
__device__ __forceinline__ double lambda1_ph(Phase<double> p) { return lambda1_r(p.v); }

// ---------------------------------------------------------------- Percus-Yevick S(q) (Table II F.11)
struct PYCoef {  // host-computed from the volume fraction (DESIGN.md R-C13)
  double alpha, beta, gamma, phi24, two_r;
};

template <typename Real>
__device__ __forceinline__ Real py_sq(Real q, const PYCoef& pc) {
  const Real x = (Real)pc.two_r * q;
  const Real a = (Real)pc.alpha, b = (Real)pc.beta, g = (Real)pc.gamma;
  const Real thr = sizeof(Real) == 4 ? (Real)2.0 : (Real)1.0;
  Real t1, t2, t3;
  if (x < thr) {
    const Real x2 = x * x;
    const Real a1[8] = {(Real)(1.0 / 3.0), (Real)(-1.0 / 30.0), (Real)(1.0 / 840.0), (Real)(-1.0 / 45360.0),
                        (Real)(1.0 / 3991680.0), (Real)(-1.0 / 518918400.0), (Real)(1.0 / 93405312000.0),
                        (Real)(-1.0 / 22230464256000.0)};
    const Real a2[8] = {(Real)(1.0 / 4.0), (Real)(-1.0 / 36.0), (Real)(1.0 / 960.0), (Real)(-1.0 / 50400.0),
                        (Real)(1.0 / 4354560.0), (Real)(-1.0 / 558835200.0), (Real)(1.0 / 99632332800.0),
                        (Real)(-1.0 / 23538138624000.0)};
    const Real a3[8] = {(Real)(1.0 / 6.0), (Real)(-1.0 / 48.0), (Real)(1.0 / 1200.0), (Real)(-1.0 / 60480.0),
                        (Real)(1.0 / 5080320.0), (Real)(-1.0 / 638668800.0), (Real)(1.0 / 112086374400.0),
                        (Real)(-1.0 / 26153487360000.0)};
    t1 = a1[7]; t2 = a2[7]; t3 = a3[7];
#pragma unroll
    for (int i = 6; i >= 0; --i) {
      t1 = fma_r(t1, x2, a1[i]);
      t2 = fma_r(t2, x2, a2[i]);
      t3 = fma_r(t3, x2, a3[i]);
    }
  } else {
    Real s, c;
    sincos_r(x, s, c);
    const Real x2 = x * x, x3 = x2 * x, x4 = x2 * x2;
    const Real i1 = rcp_r(x);
    const Real i3 = (i1 * i1) * i1;
    t1 = fma_r(-x, c, s) * i3;
    t2 = (fma_r((Real)2.0 * x, s, ((Real)2.0 - x2) * c) - (Real)2.0) * (i3 * i1);
    const Real in = fma_r(fma_r((Real)3.0, x2, (Real)-6.0), c, fma_r(x3 - (Real)6.0 * x, s, (Real)6.0));
    t3 = fma_r((Real)4.0, in, -(x4 * c)) * (i3 * i3);
  }
  return rcp_r(fma_r((Real)pc.phi24, fma_r(g, t3, fma_r(b, t2, a * t1)), (Real)1.0));
}

}  // namespace sas
