// Internal device-side parameter blocks of the CUDA tracer (not part of the ABI; not shared with oracle/).
#pragma once
#include <cstdint>

#include "device_math.cuh"

// -DSAS_DEBUG_BOUNDS (build.py: SAS_DEBUG_BOUNDS=1): the kernels trap on a queue, ring, table, pixel or work-item
// index outside its bounds (compute-sanitizer is closed on this pool; profiles/r2_debug_bounds.md records a run
// of the GPU test-suite on such a build).  The shipped build compiles the checks away.
#ifdef SAS_DEBUG_BOUNDS
#define SAS_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define SAS_CHECK(cond) do { } while (0)
#endif

namespace sas {

enum : int { ST_DETECTED = 0, ST_SLIT1 = 1, ST_SLIT2 = 2, ST_MISS_SAMPLE = 3, ST_UNREACHABLE = 4, ST_MISS_DET = 5 };

// kernel variants: one trace kernel is compiled per model form (models.cuh: eval_intensity)
enum : int {
  V_SPHERE = 0, V_CS_SPHERE = 1, V_CYL = 2, V_TRIAX = 3, V_CS_TRIAX = 4, V_FLAT = 5, V_CYL_QUAD = 6,
  V_PARA = 7, V_CS_CYL = 8, V_ELL = 9, V_BARBELL = 10, V_CAPPED = 11,  // NEXT-2: generic fp64 node loop
  V_ELL_CYL = 12, V_HOLLOW_CYL = 13, V_CS_ELL = 14, V_MICELLE = 15, V_HOLLOW_PRISM = 16,
  N_VARIANTS = 17
};

// table record widths (in Reals)
constexpr int TA_W = 4;   // per node of polydisperse axis 0
constexpr int TB_W = 4;   // per node of polydisperse axis 1
constexpr int TAB_W = 4;  // per (a,b) pair
constexpr int TOR_W = 4;  // per orientation tilt node: sin(delta), cos(delta), weight, pad (one 128-bit load)

// One virtual experiment: everything the kernel needs, precomputed on the host in fp64 with exactly the
// operations DESIGN.md section 3 writes (so that e.g. 0.5*det_xw is the same double on both sides).
struct ExpParams {
  // source and aiming (R-C2, R-C3)
  double src_xw, src_yh, focus_xw, focus_yh, focus_z, focus_area, p0_pref, dlam_w;
  double lambda_min, dlam;
  // slits (R-C4): half apertures
  double slit1_z, slit1_hx, slit1_hy, slit2_z, slit2_hx, slit2_hy;
  // sample (R-C5)
  double sample_z, hx, hy, hz, radius2;
  double mu_abs_2200, mu_inc;
  // Q choice (R-C7) and weight (R-C11)
  double q_min, dq, qnorm;
  // detector (R-C9)
  double det_z, det_hw, det_hh, det_sx, det_sy, det_nxd, det_nyd;
  double s_cut;  // classifier threshold on sin(theta); +inf when the instrument does not qualify
  // the same test in fp32 with a 2e-6 margin (geometry.cuh: surely_misses_detector_f32): lambda = w a + b, q = w a + b
  float cls_la, cls_lb, cls_qa, cls_qb, cls_lo, cls_hi;
  // model scalars (R-C12)
  double norm;        // 1e8 * scale / <V>
  double background;
  double flat_I;      // SAS_FLAT: scale + background
  double frame[9];    // particle axes A, B, C in the global frame for fixed / mean orientation (R-A7)
  double msize[4];    // mean sizes (triaxial a, b, c)
  PYCoef py;
  // Hayter MSA (R-S2): device address of this experiment's table in the fp64 pool -- the 32 node pairs 1/2 +- y_j of
  // the 64-node rule: y_j, sums and differences of the products 12 eta w Q(x) of a pair, then 12 eta D', k, 2 R_eff --
  // read once per detected neutron (models.cuh: msa_sq)
  const double* msa_tab;
  // per-event size sampling (SAS_PD_GAUSS_MC, DESIGN.md R-N1/R-N2): contrasts, 1e8 scale, widths (sizes: msize)
  double ev_sld[2], ev_scale, pd_rel[2];
  int32_t pd_mc[2];
  // slit-1 integer prefilter: when slit 1 lies in the source plane the test |x0| <= hx is a monotone
  // function of the Philox word, so it is decided on the raw 32-bit draws (bit-identical to the fp64 test)
  uint32_t s1_lo[2], s1_hi[2];
  int32_t s1_int_ok;
  int32_t sample_shape, has_mu, det_nx, det_ny;
  int32_t lateral_free;  // primary rays cannot touch the sample's lateral faces (geometry.cuh)
  int32_t slits_free;    // no stage-B ray can be cut by a slit (geometry.cuh)
  int32_t geo_fast;      // slits_free, lateral_free, box sample, no attenuation: trace_geometry<true>
  int32_t lambda_dist;   // 0 uniform band, 1 symmetric triangle (R-L1)
  int32_t model, orient_kind, sq_kind;
  int32_t n_a, n_b, n_th, n_ph;
  int32_t tab_off, tab_len;  // in doubles, inside the table pool
  int32_t lam_small;  // cylinder: (q_max * R_max)^2 <= 64, Lambda stays on its polynomial range
  int32_t exp_index;  // this experiment's index in the context (histogram slice, Philox counter word 3)
};
static_assert(sizeof(ExpParams) % 8 == 0, "ExpParams must be a multiple of 8 bytes");

struct KernelArgs {
  const ExpParams* exps;
  const uint32_t* exp_ids;       // experiments of this launch (one launch per kernel variant), [n_exp]
  const double* tab_pool;
  double* sum_p;
  double* sum_p2;
  unsigned long long* counts;
  unsigned long long* counters;  // [8]
  unsigned int* work_counter;
  // dump mode
  int32_t* d_pixel;
  double* d_weight;
  double* d_q;
  uint64_t first_id;       // id of offset 0
  uint32_t n_per_exp;      // ids per experiment in this launch (< 2^32)
  uint32_t n_exp;
  uint32_t exp_base;       // Philox counter word 3 of experiment index 0
  uint32_t item_ids;       // ids per work item (multiple of 32)
  uint32_t items_per_exp;
  uint32_t n_items;
  int32_t npix;
  int32_t tab_len_max;     // Reals of table space in shared memory
  // Work items: block b starts with item b (grid <= n_items); further items are gridDim.x + (fetch - work_base),
  // fetch = atomicAdd(work_counter, 1).  A launch with n_items > grid makes exactly n_items fetches (n_items - grid
  // that succeed, one failing one per block), one with n_items <= grid makes none: the host advances work_base by
  // that number after every launch, so the counter is never reset between launches.
  uint32_t work_base;
  int32_t use_exp0;        // single-experiment context: the parameter block travels with the kernel arguments
  PhiloxKeys keys;
  ExpParams exp0;          // (no dependent global loads before the first neutron of a small launch)
};

}  // namespace sas
