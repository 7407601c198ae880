// C-ABI shim of libsas_b200.so (include/sas.h): validation, host-side parameter and quadrature-table
// construction, launch planning, CUDA resource ownership.  All tracing runs in trace_kernel.cuh.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/sas.h"
#include "quadrature_host.h"
#include "reduce_kernel.cuh"
#include "trace_kernel.cuh"
#include "trace_kernel_ws.cuh"

using namespace sas;

namespace {

thread_local std::string g_create_error;

constexpr double TWO_PI = 6.283185307179586;
constexpr double FOUR_PI_3 = 4.1887902047863905;
constexpr double PI_D = 3.141592653589793;
constexpr int MAX_TIMED = SAS_MAX_LAUNCH_RECORDS;
#ifndef SAS_PDL
#define SAS_PDL 1   // programmatic dependent launch of the trace kernels (0: plain stream order)
#endif
constexpr int N_GROUPS = 4 * N_VARIANTS;
#ifndef SAS_ITEMS_PER_BLOCK
#define SAS_ITEMS_PER_BLOCK 16
#endif
#ifndef SAS_MIN_ITEM
#define SAS_MIN_ITEM 2048
#endif

}  // namespace

struct sas_ctx {
  std::string err;
  uint32_t n_exp = 0;
  int nx = 0, ny = 0, npix = 0;
  int precision = -1;  // set by the model(s)
  std::vector<int> exp_prec;  // precision the model arithmetic of each experiment runs in
  bool model_set = false;
  bool batch = false;
  std::vector<sas_instrument_desc> instr;
  std::vector<ExpParams> h_exps;
  std::vector<double> h_tab;
  int tab_len_max = 0;
  // device
  int device = 0, n_sm = 0;
  ExpParams* d_exps = nullptr;
  double* d_tab = nullptr;
  size_t d_tab_cap = 0;
  double *d_sum_p = nullptr, *d_sum_p2 = nullptr;
  unsigned long long* d_counts = nullptr;
  bool own_hist = true;
  unsigned long long* d_counters = nullptr;
  unsigned int* d_work = nullptr;
  uint32_t work_base = 0;   // fetches of the work counter made by every launch so far (KernelArgs::work_base)
  // experiments grouped by kernel: one launch per non-empty group (ids concatenated on the device).
  // group = variant + N_VARIANTS * (per-event sizes ? 1 : 0) + 2 N_VARIANTS * (fp64 model arithmetic ? 1 : 0)
  std::vector<uint32_t> group_ids[N_GROUPS];
  size_t group_off[N_GROUPS] = {};
  bool group_heavy[N_GROUPS] = {};  // consumer-bound group: launched in the 2 producer + 6 consumer split
  uint32_t* d_exp_ids = nullptr;
  double* d_rings = nullptr;  // ring sums of sas_reduce_radial: 3 x SAS_MAX_RINGS doubles + SAS_MAX_RINGS counts
  cudaStream_t stream = nullptr;
  bool own_stream = true;
  // bookkeeping
  uint64_t n_launches = 0;
  uint64_t launched = 0;  // neutrons traced into the detector since the last reset (counters[0])
  int last_grid = 0, last_block = 0, last_smem = 0;
  std::vector<cudaEvent_t> ev0, ev1;
  std::vector<sas_launch_record> records;  // of the timed launches (ms filled on request)
  uint64_t n_timed = 0;
  bool timing_on = true;   // sas_set_launch_timing
  double last_reduce_ms = 0.0;
};

namespace {

sas_status fail(sas_ctx* c, sas_status st, const std::string& msg) {
  if (c) c->err = msg; else g_create_error = msg;
  return st;
}

#define CUDA_TRY(ctx, call)                                                                     \
  do {                                                                                          \
    cudaError_t e_ = (call);                                                                    \
    if (e_ != cudaSuccess)                                                                      \
      return fail(ctx, SAS_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));          \
  } while (0)

__global__ void __launch_bounds__(256) zero_detector_kernel(unsigned long long* p0, unsigned long long* p1,
                                                            unsigned long long* p2, unsigned long long* counters, size_t n) {
  // programmatic dependent launch: the trace kernel that follows in the stream may be scheduled now; it touches
  // nothing this kernel writes before its own griddepcontrol.wait (trace_kernel*.cuh)
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) { p0[i] = 0ull; p1[i] = 0ull; p2[i] = 0ull; }
  if (blockIdx.x == 0 && threadIdx.x < 8) counters[threadIdx.x] = 0ull;
}

// Every call on a context runs on the device the context was created on and leaves the caller's current
// device as it found it.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(const sas_ctx* c) {
    if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) switched = cudaSetDevice(c->device) == cudaSuccess;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

bool finite_pos(double v) { return std::isfinite(v) && v > 0.0; }

sas_status validate_instrument(const sas_instrument_desc* d, std::string& why) {
  if (!d) { why = "instrument descriptor is NULL"; return SAS_EINVAL; }
  if (d->struct_size != sizeof(sas_instrument_desc)) { why = "sas_instrument_desc.struct_size mismatch"; return SAS_EINVAL; }
  if (d->sample_shape != SAS_SAMPLE_BOX && d->sample_shape != SAS_SAMPLE_CYL_Y) { why = "unknown sample_shape"; return SAS_EINVAL; }
  if (!finite_pos(d->src_xw) || !finite_pos(d->src_yh)) { why = "source size must be > 0"; return SAS_EINVAL; }
  if (!finite_pos(d->lambda_min) || !(d->lambda_max >= d->lambda_min) || !std::isfinite(d->lambda_max)) { why = "need 0 < lambda_min <= lambda_max"; return SAS_EINVAL; }
  if (!std::isfinite(d->flux) || d->flux < 0) { why = "flux must be >= 0"; return SAS_EINVAL; }
  if (!finite_pos(d->slit1_xw) || !finite_pos(d->slit1_yh) || !finite_pos(d->slit2_xw) || !finite_pos(d->slit2_yh)) { why = "slit apertures must be > 0"; return SAS_EINVAL; }
  if (!(d->slit1_z >= 0.0) || !(d->slit2_z >= d->slit1_z)) { why = "need 0 <= slit1_z <= slit2_z"; return SAS_EINVAL; }
  if (!finite_pos(d->focus_z) || !finite_pos(d->focus_xw) || !finite_pos(d->focus_yh)) { why = "focus rectangle must have z, width, height > 0"; return SAS_EINVAL; }
  if (!(d->sample_z > 0.0) || !finite_pos(d->sample_yh)) { why = "sample_z and sample_yh must be > 0"; return SAS_EINVAL; }
  if (d->sample_shape == SAS_SAMPLE_BOX && (!finite_pos(d->sample_xw) || !finite_pos(d->sample_zd))) { why = "box sample extents must be > 0"; return SAS_EINVAL; }
  if (d->sample_shape == SAS_SAMPLE_CYL_Y && !finite_pos(d->sample_radius)) { why = "cylinder sample radius must be > 0"; return SAS_EINVAL; }
  if (!(d->mu_abs_2200 >= 0.0) || !(d->mu_inc >= 0.0)) { why = "attenuation coefficients must be >= 0"; return SAS_EINVAL; }
  if (!(d->q_min >= 0.0) || !(d->q_max > d->q_min) || !std::isfinite(d->q_max)) { why = "need 0 <= q_min < q_max"; return SAS_EINVAL; }
  if (!finite_pos(d->det_dist) || !finite_pos(d->det_xw) || !finite_pos(d->det_yh)) { why = "detector distance and size must be > 0"; return SAS_EINVAL; }
  if (d->lambda_dist != SAS_LAMBDA_UNIFORM && d->lambda_dist != SAS_LAMBDA_TRIANGLE) { why = "unknown lambda_dist"; return SAS_EINVAL; }
  if (d->det_nx < 1 || d->det_ny < 1 || d->det_nx > 16384 || d->det_ny > 16384) { why = "detector pixels must be in 1..16384 per axis"; return SAS_EINVAL; }
  return SAS_OK;
}

sas_status validate_model(const sas_model_desc* m, std::string& why) {
  if (!m) { why = "model descriptor is NULL"; return SAS_EINVAL; }
  if (m->struct_size != sizeof(sas_model_desc)) { why = "sas_model_desc.struct_size mismatch"; return SAS_EINVAL; }
  if (m->model < SAS_SPHERE || m->model > SAS_HOLLOW_PRISM_THIN) { why = "unknown model"; return SAS_EINVAL; }
  if (m->precision != SAS_FP32 && m->precision != SAS_FP64) { why = "unknown precision"; return SAS_EINVAL; }
  if (m->orient_kind < SAS_ORIENT_FIXED || m->orient_kind > SAS_ORIENT_UNIFORM_ANGLES_MC) { why = "unknown orient_kind"; return SAS_EINVAL; }
  if (m->sq_kind != SAS_SQ_NONE && m->sq_kind != SAS_SQ_HARD_SPHERE_PY && m->sq_kind != SAS_SQ_HAYTER_MSA) { why = "unknown sq_kind"; return SAS_EINVAL; }
  if (!std::isfinite(m->scale) || !std::isfinite(m->background)) { why = "scale/background not finite"; return SAS_EINVAL; }
  static const int n_sizes[16] = {1, 2, 2, 3, 4, 0, 3, 3, 2, 3, 3, 3, 3, 3, 4, 4};
  static const int n_pd[16] = {1, 2, 2, 1, 2, 0, 1, 2, 2, 2, 2, 2, 2, 2, 1, 1};
  for (int i = 0; i < n_sizes[m->model]; ++i) {
    // a shell thickness may be 0, every other size must be > 0
    const bool may_be_zero = (m->model == SAS_CORE_SHELL_SPHERE && i == 1) || (m->model == SAS_CORE_SHELL_TRIAXIAL && i == 3) ||
                             (m->model == SAS_CORE_SHELL_CYLINDER && i == 2) || (m->model == SAS_CORE_SHELL_ELLIPSOID && i == 2) ||
                             (m->model == SAS_POLYMER_MICELLE && i >= 1);
    if (!std::isfinite(m->size[i]) || m->size[i] < 0.0 || (!may_be_zero && m->size[i] == 0.0)) { why = "model sizes must be > 0"; return SAS_EINVAL; }
  }
  if (m->model == SAS_POLYMER_MICELLE && m->size[3] != 0.0 && !(m->size[3] >= 1.0)) { why = "a micelle has 0 or >= 1 chains"; return SAS_EINVAL; }
  if ((m->model == SAS_BARBELL || m->model == SAS_CAPPED_CYLINDER) && !(m->size[2] >= m->size[0])) { why = "the end-piece radius must be >= the cylinder radius"; return SAS_EINVAL; }
  for (int k = 0; k < 2; ++k) {
    if (m->pd_kind[k] != SAS_PD_NONE && m->pd_kind[k] != SAS_PD_SCHULZ_QUAD && m->pd_kind[k] != SAS_PD_GAUSS_MC) { why = "unknown pd_kind"; return SAS_EINVAL; }
    if (m->pd_kind[k] == SAS_PD_GAUSS_MC) {
      if (k >= n_pd[m->model]) { why = "this model has no such polydisperse length"; return SAS_EINVAL; }
      if (!(m->pd_rel[k] >= 0.0) || !std::isfinite(m->pd_rel[k])) { why = "pd_rel must be >= 0"; return SAS_EINVAL; }
      if (m->pd_kind[1 - k] == SAS_PD_SCHULZ_QUAD || m->orient_kind == SAS_ORIENT_GAUSS_QUAD) {
        why = "per-event sizes (SAS_PD_GAUSS_MC) do not combine with fixed-node averages (DESIGN.md R-N1)";
        return SAS_EUNSUPPORTED;
      }
    }
    if (m->pd_kind[k] == SAS_PD_SCHULZ_QUAD) {
      if (k >= n_pd[m->model]) { why = "this model has no such polydisperse length"; return SAS_EINVAL; }
      if (m->pd_nodes[k] < 1 || m->pd_nodes[k] > SAS_MAX_NODES) { why = "pd_nodes must be in 1..SAS_MAX_NODES"; return SAS_EINVAL; }
      if (!(m->pd_rel[k] >= 0.0) || !(m->pd_rel[k] < 1.0)) { why = "pd_rel must be in [0,1)"; return SAS_EINVAL; }
    }
  }
  const int na = m->pd_kind[0] == SAS_PD_SCHULZ_QUAD ? m->pd_nodes[0] : 1;
  const int nb = m->pd_kind[1] == SAS_PD_SCHULZ_QUAD ? m->pd_nodes[1] : 1;
  if (na * nb > SAS_MAX_PD_PAIRS) { why = "pd_nodes[0]*pd_nodes[1] exceeds SAS_MAX_PD_PAIRS"; return SAS_EINVAL; }
  if (m->orient_kind == SAS_ORIENT_GAUSS_QUAD) {
    if (m->n_theta < 1 || m->n_theta > SAS_MAX_NODES || m->n_phi < 1 || m->n_phi > SAS_MAX_NODES) { why = "n_theta/n_phi must be in 1..SAS_MAX_NODES"; return SAS_EINVAL; }
    if (!(m->sigma_theta >= 0.0) || !(m->sigma_phi >= 0.0)) { why = "orientation spreads must be >= 0"; return SAS_EINVAL; }
    if (m->model != SAS_CYLINDER) {
      why = "SAS_ORIENT_GAUSS_QUAD is built for the cylinder only (DESIGN.md R-A11)";
      return SAS_EUNSUPPORTED;
    }
  }
  if (!std::isfinite(m->theta) || !std::isfinite(m->phi) || !std::isfinite(m->psi)) { why = "orientation angles not finite"; return SAS_EINVAL; }
  if (m->sq_kind == SAS_SQ_HAYTER_MSA) {
    const int32_t k = m->model;
    if (!(k == SAS_SPHERE || k == SAS_CORE_SHELL_SPHERE || k == SAS_TRIAXIAL_ELLIPSOID || k == SAS_CORE_SHELL_TRIAXIAL ||
          k == SAS_ELLIPSOID || k == SAS_CORE_SHELL_ELLIPSOID || k == SAS_POLYMER_MICELLE)) {
      why = "Hayter MSA is offered for the globular models only (spheres, ellipsoids, micelle)";
      return SAS_EUNSUPPORTED;
    }
    if (!finite_pos(m->sq_radius_eff) || !(m->sq_volfrac > 0.0) || !(m->sq_volfrac < 0.6)) { why = "Hayter MSA needs radius_eff > 0 and 0 < volfrac < 0.6"; return SAS_EINVAL; }
    if (!(m->sq_contact_kT >= 0.0) || !std::isfinite(m->sq_contact_kT)) { why = "Hayter MSA: sq_contact_kT must be >= 0"; return SAS_EINVAL; }
    if (!(m->sq_kappa_sigma >= 0.05) || !(m->sq_kappa_sigma <= 400.0)) { why = "Hayter MSA: sq_kappa_sigma must be in [0.05, 400]"; return SAS_EINVAL; }
  }
  if (m->sq_kind == SAS_SQ_HARD_SPHERE_PY) {
    if (!finite_pos(m->sq_radius_eff) || !(m->sq_volfrac >= 0.0) || !(m->sq_volfrac < 0.74)) { why = "PY S(q) needs radius_eff > 0 and 0 <= volfrac < 0.74"; return SAS_EINVAL; }
  }
  return SAS_OK;
}

// smallest / largest 32-bit word whose source coordinate passes |(u - 1/2) width| <= half
void slit1_word_window(double width, double half, uint32_t& lo, uint32_t& hi) {
  auto coord = [&](uint64_t w) {
    const double u = ((double)(uint32_t)w + 0.5) * 2.3283064365386963e-10;
    return (u - 0.5) * width;
  };
  auto pass = [&](uint64_t w) { return !(std::fabs(coord(w)) > half); };
  // coord is non-decreasing in w: the pass set is one interval (possibly empty)
  uint64_t a = 0, b = 0xFFFFFFFFull;
  // first w with coord(w) >= -half
  while (a < b) { uint64_t m = (a + b) / 2; if (coord(m) >= -half) b = m; else a = m + 1; }
  uint64_t first = a;
  a = 0; b = 0xFFFFFFFFull;
  // last w with coord(w) <= half
  while (a < b) { uint64_t m = (a + b + 1) / 2; if (coord(m) <= half) a = m; else b = m - 1; }
  uint64_t last = a;
  if (first <= last && pass(first) && pass(last)) { lo = (uint32_t)first; hi = (uint32_t)last; }
  else { lo = 1; hi = 0; }
}

void fill_instrument(const sas_instrument_desc& d, ExpParams& P) {
  P.src_xw = d.src_xw; P.src_yh = d.src_yh;
  P.focus_xw = d.focus_xw; P.focus_yh = d.focus_yh; P.focus_z = d.focus_z;
  P.focus_area = d.focus_xw * d.focus_yh;
  P.p0_pref = d.flux * ((d.src_xw * d.src_yh) * 1.0e4);
  P.lambda_min = d.lambda_min;
  P.dlam = d.lambda_max - d.lambda_min;
  P.dlam_w = P.dlam > 0.0 ? P.dlam : 1.0;
  P.lambda_dist = d.lambda_dist;
  P.slit1_z = d.slit1_z; P.slit1_hx = 0.5 * d.slit1_xw; P.slit1_hy = 0.5 * d.slit1_yh;
  P.slit2_z = d.slit2_z; P.slit2_hx = 0.5 * d.slit2_xw; P.slit2_hy = 0.5 * d.slit2_yh;
  P.sample_shape = d.sample_shape;
  P.sample_z = d.sample_z;
  P.hx = 0.5 * d.sample_xw; P.hy = 0.5 * d.sample_yh; P.hz = 0.5 * d.sample_zd;
  P.radius2 = d.sample_radius * d.sample_radius;
  P.mu_abs_2200 = d.mu_abs_2200; P.mu_inc = d.mu_inc;
  P.has_mu = (d.mu_abs_2200 != 0.0 || d.mu_inc != 0.0) ? 1 : 0;
  P.q_min = d.q_min; P.dq = d.q_max - d.q_min;
  P.qnorm = TWO_PI * (d.q_max - d.q_min);
  P.det_z = d.sample_z + d.det_dist;
  P.det_hw = 0.5 * d.det_xw; P.det_hh = 0.5 * d.det_yh;
  P.det_sx = (double)d.det_nx / d.det_xw; P.det_sy = (double)d.det_ny / d.det_yh;
  P.det_nxd = (double)d.det_nx; P.det_nyd = (double)d.det_ny;
  P.det_nx = d.det_nx; P.det_ny = d.det_ny;
  P.s_cut = INFINITY;
  P.s1_int_ok = 0;
  // the word window of the integer slit-1 test: everything passes unless slit 1 lies in the source plane
  P.s1_lo[0] = P.s1_lo[1] = 0u; P.s1_hi[0] = P.s1_hi[1] = 0xFFFFFFFFu;
  P.lateral_free = 0; P.slits_free = 0; P.geo_fast = 0;
  if (d.slit1_z == 0.0) {
    // slit 1 in the source plane: xs = x0 + dx*0 = x0 exactly, so the test depends on draws 0, 1 only
    slit1_word_window(d.src_xw, P.slit1_hx, P.s1_lo[0], P.s1_hi[0]);
    slit1_word_window(d.src_yh, P.slit1_hy, P.s1_lo[1], P.s1_hi[1]);
    P.s1_int_ok = 1;
    if (P.s1_lo[0] > P.s1_hi[0] || P.s1_lo[1] > P.s1_hi[1]) {
      // a slit narrower than the spacing of the source coordinates passes no draw at all: the kernels' window
      // test (w - lo <= hi - lo) cannot express an empty window, so the fp64 slit test decides (all absorbed)
      P.s1_lo[0] = P.s1_lo[1] = 0u; P.s1_hi[0] = P.s1_hi[1] = 0xFFFFFFFFu;
      P.s1_int_ok = 0;
    }
  }
  // Certain-miss classifier (geometry.cuh: surely_misses_detector).  Qualifies when, for EVERY ray the
  // source can emit through slit 1, (i) slit 2 cannot cut (it is the focus rectangle or larger),
  // (ii) the ray crosses the sample (beam envelope inside the sample's lateral extent).
  {
    const double m = 1.0e-6;
    const double x0m = 0.5 * d.src_xw, y0m = 0.5 * d.src_yh, xf = 0.5 * d.focus_xw, yf = 0.5 * d.focus_yh;
    const bool cyl = d.sample_shape == SAS_SAMPLE_CYL_Y;
    const double depth = cyl ? d.sample_radius : 0.5 * d.sample_zd;
    const double z_near = d.sample_z - depth, z_far = d.sample_z + depth;
    auto envelope = [&](double a0, double af, double z) {  // max |coordinate| of the beam at z
      const double slope = (af + a0) / d.focus_z;
      return z <= d.focus_z ? std::max(a0, af) : af + (z - d.focus_z) * slope;
    };
    const double bx = std::max(envelope(x0m, xf, z_near), envelope(x0m, xf, z_far));
    const double by = std::max(envelope(y0m, yf, z_near), envelope(y0m, yf, z_far));
    const bool slit2_sure = d.focus_z == d.slit2_z && d.focus_xw <= d.slit2_xw && d.focus_yh <= d.slit2_yh;
    const bool sample_sure = z_near > 0.0 && by <= 0.5 * d.sample_yh * (1.0 - m) &&
                             bx <= (cyl ? d.sample_radius : 0.5 * d.sample_xw) * (1.0 - m);
    // the lateral slabs of the sample cannot bind for a primary ray (needs the ray to start before the sample
    // and to move forward: z_near > 0, dz > 0 always); the cylinder's y slab likewise
    P.lateral_free = sample_sure ? 1 : 0;
    P.slits_free = (P.s1_int_ok && slit2_sure) ? 1 : 0;
    P.geo_fast = (P.slits_free && P.lateral_free && d.sample_shape == SAS_SAMPLE_BOX && !P.has_mu) ? 1 : 0;
    const double d_min = (d.sample_z + d.det_dist) - z_far;
    if (P.s1_int_ok && slit2_sure && sample_sure && d_min > 0.0) {
      const double delta = std::atan(std::hypot(xf + x0m, yf + y0m) / d.focus_z);  // max tilt of d^ from z
      const double r_diag = std::hypot(0.5 * d.det_xw, 0.5 * d.det_yh);
      const double t_cut = (r_diag * (1.0 + m) + std::hypot(bx, by)) / d_min;
      const double a_cut = (std::atan(t_cut) + delta) * (1.0 + m) + 1.0e-9;         // on 2 theta
      if (a_cut < 3.0) P.s_cut = std::sin(0.5 * a_cut) * (1.0 + m);
    }
  }
  // fp32 form of the classifier: u = (w + 1/2) 2^-32, lambda = lambda_min + u dlam, q = q_min + u dq, and
  // sin(theta) = q lambda / 4 pi in (s_cut, 0.999999), with both thresholds moved 2e-6 into the certain region
  {
    const double t = 2.3283064365386963e-10;  // 2^-32
    P.cls_la = (float)(P.dlam * t); P.cls_lb = (float)(P.lambda_min + 0.5 * t * P.dlam);
    P.cls_qa = (float)(P.dq * t); P.cls_qb = (float)(P.q_min + 0.5 * t * P.dq);
    const double four_pi = 4.0 * PI_D;
    P.cls_lo = std::isfinite(P.s_cut) ? std::nextafterf((float)(four_pi * P.s_cut * (1.0 + 2.0e-6)), INFINITY) : INFINITY;
    P.cls_hi = std::nextafterf((float)(four_pi * 0.999999 * (1.0 - 2.0e-6)), 0.0f);
    if (d.lambda_dist != SAS_LAMBDA_UNIFORM) {
      // a law that is not linear in the draw (R-L1): the fp32 test takes lambda_min, a lower bound of every
      // wavelength, in its first comparison; its second comparison (|Q| reachable: q lambda / 4 pi < 0.999999) must
      // then hold for the whole instrument, else the fp32 classifier is switched off (the fp64 geometry decides)
      P.cls_la = 0.0f;
      P.cls_lb = std::nextafterf((float)P.lambda_min, 0.0f);
      if (d.q_max * d.lambda_max < four_pi * 0.99) P.cls_hi = INFINITY; else P.cls_lo = INFINITY;
    }
  }
}

// Folds every Q-independent factor of the model into the node tables (models.cuh lists the layout).
void fill_model(const sas_model_desc& m, ExpParams& P, std::vector<double>& pool) {
  P.model = m.model; P.orient_kind = m.orient_kind; P.sq_kind = m.sq_kind;
  P.background = m.background;
  // per-event size sampling (R-N1, R-N2): the event evaluates Eq. 4 from the descriptor's own numbers
  for (int k = 0; k < 2; ++k) { P.pd_mc[k] = m.pd_kind[k] == SAS_PD_GAUSS_MC ? 1 : 0; P.pd_rel[k] = m.pd_rel[k]; }
  P.ev_sld[0] = m.sld[0]; P.ev_sld[1] = m.sld[1];
  P.ev_scale = 1.0e8 * m.scale;
  P.flat_I = m.scale + m.background;
  std::vector<double> xa, wa, xb, wb, dth, wth, dph, wph;
  schulz_rule(m.pd_kind[0] == SAS_PD_SCHULZ_QUAD ? m.pd_rel[0] : 0.0, m.pd_nodes[0], xa, wa);
  schulz_rule(m.pd_kind[1] == SAS_PD_SCHULZ_QUAD ? m.pd_rel[1] : 0.0, m.pd_nodes[1], xb, wb);
  if (m.orient_kind == SAS_ORIENT_GAUSS_QUAD) {
    gauss_tilt_rule(m.sigma_theta, m.n_theta, dth, wth);
    gauss_tilt_rule(m.sigma_phi, m.n_phi, dph, wph);
  } else {
    dth.assign(1, 0.0); wth.assign(1, 1.0); dph.assign(1, 0.0); wph.assign(1, 1.0);
  }
  const int na = (int)xa.size(), nb = (int)xb.size();
  P.n_a = na; P.n_b = nb; P.n_th = (int)dth.size(); P.n_ph = (int)dph.size();
  std::vector<double> ta(na * TA_W, 0.0), tb(nb * TB_W, 0.0), tab(na * nb * TAB_W, 0.0);
  double SV = 0.0;  // <V>
  const double s0 = m.sld[0], s1 = m.sld[1];
  for (int k = 0; k < 4; ++k) P.msize[k] = m.size[k];
  for (int a = 0; a < na; ++a)
    for (int b = 0; b < nb; ++b) {
      const double w = wa[a] * wb[b];
      double V = 1.0;
      switch (m.model) {
        case SAS_SPHERE: { const double R = m.size[0] * xa[a]; V = FOUR_PI_3 * R * R * R; } break;
        case SAS_CORE_SHELL_SPHERE: { const double Rt = m.size[0] * xa[a] + m.size[1] * xb[b]; V = FOUR_PI_3 * Rt * Rt * Rt; } break;
        case SAS_CYLINDER: { const double R = m.size[0] * xa[a], L = m.size[1] * xb[b]; V = PI_D * R * R * L; } break;
        case SAS_TRIAXIAL_ELLIPSOID: V = FOUR_PI_3 * (m.size[0] * xa[a]) * (m.size[1] * xa[a]) * (m.size[2] * xa[a]); break;
        case SAS_CORE_SHELL_TRIAXIAL: {
          const double t = m.size[3] * xb[b];
          V = FOUR_PI_3 * (m.size[0] * xa[a] + t) * (m.size[1] * xa[a] + t) * (m.size[2] * xa[a] + t);
        } break;
        case SAS_PARALLELEPIPED: V = (m.size[0] * xa[a]) * (m.size[1] * xa[a]) * (m.size[2] * xa[a]); break;
        case SAS_HOLLOW_PRISM_THIN: {
          const double pa = m.size[0] * xa[a], pb = m.size[1] * xa[a], pc = m.size[2] * xa[a];
          V = m.size[3] * (2.0 * (pa * pb + pb * pc + pc * pa));   // wall volume (R-M5)
        } break;
        case SAS_CORE_SHELL_CYLINDER: {
          const double Rt = m.size[0] * xa[a] + m.size[2], Lt = m.size[1] * xb[b] + 2.0 * m.size[2];
          V = PI_D * Rt * Rt * Lt;
        } break;
        case SAS_ELLIPSOID: { const double Re = m.size[0] * xa[a], Rp = m.size[1] * xb[b]; V = FOUR_PI_3 * Re * Re * Rp; } break;
        case SAS_ELLIPTICAL_CYLINDER: V = PI_D * (m.size[0] * xa[a]) * (m.size[1] * xa[a]) * (m.size[2] * xb[b]); break;
        case SAS_HOLLOW_CYLINDER: {
          const double Ri = m.size[0] * xa[a], Ro = Ri + m.size[2], L = m.size[1] * xb[b];
          V = PI_D * (Ro * Ro - Ri * Ri) * L;
        } break;
        case SAS_CORE_SHELL_ELLIPSOID: {
          const double Ret = m.size[0] * xa[a] + m.size[2], Rpt = m.size[1] * xb[b] + m.size[2];
          V = FOUR_PI_3 * Ret * Ret * Rpt;
        } break;
        case SAS_POLYMER_MICELLE: { const double R = m.size[0] * xa[a]; V = FOUR_PI_3 * R * R * R + m.size[3] * m.size[2]; } break;
        case SAS_BARBELL: case SAS_CAPPED_CYLINDER: {
          // cylinder + two sphere pieces z in [L/2, zc + Rb] (R-M2)
          const double R = m.size[0] * xa[a], L = m.size[1] * xb[b], Rb = m.size[2];
          const double h = std::sqrt(std::max(Rb * Rb - R * R, 0.0));
          const double zc = m.model == SAS_BARBELL ? 0.5 * L + h : 0.5 * L - h;
          const double z0 = 0.5 * L, z1 = zc + Rb, p = z1 - zc, q = z0 - zc;
          V = PI_D * R * R * L + 2.0 * PI_D * (Rb * Rb * (z1 - z0) - (p * p * p - q * q * q) / 3.0);
        } break;
        default: break;
      }
      SV += w * V;
    }
  // a length that multiplies a projection of Q: (hi, lo) split for the fp32 path (device_math.cuh)
  const bool f32 = m.precision == SAS_FP32;
  auto split = [&](double L, double* dst) {
    if (f32) { const float h = (float)L; dst[0] = (double)h; dst[1] = L - (double)h; }
    else { dst[0] = L; dst[1] = 0.0; }
  };
  for (int a = 0; a < na; ++a) {
    double* r = &ta[a * TA_W];
    switch (m.model) {
      case SAS_SPHERE: {
        const double R = m.size[0] * xa[a], V = FOUR_PI_3 * R * R * R;
        split(R, r); r[2] = wa[a] * (s0 * V) * (s0 * V);
        r[3] = wa[a] * ((4.0 * PI_D * s0) * (4.0 * PI_D * s0));   // 9 w (drho V)^2 / R^6: the fp64 node loop (models.cuh)
      } break;
      case SAS_CORE_SHELL_SPHERE: { const double R = m.size[0] * xa[a], V = FOUR_PI_3 * R * R * R; split(R, r); r[2] = (s0 - s1) * V; r[3] = wa[a]; } break;
      case SAS_CYLINDER: { const double R = m.size[0] * xa[a], c = s0 * PI_D * R * R; split(R, r); r[2] = wa[a] * c * c; r[3] = R * R; } break;
      case SAS_TRIAXIAL_ELLIPSOID: { const double x = xa[a], V = FOUR_PI_3 * (m.size[0] * x) * (m.size[1] * x) * (m.size[2] * x); split(x, r); r[2] = wa[a] * (s0 * V) * (s0 * V); } break;
      case SAS_CORE_SHELL_TRIAXIAL: { const double x = xa[a], V = FOUR_PI_3 * (m.size[0] * x) * (m.size[1] * x) * (m.size[2] * x); split(x, r); r[2] = (s0 - s1) * V; r[3] = wa[a]; } break;
      // NEXT-2 models: the node value and its weight; the kernel forms the amplitude itself (models.cuh)
      case SAS_PARALLELEPIPED: case SAS_CORE_SHELL_CYLINDER: case SAS_ELLIPSOID: case SAS_BARBELL: case SAS_CAPPED_CYLINDER:
      case SAS_ELLIPTICAL_CYLINDER: case SAS_HOLLOW_CYLINDER: case SAS_CORE_SHELL_ELLIPSOID: case SAS_POLYMER_MICELLE:
      case SAS_HOLLOW_PRISM_THIN:
        r[0] = xa[a]; r[2] = wa[a]; break;
      default: break;
    }
  }
  for (int b = 0; b < nb; ++b) {
    double* r = &tb[b * TB_W];
    switch (m.model) {
      case SAS_CYLINDER: { const double L = m.size[1] * xb[b]; split(0.5 * L, r); r[2] = wb[b] * L * L; } break;
      case SAS_CORE_SHELL_TRIAXIAL: { const double t = m.size[3] * xb[b]; r[0] = t; r[1] = wb[b]; r[2] = t * t; } break;
      case SAS_PARALLELEPIPED: case SAS_CORE_SHELL_CYLINDER: case SAS_ELLIPSOID: case SAS_BARBELL: case SAS_CAPPED_CYLINDER:
      case SAS_ELLIPTICAL_CYLINDER: case SAS_HOLLOW_CYLINDER: case SAS_CORE_SHELL_ELLIPSOID: case SAS_POLYMER_MICELLE:
      case SAS_HOLLOW_PRISM_THIN:
        r[0] = xb[b]; r[2] = wb[b]; break;
      default: r[1] = wb[b]; break;
    }
  }
  for (int a = 0; a < na; ++a)
    for (int b = 0; b < nb; ++b) {
      double* r = &tab[(a * nb + b) * TAB_W];
      if (m.model == SAS_CORE_SHELL_SPHERE) {
        const double Rt = m.size[0] * xa[a] + m.size[1] * xb[b];
        split(Rt, r); r[2] = s1 * (FOUR_PI_3 * Rt * Rt * Rt);
      } else if (m.model == SAS_CORE_SHELL_TRIAXIAL) {
        const double x = xa[a], t = m.size[3] * xb[b];
        r[0] = s1 * (FOUR_PI_3 * (m.size[0] * x + t) * (m.size[1] * x + t) * (m.size[2] * x + t));
        r[1] = 2.0 * x * t;
      }
    }
  P.norm = (1.0e8 * m.scale) / SV;
  // mean particle frame (R-A7)
  {
    const double st = std::sin(m.theta), ct = std::cos(m.theta), sp = std::sin(m.phi), cp = std::cos(m.phi);
    const double ss = std::sin(m.psi), cs = std::cos(m.psi);
    const double a0[3] = {ct * cp, ct * sp, -st}, b0[3] = {-sp, cp, 0.0};
    const double c0[3] = {st * cp, st * sp, ct};
    for (int i = 0; i < 3; ++i) {
      P.frame[i] = cs * a0[i] + ss * b0[i];
      P.frame[3 + i] = cs * b0[i] - ss * a0[i];
      P.frame[6 + i] = c0[i];
    }
  }
  // Percus-Yevick coefficients (R-C13)
  {
    const double phi = m.sq_volfrac, om = 1.0 - phi, om4 = (om * om) * (om * om);
    P.py.alpha = ((1.0 + 2.0 * phi) * (1.0 + 2.0 * phi)) / om4;
    P.py.beta = (-6.0 * phi) * ((1.0 + 0.5 * phi) * (1.0 + 0.5 * phi)) / om4;
    P.py.gamma = (phi * P.py.alpha) * 0.5;
    P.py.phi24 = 24.0 * phi;
    P.py.two_r = 2.0 * m.sq_radius_eff;
  }
  P.tab_off = (int)pool.size();
  P.msa_tab = nullptr;
  pool.insert(pool.end(), ta.begin(), ta.end());
  pool.insert(pool.end(), tb.begin(), tb.end());
  pool.insert(pool.end(), tab.begin(), tab.end());
  for (size_t i = 0; i < dth.size(); ++i) { pool.push_back(std::sin(dth[i])); pool.push_back(std::cos(dth[i])); pool.push_back(wth[i]); pool.push_back(0.0); }
  // the phi tilts in pairs, [sin0, sin1, cos0, cos1, w0, w1, 0, 0] (models.cuh: cyl_quad_row); an odd count is
  // padded with a node of weight 0 on the mean axis
  for (size_t i = 0; i < dph.size(); i += 2) {
    const bool two = i + 1 < dph.size();
    pool.push_back(std::sin(dph[i])); pool.push_back(two ? std::sin(dph[i + 1]) : 0.0);
    pool.push_back(std::cos(dph[i])); pool.push_back(two ? std::cos(dph[i + 1]) : 1.0);
    pool.push_back(wph[i]); pool.push_back(two ? wph[i + 1] : 0.0);
    pool.push_back(0.0); pool.push_back(0.0);
  }
  P.tab_len = (int)pool.size() - P.tab_off;
}

// Hayter MSA (R-S2): solve the closure and append the experiment's S(q) table to the pool; *off = its offset in the
// pool (the device address is formed when the pool is uploaded)
sas_status fill_msa(const sas_model_desc& m, const sas_instrument_desc& ins, std::vector<double>& pool, size_t* off,
                    std::string& why) {
  if (2.0 * ins.q_max * m.sq_radius_eff > 64.0) { why = "Hayter MSA: 2 q_max sq_radius_eff exceeds 64, the range of the 64-node rule"; return SAS_EUNSUPPORTED; }
  double u[5], g1 = 0.0;
  if (!msa_solve(m.sq_volfrac, m.sq_contact_kT, m.sq_kappa_sigma, u, &g1)) { why = "Hayter MSA: the closure did not converge"; return SAS_EUNSUPPORTED; }
  if (!(g1 >= 0.0)) { why = "Hayter MSA: negative contact value g(1+): the closure fails for this dilute, strongly charged system (rescaled MSA not implemented)"; return SAS_EUNSUPPORTED; }
  std::vector<double> x, w;
  legendre_rule_01(64, x, w);
  const double eta12 = 12.0 * m.sq_volfrac, k = m.sq_kappa_sigma;
  // the nodes lie in pairs 1/2 +- y (ascending: x[j] and x[63 - j]); rows: y_j, c+ + c-, c+ - c- (models.cuh: msa_sq)
  std::vector<double> cq(64);
  for (int j = 0; j < 64; ++j)
    cq[j] = eta12 * w[j] * (((0.5 * u[0]) * (x[j] * x[j] - 1.0) + u[1] * (x[j] - 1.0)) + (u[2] * std::exp(-k * x[j]) - u[3]));
  for (int j = 0; j < 32; ++j)
    if (!(x[63 - j] > x[j]) || std::fabs((x[63 - j] + x[j]) - 1.0) > 1e-14) { why = "Hayter MSA: the 64-node rule is not symmetric"; return SAS_EUNSUPPORTED; }
  *off = pool.size();
  for (int j = 0; j < 32; ++j) pool.push_back(0.5 * (x[63 - j] - x[j]));
  for (int j = 0; j < 32; ++j) pool.push_back(cq[63 - j] + cq[j]);
  for (int j = 0; j < 32; ++j) pool.push_back(cq[63 - j] - cq[j]);
  pool.push_back(eta12 * u[4]);
  pool.push_back(k);
  pool.push_back(2.0 * m.sq_radius_eff);
  pool.push_back(0.0);
  return SAS_OK;
}

}  // namespace

// ===================================================================== context plumbing
namespace {

sas_status alloc_common(sas_ctx* c) {
  CUDA_TRY(c, cudaGetDevice(&c->device));
  {
    // Gauss-Legendre rule of the end-piece integrals (models.cuh: c_gl), the host's own Jacobi-matrix rule
    std::vector<double> a(GL_N, 0.0), b(GL_N, 0.0), x, w, both;
    for (int k = 1; k < GL_N; ++k) b[k] = (double)k / std::sqrt(4.0 * (double)k * (double)k - 1.0);
    gauss_from_jacobi(a, b, x, w);
    both.insert(both.end(), x.begin(), x.end());
    both.insert(both.end(), w.begin(), w.end());
    CUDA_TRY(c, cudaMemcpyToSymbol(c_gl, both.data(), both.size() * sizeof(double)));
  }
  CUDA_TRY(c, cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, c->device));
  CUDA_TRY(c, cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking));
  c->own_stream = true;
  c->own_hist = true;  // the context's own histograms are allocated by the first call that needs them (ensure_hist)
  CUDA_TRY(c, cudaMalloc(&c->d_counters, 8 * sizeof(unsigned long long)));
  CUDA_TRY(c, cudaMalloc(&c->d_work, sizeof(unsigned int)));
  CUDA_TRY(c, cudaMemset(c->d_work, 0, sizeof(unsigned int)));
  CUDA_TRY(c, cudaMalloc(&c->d_exp_ids, (size_t)c->n_exp * sizeof(uint32_t)));
  CUDA_TRY(c, cudaMalloc(&c->d_exps, (size_t)c->n_exp * sizeof(ExpParams)));
  CUDA_TRY(c, cudaMemsetAsync(c->d_counters, 0, 8 * sizeof(unsigned long long), c->stream));
  c->launched = 0;
  return SAS_OK;
}

// The context's own zeroed histograms, unless the caller bound its buffers (sas_bind_buffers) before anything
// needed them: a batch of 1024 detectors is 1.2 GB that a binding caller never wants allocated twice.
sas_status ensure_hist(sas_ctx* c) {
  if (c->d_sum_p) return SAS_OK;
  const size_t nh = (size_t)c->n_exp * c->npix;
  CUDA_TRY(c, cudaMalloc(&c->d_sum_p, nh * sizeof(double)));
  CUDA_TRY(c, cudaMalloc(&c->d_sum_p2, nh * sizeof(double)));
  CUDA_TRY(c, cudaMalloc(&c->d_counts, nh * sizeof(unsigned long long)));
  CUDA_TRY(c, cudaMemsetAsync(c->d_sum_p, 0, nh * sizeof(double), c->stream));
  CUDA_TRY(c, cudaMemsetAsync(c->d_sum_p2, 0, nh * sizeof(double), c->stream));
  CUDA_TRY(c, cudaMemsetAsync(c->d_counts, 0, nh * sizeof(unsigned long long), c->stream));
  c->own_hist = true;
  return SAS_OK;
}

// how many amplitude evaluations one detected neutron costs
int node_evaluations(const sas_model_desc& m) {
  if (m.model == SAS_FLAT) return 1;
  auto pd = [&](int k) { return (m.pd_kind[k] == SAS_PD_SCHULZ_QUAD && m.pd_rel[k] > 0.0 && m.pd_nodes[k] > 1) ? m.pd_nodes[k] : 1; };
  int n = pd(0) * pd(1);
  if (m.orient_kind == SAS_ORIENT_GAUSS_QUAD && m.model == SAS_CYLINDER) {
    n *= (m.sigma_theta > 0.0 && m.n_theta > 1) ? m.n_theta : 1;
    n *= (m.sigma_phi > 0.0 && m.n_phi > 1) ? m.n_phi : 1;
  }
  return n;
}

// largest phase q x length the fp32 node loops of this experiment can see (sizes times their largest node)
double max_phase(const sas_model_desc& m, const sas_instrument_desc& ins) {
  double f[2] = {1.0, 1.0};
  for (int k = 0; k < 2; ++k)
    if (m.pd_kind[k] == SAS_PD_SCHULZ_QUAD && m.pd_rel[k] > 0.0 && m.pd_nodes[k] > 1) {
      std::vector<double> x, w;
      schulz_rule(m.pd_rel[k], m.pd_nodes[k], x, w);
      f[k] = *std::max_element(x.begin(), x.end());
    }
  double len = 0.0;
  switch (m.model) {
    case SAS_SPHERE: len = m.size[0] * f[0]; break;
    case SAS_CORE_SHELL_SPHERE: len = m.size[0] * f[0] + m.size[1] * f[1]; break;
    case SAS_CYLINDER: len = std::max(m.size[0] * f[0], 0.5 * m.size[1] * f[1]); break;
    case SAS_TRIAXIAL_ELLIPSOID: len = std::max(m.size[0], std::max(m.size[1], m.size[2])) * f[0]; break;
    case SAS_CORE_SHELL_TRIAXIAL: len = std::max(m.size[0], std::max(m.size[1], m.size[2])) * f[0] + m.size[3] * f[1]; break;
    case SAS_POLYMER_MICELLE: len = m.size[0] * f[0] + m.size[1]; break;
    case SAS_FLAT: break;
    default:  // NEXT-2 bodies: every size is a length; a generous bound
      len = (std::max(std::max(m.size[0], m.size[1]), std::max(m.size[2], m.size[3])) + m.size[2]) * std::max(f[0], f[1]);
      break;
  }
  return ins.q_max * len;
}

// Precision the model arithmetic of one experiment really runs in.  A model without any node loop is evaluated
// once per detected neutron; that single evaluation is done in fp64 whatever precision was asked for: it costs
// little next to the fp64 geometry before it, and a monodisperse form factor near its zeros cannot meet 1e-5 in
// fp32.  Per-event sizes (SAS_PD_GAUSS_MC) and the NEXT-2 models are fp64 as well (R-N2).
// So is an experiment whose phases leave the range the fp32 argument reductions are proven for (|x| < 1e3).
constexpr double FP32_MAX_PHASE = 1.0e3;
int effective_precision(const sas_model_desc& m, const sas_instrument_desc& ins) {
  if (m.precision == SAS_FP64) return SAS_FP64;
  if (node_evaluations(m) <= 1) return SAS_FP64;
  if (m.pd_kind[0] == SAS_PD_GAUSS_MC || m.pd_kind[1] == SAS_PD_GAUSS_MC || m.model >= SAS_PARALLELEPIPED) return SAS_FP64;
  if (max_phase(m, ins) > FP32_MAX_PHASE) return SAS_FP64;
  return SAS_FP32;
}

// Is a launch of this experiment on the warp-specialised kernel bound by its consumers (stages B and C) rather than
// by the Philox producers?  Then the block is split into one producer and three consumer warpgroups instead of one
// and one (trace_kernel_ws.cuh).  Measured at 1e8..1e9 neutrons, heavy split against default: barbell per event
// +9 %, Hayter MSA +3 %, 32 fp64 sphere nodes +5 % (break-even at 20-24 nodes), 2 x 2 nodes of a core-shell
// cylinder +12 %, 3 x 3 of an elliptical cylinder +8 % (2 x 2: even), 5 x 4 nodes of a plain cylinder -7 %; one fp64
// evaluation per neutron (sphere -13 %, per-event cylinder -5 %) and the fp32 node loops (32 sphere nodes -8 %) stay
// with the default split.  The rule: node evaluations, each weighted by what one costs next to an fp64 sphere node
// (slope of the kernel time against the node count: sphere 0.0102, cylinder 0.0045, elliptical cylinder 0.039,
// core-shell cylinder 0.081 ms per evaluation and 1e8 neutrons; the other models by their instruction mix).
#ifndef SAS_WS_MSA_HEAVY
#define SAS_WS_MSA_HEAVY 1
#endif
#ifndef SAS_WS_HEAVY_EVALS
#define SAS_WS_HEAVY_EVALS 24
#endif
double eval_weight(int model) {
  switch (model) {
    case SAS_SPHERE: return 1.0;                  // measured
    case SAS_CORE_SHELL_SPHERE: return 2.0;
    case SAS_CYLINDER: return 0.5;                // measured (0.45)
    case SAS_TRIAXIAL_ELLIPSOID: return 1.2;
    case SAS_PARALLELEPIPED: return 3.0;
    case SAS_CORE_SHELL_CYLINDER: return 8.0;     // measured
    case SAS_ELLIPSOID: return 1.2;
    case SAS_ELLIPTICAL_CYLINDER: return 3.8;     // measured
    case SAS_HOLLOW_CYLINDER: return 6.0;
    case SAS_CORE_SHELL_ELLIPSOID: return 2.4;
    case SAS_POLYMER_MICELLE: return 4.0;
    case SAS_HOLLOW_PRISM_THIN: return 5.0;
    default: return 1.0;
  }
}
bool consumer_bound(const ExpParams& P, int precision) {
  if (precision != SAS_FP64 || P.model == SAS_FLAT) return false;
  if (P.model == SAS_BARBELL || P.model == SAS_CAPPED_CYLINDER) return true;  // 64 slices with a Bessel J1 each
  if (P.sq_kind == SAS_SQ_HAYTER_MSA) return SAS_WS_MSA_HEAVY != 0;            // 33 fp64 sine/cosine pairs
  const long evals = (long)std::max(P.n_a, 1) * std::max(P.n_b, 1) * std::max(P.n_th, 1) * std::max(P.n_ph, 1);
  if (SAS_WS_HEAVY_EVALS == 0) return true;     // (test builds: every fp64 launch in the heavy split)
  return evals > 1 && (double)evals * eval_weight(P.model) >= (double)SAS_WS_HEAVY_EVALS;
}

// (re)build ExpParams + tables of every experiment and upload them
sas_status upload_models(sas_ctx* c, const sas_model_desc* models) {
  c->h_tab.clear();
  c->tab_len_max = 0;
  std::vector<std::pair<uint32_t, size_t>> msa_offsets;   // experiments with a Hayter MSA table and where it starts
  c->exp_prec.assign(c->n_exp, SAS_FP64);
  c->precision = SAS_FP32;  // of the context: fp64 as soon as one experiment runs in fp64 (introspection only)
  for (uint32_t e = 0; e < c->n_exp; ++e)
    if (max_phase(models[e], c->instr[e]) > 1.0e6)   // the tracer's own fp64 sin/cos reduce exactly below 2^20 pi/2
      return fail(c, SAS_EUNSUPPORTED, "experiment " + std::to_string(e) + ": q_max x particle size exceeds 1e6 rad");
  for (uint32_t e = 0; e < c->n_exp; ++e) {
    ExpParams& P = c->h_exps[e];
    fill_instrument(c->instr[e], P);
    P.exp_index = (int32_t)e;
    sas_model_desc m = models[e];
    m.precision = c->exp_prec[e] = effective_precision(models[e], c->instr[e]);
    if (m.precision == SAS_FP64) c->precision = SAS_FP64;
    fill_model(m, P, c->h_tab);
    if (m.sq_kind == SAS_SQ_HAYTER_MSA) {
      std::string why;
      size_t off = 0;
      sas_status st = fill_msa(m, c->instr[e], c->h_tab, &off, why);
      if (st != SAS_OK) return fail(c, st, "experiment " + std::to_string(e) + ": " + why);
      msa_offsets.push_back(std::make_pair(e, off));
    }
    P.lam_small = 0;
    if (m.model == SAS_CYLINDER) {
      // largest Lambda argument this experiment can produce: |Q| <= q_max, radius <= largest node
      double r_max = 0.0;
      for (int a = 0; a < P.n_a; ++a) r_max = std::max(r_max, c->h_tab[P.tab_off + a * TA_W] + c->h_tab[P.tab_off + a * TA_W + 1]);
      // ... and a detected neutron has sin(theta) = q lambda / 4 pi <= s_cut (the classifier's bound)
      double q_top = c->instr[e].q_max;
      if (std::isfinite(P.s_cut)) q_top = std::min(q_top, 4.0 * PI_D * P.s_cut / c->instr[e].lambda_min);
      const double x_max = q_top * r_max * 1.001;
      const double x2 = x_max * x_max;
      P.lam_small = x2 <= 16.0 ? 4 : x2 <= 25.0 ? 3 : x2 <= 36.0 ? 2 : x2 <= 64.0 ? 1 : 0;
    }
    c->tab_len_max = std::max(c->tab_len_max, P.tab_len);
  }
  // kernel variant of every experiment, and the launch groups
  for (auto& g : c->group_ids) g.clear();
  for (uint32_t e = 0; e < c->n_exp; ++e) {
    const ExpParams& P = c->h_exps[e];
    const int v = (P.model == SAS_CYLINDER && P.orient_kind == SAS_ORIENT_GAUSS_QUAD) ? (int)V_CYL_QUAD
                  : P.model >= SAS_PARALLELEPIPED ? (int)V_PARA + (P.model - SAS_PARALLELEPIPED) : P.model;
    const bool event = (P.pd_mc[0] | P.pd_mc[1]) != 0 && P.model != SAS_FLAT;
    c->group_ids[v + (event ? (int)N_VARIANTS : 0) + (c->exp_prec[e] == SAS_FP64 ? 2 * (int)N_VARIANTS : 0)].push_back(e);
  }
  for (int g = 0; g < N_GROUPS; ++g) {
    size_t n_heavy = 0;
    for (uint32_t e : c->group_ids[g]) n_heavy += consumer_bound(c->h_exps[e], c->exp_prec[e]) ? 1 : 0;
    c->group_heavy[g] = !c->group_ids[g].empty() && 2 * n_heavy >= c->group_ids[g].size();
  }
  std::vector<uint32_t> ids;
  for (int v = 0; v < N_GROUPS; ++v) {
    c->group_off[v] = ids.size();
    ids.insert(ids.end(), c->group_ids[v].begin(), c->group_ids[v].end());
  }
  CUDA_TRY(c, cudaMemcpy(c->d_exp_ids, ids.data(), ids.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
  const size_t tb = c->h_tab.size() * sizeof(double);
  if (tb > c->d_tab_cap) {
    if (c->d_tab) { CUDA_TRY(c, cudaStreamSynchronize(c->stream)); CUDA_TRY(c, cudaFree(c->d_tab)); c->d_tab = nullptr; }
    CUDA_TRY(c, cudaMalloc(&c->d_tab, tb));
    c->d_tab_cap = tb;
  }
  for (const auto& mo : msa_offsets) c->h_exps[mo.first].msa_tab = c->d_tab + mo.second;
  // the host vectors stay alive in the context, so asynchronous copies from them are safe to order on
  // the stream; a later set_model first synchronises (below) before overwriting them
  CUDA_TRY(c, cudaMemcpyAsync(c->d_tab, c->h_tab.data(), tb, cudaMemcpyHostToDevice, c->stream));
  CUDA_TRY(c, cudaMemcpyAsync(c->d_exps, c->h_exps.data(), (size_t)c->n_exp * sizeof(ExpParams),
                              cudaMemcpyHostToDevice, c->stream));
  c->model_set = true;
  return SAS_OK;
}

// Which kernel serves a variant: the warp-specialised one (trace_kernel_ws.cuh) where the integer stages A/B0
// are a large share of the work (at most a few dozen node evaluations per detected neutron), the unified one
// (trace_kernel.cuh) where the node loops dominate and every resident warp should run them: the tilt quadrature
// of the cylinder (c2) and the core-shell triaxial ellipsoid (c3).  The NEXT-2 models are served by the
// warp-specialised kernel whatever their node counts: measured at 1e8 neutrons, one evaluation per neutron
// gains 20 % there (micelle 121 -> 145, parallelepiped 131 -> 159 G n/s, barbell per event 52 -> 57), 16 x 16 nodes
// of a core-shell cylinder lose 3 %.
#ifndef SAS_WS_VARIANTS
#define SAS_WS_VARIANTS (((1u << N_VARIANTS) - 1u) & ~((1u << V_CS_TRIAX) | (1u << V_CYL_QUAD)))
#endif
constexpr bool use_ws(int v) { return ((SAS_WS_VARIANTS >> v) & 1u) != 0; }

// occupancy and shared-memory opt-in of one kernel instantiation, asked from the runtime once per (kernel, smem)
struct KernelPlan { size_t smem = ~(size_t)0; int bps = 0; };

template <typename Real, int V, bool EV, int CWG>
sas_status launch(sas_ctx* c, KernelArgs& a) {
  const bool DUMP = a.d_pixel != nullptr;
  constexpr bool WS = use_ws(V);
  constexpr int BLOCK_THREADS = WS ? WsCfg<CWG>::THREADS : block_threads(V);
  constexpr int ROW_WARPS = WS ? WS_PAIRS : BLOCK_THREADS / 32;  // warps that share the rows of a work item
  const size_t smem = WS ? ws_smem_bytes<Real, CWG>(c->tab_len_max) : trace_smem_bytes<Real>(c->tab_len_max, BLOCK_THREADS / 32);
  void (*kern)(const KernelArgs);
  if constexpr (WS) kern = trace_kernel_ws<Real, V, EV, CWG>; else kern = trace_kernel<Real, V, EV>;
  if (smem > 227 * 1024) return fail(c, SAS_EINVAL, "quadrature tables do not fit in shared memory");
  static thread_local KernelPlan plan[8];  // per device ordinal
  KernelPlan& pl = plan[c->device & 7];
  if (pl.smem != smem) {
    CUDA_TRY(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int bps = 0;
    CUDA_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kern, BLOCK_THREADS, smem));
    if (bps < 1) return fail(c, SAS_ECUDA, "trace kernel does not fit on an SM");
    pl.smem = smem; pl.bps = bps;
  }
  const int bps = pl.bps;
  const uint64_t total = (uint64_t)a.n_per_exp * a.n_exp;
  const int grid_full = c->n_sm * bps;
  // work items: ~16 per resident block, up to 262144 ids each, multiple of 256 ids.  A launch too small for that
  // (fewer than 16 rows of 32 ids per warp and item) is cut into one item per resident block instead, so that a
  // 1e6-neutron launch fills the chip evenly with a single static item per block and no work-counter traffic.
  uint64_t item = total / ((uint64_t)grid_full * (uint64_t)SAS_ITEMS_PER_BLOCK);
  if (item < (uint64_t)SAS_MIN_ITEM / 4 * ROW_WARPS) item = std::max<uint64_t>((a.n_per_exp + (uint64_t)grid_full - 1) / grid_full, 256);
  item = std::min<uint64_t>(item, 262144);
  item = (item + 255) / 256 * 256;
  a.item_ids = (uint32_t)item;
  a.items_per_exp = (uint32_t)(((uint64_t)a.n_per_exp + item - 1) / item);
  const uint64_t n_items = (uint64_t)a.items_per_exp * a.n_exp;
  if (n_items >= 0xFFFFFFFFull) return fail(c, SAS_EINVAL, "too many work items in one launch");
  a.n_items = (uint32_t)n_items;
  a.tab_len_max = c->tab_len_max;
  const int grid = (int)std::min<uint64_t>((uint64_t)grid_full, n_items);
  a.work_base = c->work_base;
  a.use_exp0 = (!c->batch && c->n_exp == 1) ? 1 : 0;
  if (a.use_exp0) a.exp0 = c->h_exps[0];
  const bool timed = c->timing_on && !DUMP && c->n_timed < (uint64_t)MAX_TIMED;
  if (timed) {
    if (c->ev0.size() <= c->n_timed) {
      cudaEvent_t e0, e1;
      CUDA_TRY(c, cudaEventCreate(&e0));
      CUDA_TRY(c, cudaEventCreate(&e1));
      c->ev0.push_back(e0);
      c->ev1.push_back(e1);
    }
    CUDA_TRY(c, cudaEventRecord(c->ev0[c->n_timed], c->stream));
  }
  // Programmatic stream serialisation: when the previous operation of the stream is a kernel, this one may be
  // scheduled as soon as every block of that kernel has exited or released its dependents (the zeroing kernel of
  // sas_reset_detector does so at once), and waits for its completion (griddepcontrol.wait) only where it first
  // needs the detector, the counters or the work counter: block set-up and the first Philox rows overlap the
  // zeroing and the launch latency.
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3((unsigned)grid);
  lc.blockDim = dim3((unsigned)BLOCK_THREADS);
  lc.dynamicSmemBytes = smem;
  lc.stream = c->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = SAS_PDL;
  lc.attrs = at;
  lc.numAttrs = 1;
  CUDA_TRY(c, cudaLaunchKernelEx(&lc, kern, a));
  CUDA_TRY(c, cudaGetLastError());
  if (n_items > (uint64_t)grid) c->work_base += (uint32_t)n_items;  // the fetches this launch makes (sas_types.h)
  if (timed) {
    CUDA_TRY(c, cudaEventRecord(c->ev1[c->n_timed], c->stream));
    sas_launch_record r;
    r.variant = V; r.per_event = EV ? 1 : 0; r.precision = sizeof(Real) == 8 ? SAS_FP64 : SAS_FP32;
    r.warp_specialised = WS ? 1 : 0; r.n_exp = a.n_exp; r.n_per_exp = a.n_per_exp; r.grid = grid; r.block = BLOCK_THREADS;
    r.ms = 0.0;
    if (c->records.size() <= c->n_timed) c->records.resize(c->n_timed + 1);
    c->records[c->n_timed] = r;
    c->n_timed += 1;
  }
  c->n_launches += 1;
  c->last_grid = grid; c->last_block = BLOCK_THREADS; c->last_smem = (int)smem;
  return SAS_OK;
}

// The warp-specialised kernel in the split the group asks for: the fp64 instantiations exist in both splits
// (consumer_bound), everything else in the default one only.
template <typename Real, int V, bool EV>
sas_status launch_split(sas_ctx* c, KernelArgs& a, bool heavy) {
  if constexpr (use_ws(V) && sizeof(Real) == 8 && V != V_FLAT) {
    if (heavy) return launch<Real, V, EV, SAS_WS_CWG_HEAVY>(c, a);
  }
  return launch<Real, V, EV, SAS_WS_CWG>(c, a);
}

// one launch of the kernel compiled for group g (variant, fixed-node or per-event sizes) over its experiments
template <typename Real, bool EV>
sas_status launch_variant(sas_ctx* c, KernelArgs& a, int v, int g) {
  a.exp_ids = c->d_exp_ids + c->group_off[g];
  a.n_exp = (uint32_t)c->group_ids[g].size();
  const bool heavy = c->group_heavy[g];
  switch (v) {
    case V_SPHERE: return launch_split<Real, V_SPHERE, EV>(c, a, heavy);
    case V_CS_SPHERE: return launch_split<Real, V_CS_SPHERE, EV>(c, a, heavy);
    case V_CYL: return launch_split<Real, V_CYL, EV>(c, a, heavy);
    case V_TRIAX: return launch_split<Real, V_TRIAX, EV>(c, a, heavy);
    case V_CS_TRIAX: return launch_split<Real, V_CS_TRIAX, EV>(c, a, heavy);
    case V_FLAT: return launch_split<Real, V_FLAT, false>(c, a, heavy);
    case V_CYL_QUAD: return launch_split<Real, V_CYL_QUAD, false>(c, a, heavy);
    case V_PARA: return launch_split<double, V_PARA, EV>(c, a, heavy);
    case V_CS_CYL: return launch_split<double, V_CS_CYL, EV>(c, a, heavy);
    case V_ELL: return launch_split<double, V_ELL, EV>(c, a, heavy);
    case V_BARBELL: return launch_split<double, V_BARBELL, EV>(c, a, heavy);
    case V_CAPPED: return launch_split<double, V_CAPPED, EV>(c, a, heavy);
    case V_ELL_CYL: return launch_split<double, V_ELL_CYL, EV>(c, a, heavy);
    case V_HOLLOW_CYL: return launch_split<double, V_HOLLOW_CYL, EV>(c, a, heavy);
    case V_CS_ELL: return launch_split<double, V_CS_ELL, EV>(c, a, heavy);
    case V_MICELLE: return launch_split<double, V_MICELLE, EV>(c, a, heavy);
    case V_HOLLOW_PRISM: return launch_split<double, V_HOLLOW_PRISM, EV>(c, a, heavy);
    default: return fail(c, SAS_EINVAL, "unknown kernel variant");
  }
}

sas_status launch_groups(sas_ctx* c, KernelArgs& a) {
  for (int g = 0; g < N_GROUPS; ++g) {
    if (c->group_ids[g].empty()) continue;
    const int v = g % N_VARIANTS;
    const bool event = (g / N_VARIANTS) & 1, fp64 = g >= 2 * N_VARIANTS;
    sas_status st;
    if (event) st = launch_variant<double, true>(c, a, v, g);  // effective_precision: always fp64
    else st = fp64 ? launch_variant<double, false>(c, a, v, g) : launch_variant<float, false>(c, a, v, g);
    if (st != SAS_OK) return st;
  }
  return SAS_OK;
}

// ids one launch may take from `first`: at most 2^31, at most n, and up to the next multiple of 2^32
uint64_t launch_span(uint64_t first, uint64_t n) {
  const uint64_t to_boundary = (1ull << 32) - (first & 0xFFFFFFFFull);
  return std::min<uint64_t>(std::min<uint64_t>(n, 1ull << 31), to_boundary);
}

sas_status trace_common(sas_ctx* c, uint64_t first_id, uint64_t n_each, uint64_t seed) {
  if (!c) return SAS_EINVAL;
  if (!c->model_set) return fail(c, SAS_ESTATE, "sas_set_model must precede tracing");
  if (n_each == 0) return SAS_OK;
  if (first_id + n_each < first_id) return fail(c, SAS_EINVAL, "neutron id range overflows 64 bits");
  { sas_status st = ensure_hist(c); if (st != SAS_OK) return st; }
  KernelArgs a;
  std::memset(&a, 0, sizeof(a));
  a.exps = c->d_exps; a.tab_pool = c->d_tab;
  a.sum_p = c->d_sum_p; a.sum_p2 = c->d_sum_p2; a.counts = c->d_counts;
  a.counters = c->d_counters; a.work_counter = c->d_work;
  a.n_exp = c->n_exp; a.exp_base = 0; a.npix = c->npix;
  philox_make_keys(seed, a.keys);
  // one launch covers at most 2^31 ids per experiment (32-bit id offsets inside the kernel) and never crosses a
  // multiple of 2^32 (the kernel keeps the high Philox counter word of the ids as one number per launch)
  for (uint64_t done = 0; done < n_each;) {
    a.first_id = first_id + done;
    a.n_per_exp = (uint32_t)launch_span(a.first_id, n_each - done);
    sas_status st = launch_groups(c, a);
    if (st != SAS_OK) return st;
    c->launched += (uint64_t)a.n_per_exp * c->n_exp;
    done += a.n_per_exp;
  }
  return SAS_OK;
}

void destroy_ctx(sas_ctx* c) {
  if (!c) return;
  DeviceGuard g(c);
  if (c->stream) cudaStreamSynchronize(c->stream);
  for (auto e : c->ev0) cudaEventDestroy(e);
  for (auto e : c->ev1) cudaEventDestroy(e);
  if (c->own_hist) { cudaFree(c->d_sum_p); cudaFree(c->d_sum_p2); cudaFree(c->d_counts); }
  cudaFree(c->d_counters); cudaFree(c->d_work); cudaFree(c->d_exp_ids); cudaFree(c->d_rings); cudaFree(c->d_exps); cudaFree(c->d_tab);
  if (c->own_stream && c->stream) cudaStreamDestroy(c->stream);
  delete c;
}

}  // namespace

// ===================================================================== the ABI
// for the entry points that live in other translation units and have no context (reduce_static.cu): the message
// sas_last_error(NULL) returns
namespace sas {
void set_global_error(const std::string& msg) { g_create_error = msg; }
}  // namespace sas

extern "C" {

const char* sas_version(void) { return "sas_b200 0.1 (sm_100a)"; }

const char* sas_last_error(const sas_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

sas_status sas_quadrature_nodes(int32_t kind, double param, int32_t n, double* h_values, double* h_weights) {
  if (!h_values || !h_weights || n < 1 || n > SAS_MAX_NODES || !(param >= 0.0)) return fail(nullptr, SAS_EINVAL, "bad sas_quadrature_nodes argument");
  std::vector<double> x, w;
  if (kind == 0) {
    if (!(param < 1.0)) return fail(nullptr, SAS_EINVAL, "Schulz relative width must be < 1");
    schulz_rule(param, n, x, w);
  } else if (kind == 1) {
    gauss_tilt_rule(param, n, x, w);
  } else {
    return fail(nullptr, SAS_EINVAL, "unknown quadrature kind");
  }
  // degenerate rules collapse to one node; pad so that the caller always gets n entries
  for (int i = 0; i < n; ++i) {
    h_values[i] = i < (int)x.size() ? x[i] : x[0];
    h_weights[i] = i < (int)w.size() ? w[i] : 0.0;
  }
  return SAS_OK;
}

sas_status sas_create_instrument(const sas_instrument_desc* instr, sas_ctx** out) {
  if (!out) return fail(nullptr, SAS_EINVAL, "out is NULL");
  std::string why;
  sas_status st = validate_instrument(instr, why);
  if (st != SAS_OK) return fail(nullptr, st, why);
  sas_ctx* c = new (std::nothrow) sas_ctx();
  if (!c) return fail(nullptr, SAS_ENOMEM, "out of host memory");
  c->n_exp = 1; c->batch = false;
  c->nx = instr->det_nx; c->ny = instr->det_ny; c->npix = c->nx * c->ny;
  c->instr.assign(1, *instr);
  c->h_exps.assign(1, ExpParams());
  std::memset(c->h_exps.data(), 0, sizeof(ExpParams));
  st = alloc_common(c);
  if (st != SAS_OK) { g_create_error = c->err; destroy_ctx(c); return st; }
  *out = c;
  return SAS_OK;
}

sas_status sas_create_batch(const sas_instrument_desc* instr, const sas_model_desc* model, uint32_t n_exp, sas_ctx** out) {
  if (!out || !instr || !model || n_exp == 0) return fail(nullptr, SAS_EINVAL, "bad sas_create_batch argument");
  std::string why;
  for (uint32_t e = 0; e < n_exp; ++e) {
    sas_status st = validate_instrument(instr + e, why);
    if (st == SAS_OK) st = validate_model(model + e, why);
    if (st == SAS_OK && (instr[e].det_nx != instr[0].det_nx || instr[e].det_ny != instr[0].det_ny)) { st = SAS_EINVAL; why = "all experiments of a batch need the same det_nx, det_ny"; }
    if (st != SAS_OK) return fail(nullptr, st, "experiment " + std::to_string(e) + ": " + why);
  }
  sas_ctx* c = new (std::nothrow) sas_ctx();
  if (!c) return fail(nullptr, SAS_ENOMEM, "out of host memory");
  c->n_exp = n_exp; c->batch = true;
  c->nx = instr[0].det_nx; c->ny = instr[0].det_ny; c->npix = c->nx * c->ny;
  c->instr.assign(instr, instr + n_exp);
  c->h_exps.assign(n_exp, ExpParams());
  std::memset(c->h_exps.data(), 0, sizeof(ExpParams) * n_exp);
  sas_status st = alloc_common(c);
  if (st == SAS_OK) st = upload_models(c, model);
  if (st != SAS_OK) { g_create_error = c->err; destroy_ctx(c); return st; }
  *out = c;
  return SAS_OK;
}

sas_status sas_bind_buffers(sas_ctx* c, void* d_sum_p, void* d_sum_p2, void* d_counts, void* cuda_stream) {
  if (!c) return SAS_EINVAL;
  DeviceGuard g(c);
  if (!d_sum_p || !d_sum_p2 || !d_counts) return fail(c, SAS_EINVAL, "histogram pointers must not be NULL");
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (c->own_hist) { cudaFree(c->d_sum_p); cudaFree(c->d_sum_p2); cudaFree(c->d_counts); }
  c->d_sum_p = (double*)d_sum_p; c->d_sum_p2 = (double*)d_sum_p2; c->d_counts = (unsigned long long*)d_counts;
  c->own_hist = false;
  if (c->own_stream && c->stream) cudaStreamDestroy(c->stream);
  c->stream = (cudaStream_t)cuda_stream;
  c->own_stream = false;
  // re-issue the uploads on the new stream so that ordering holds there
  if (c->model_set) {
    CUDA_TRY(c, cudaMemcpyAsync(c->d_tab, c->h_tab.data(), c->h_tab.size() * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_exps, c->h_exps.data(), (size_t)c->n_exp * sizeof(ExpParams), cudaMemcpyHostToDevice, c->stream));
  }
  CUDA_TRY(c, cudaMemsetAsync(c->d_counters, 0, 8 * sizeof(unsigned long long), c->stream));
  c->launched = 0;
  return SAS_OK;
}

sas_status sas_set_model(sas_ctx* c, const sas_model_desc* model) {
  if (!c) return SAS_EINVAL;
  DeviceGuard g(c);
  if (c->batch) return fail(c, SAS_ESTATE, "batched contexts take their models at sas_create_batch");
  std::string why;
  sas_status st = validate_model(model, why);
  if (st != SAS_OK) return fail(c, st, why);
  // pending asynchronous uploads read the host vectors we are about to rewrite
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return upload_models(c, model);
}

sas_status sas_trace(sas_ctx* c, uint64_t n_neutrons, uint64_t seed) {
  if (c && c->batch) return fail(c, SAS_ESTATE, "use sas_trace_batch on a batched context");
  DeviceGuard g(c);
  return trace_common(c, 0, n_neutrons, seed);
}

sas_status sas_trace_range(sas_ctx* c, uint64_t first_id, uint64_t n, uint64_t seed) {
  if (c && c->batch) return fail(c, SAS_ESTATE, "use sas_trace_batch on a batched context");
  DeviceGuard g(c);
  return trace_common(c, first_id, n, seed);
}

sas_status sas_trace_batch(sas_ctx* c, uint64_t n_neutrons_each, uint64_t seed) {
  if (c && !c->batch) return fail(c, SAS_ESTATE, "sas_trace_batch needs a context from sas_create_batch");
  DeviceGuard g(c);
  return trace_common(c, 0, n_neutrons_each, seed);
}

sas_status sas_trace_batch_range(sas_ctx* c, uint64_t first_id, uint64_t n_each, uint64_t seed) {
  if (c && !c->batch) return fail(c, SAS_ESTATE, "sas_trace_batch_range needs a context from sas_create_batch");
  DeviceGuard g(c);
  return trace_common(c, first_id, n_each, seed);
}

sas_status sas_get_launch_records(sas_ctx* c, sas_launch_record* h_records, uint32_t cap, uint32_t* n) {
  if (!c || !n || (cap && !h_records)) return SAS_EINVAL;
  DeviceGuard g(c);
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  for (uint64_t i = 0; i < c->n_timed; ++i) {
    float ms = 0.f;
    CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev0[i], c->ev1[i]));
    c->records[i].ms = ms;
    if (i < cap) h_records[i] = c->records[i];
  }
  *n = (uint32_t)c->n_timed;
  return SAS_OK;
}

sas_status sas_trace_dump(sas_ctx* c, uint64_t first_id, uint64_t n, uint64_t seed, uint32_t exp_index,
                          int32_t* d_pixel, double* d_weight, double* d_q) {
  if (!c) return SAS_EINVAL;
  if (c->batch) return fail(c, SAS_ESTATE, "sas_trace_dump works on single-experiment contexts");
  DeviceGuard g(c);
  if (!c->model_set) return fail(c, SAS_ESTATE, "sas_set_model must precede tracing");
  if (!d_pixel || !d_weight) return fail(c, SAS_EINVAL, "d_pixel and d_weight must not be NULL");
  if (n == 0) return SAS_OK;
  if (n > (1ull << 31)) return fail(c, SAS_EINVAL, "sas_trace_dump handles at most 2^31 ids per call");
  KernelArgs a;
  std::memset(&a, 0, sizeof(a));
  a.exps = c->d_exps; a.tab_pool = c->d_tab;
  a.counters = c->d_counters; a.work_counter = c->d_work;
  a.d_pixel = d_pixel; a.d_weight = d_weight; a.d_q = d_q;
  a.n_exp = 1; a.exp_base = exp_index; a.npix = c->npix;
  philox_make_keys(seed, a.keys);
  CUDA_TRY(c, cudaMemsetAsync(d_pixel, 0xFF, n * sizeof(int32_t), c->stream));
  CUDA_TRY(c, cudaMemsetAsync(d_weight, 0, n * sizeof(double), c->stream));
  if (d_q) CUDA_TRY(c, cudaMemsetAsync(d_q, 0, n * sizeof(double), c->stream));
  for (uint64_t done = 0; done < n;) {
    a.first_id = first_id + done;
    a.n_per_exp = (uint32_t)launch_span(a.first_id, n - done);
    a.d_pixel = d_pixel + done; a.d_weight = d_weight + done; a.d_q = d_q ? d_q + done : nullptr;
    sas_status st = launch_groups(c, a);
    if (st != SAS_OK) return st;
    done += a.n_per_exp;
  }
  return SAS_OK;
}

sas_status sas_read_detector(sas_ctx* c, double* h_sum_p, double* h_sum_p2, uint64_t* h_counts) {
  if (!c) return SAS_EINVAL;
  DeviceGuard g(c);
  { sas_status st = ensure_hist(c); if (st != SAS_OK) return st; }
  const size_t nh = (size_t)c->n_exp * c->npix;
  if (h_sum_p) CUDA_TRY(c, cudaMemcpyAsync(h_sum_p, c->d_sum_p, nh * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  if (h_sum_p2) CUDA_TRY(c, cudaMemcpyAsync(h_sum_p2, c->d_sum_p2, nh * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  if (h_counts) CUDA_TRY(c, cudaMemcpyAsync(h_counts, c->d_counts, nh * sizeof(uint64_t), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return SAS_OK;
}

sas_status sas_get_counters(sas_ctx* c, uint64_t out[8]) {
  if (!c || !out) return SAS_EINVAL;
  DeviceGuard g(c);
  CUDA_TRY(c, cudaMemcpyAsync(out, c->d_counters, 8 * sizeof(uint64_t), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  // the kernel counts the outcomes it decides in its queued stages (slots 2..7); launched is the host's
  // own sum of the traced ranges and every neutron has exactly one outcome, so slit 1 takes the rest
  out[0] = c->launched;
  uint64_t other = 0;
  for (int i = 2; i <= 6; ++i) other += out[i];
  out[1] = c->launched - other;
  return SAS_OK;
}

sas_status sas_reset_detector(sas_ctx* c) {
  if (!c) return SAS_EINVAL;
  DeviceGuard g(c);
  { sas_status st = ensure_hist(c); if (st != SAS_OK) return st; }
  const size_t nh = (size_t)c->n_exp * c->npix;
  // one launch for the three histograms and the counters (four memsets cost four stream operations: as much as
  // the trace kernel itself at 1e6 neutrons)
  const int grid = (int)std::max<size_t>(1, std::min<size_t>((size_t)c->n_sm * 8, (nh + 255) / 256));
  zero_detector_kernel<<<grid, 256, 0, c->stream>>>(reinterpret_cast<unsigned long long*>(c->d_sum_p),
                                                    reinterpret_cast<unsigned long long*>(c->d_sum_p2), c->d_counts,
                                                    c->d_counters, nh);
  CUDA_TRY(c, cudaGetLastError());
  c->launched = 0;
  return SAS_OK;
}

sas_status sas_get_launch_info(sas_ctx* c, uint64_t* n_launches, int32_t* grid, int32_t* block, int32_t* smem_bytes) {
  if (!c) return SAS_EINVAL;
  if (n_launches) *n_launches = c->n_launches;
  if (grid) *grid = c->last_grid;
  if (block) *block = c->last_block;
  if (smem_bytes) *smem_bytes = c->last_smem;
  return SAS_OK;
}

sas_status sas_set_launch_timing(sas_ctx* c, int32_t enabled) {
  if (!c) return SAS_EINVAL;
  c->timing_on = enabled != 0;
  return SAS_OK;
}

sas_status sas_get_kernel_time(sas_ctx* c, int32_t reset, double* avg_ms, uint64_t* n_timed) {
  if (!c) return SAS_EINVAL;
  DeviceGuard g(c);
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  double sum = 0.0;
  for (uint64_t i = 0; i < c->n_timed; ++i) {
    float ms = 0.f;
    CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev0[i], c->ev1[i]));
    sum += ms;
  }
  if (avg_ms) *avg_ms = c->n_timed ? sum / (double)c->n_timed : 0.0;
  if (n_timed) *n_timed = c->n_timed;
  if (reset) c->n_timed = 0;
  return SAS_OK;
}

sas_status sas_get_upload_bytes(sas_ctx* c, uint64_t* bytes) {
  if (!c || !bytes) return SAS_EINVAL;
  *bytes = c->h_tab.size() * sizeof(double) + (uint64_t)c->n_exp * sizeof(ExpParams);
  return SAS_OK;
}

sas_status sas_reduce_radial(sas_ctx* c, const sas_radial_desc* d, double* h_q, double* h_I, double* h_sigma,
                             uint64_t* h_npix) {
  if (!c) return SAS_EINVAL;
  DeviceGuard g(c);
  if (!d || d->struct_size != sizeof(sas_radial_desc)) return fail(c, SAS_EINVAL, "sas_radial_desc.struct_size mismatch");
  if (d->n_bins < 1 || d->n_bins > SAS_MAX_RINGS) return fail(c, SAS_EINVAL, "n_bins must be in 1..SAS_MAX_RINGS");
  if (!(d->q_hi > d->q_lo) || !(d->q_lo >= 0.0) || !std::isfinite(d->q_hi)) return fail(c, SAS_EINVAL, "need 0 <= q_lo < q_hi");
  if (!(d->lambda_ref > 0.0) || !std::isfinite(d->lambda_ref)) return fail(c, SAS_EINVAL, "lambda_ref must be > 0");
  if (d->exp_index >= c->n_exp) return fail(c, SAS_EINVAL, "exp_index out of range");
  { sas_status st = ensure_hist(c); if (st != SAS_OK) return st; }
  const int nb = d->n_bins;
  // ring scratch: sum P, sum P2, sum dOmega, pixel count, nb entries each (one memset, one copy of what is used)
  if (!c->d_rings) CUDA_TRY(c, cudaMalloc(&c->d_rings, 4 * (size_t)SAS_MAX_RINGS * sizeof(double)));
  CUDA_TRY(c, cudaMemsetAsync(c->d_rings, 0, 4 * (size_t)nb * sizeof(double), c->stream));
  const sas_instrument_desc& ins = c->instr[d->exp_index];
  ReduceArgs a;
  a.sum_p = c->d_sum_p + (size_t)d->exp_index * c->npix;
  a.sum_p2 = c->d_sum_p2 + (size_t)d->exp_index * c->npix;
  a.ring_p = c->d_rings;
  a.ring_p2 = c->d_rings + nb;
  a.ring_omega = c->d_rings + 2 * nb;
  a.ring_n = reinterpret_cast<unsigned long long*>(c->d_rings + 3 * nb);
  a.det_xw = ins.det_xw; a.det_yh = ins.det_yh; a.det_dist = ins.det_dist;
  a.px = ins.det_xw / (double)ins.det_nx; a.py = ins.det_yh / (double)ins.det_ny;
  a.a_pix_d = (a.px * a.py) * ins.det_dist;
  a.two_k = 2.0 * (TWO_PI / d->lambda_ref);
  a.q_lo = d->q_lo; a.q_hi = d->q_hi; a.scale = (double)nb / (d->q_hi - d->q_lo);
  a.nx = ins.det_nx; a.ny = ins.det_ny; a.n_bins = nb;
  const int grid = std::max(1, std::min(c->n_sm * 4, (c->npix + REDUCE_THREADS - 1) / REDUCE_THREADS));
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  CUDA_TRY(c, cudaEventCreate(&e0));
  CUDA_TRY(c, cudaEventCreate(&e1));
  CUDA_TRY(c, cudaEventRecord(e0, c->stream));
  reduce_radial_kernel<<<grid, REDUCE_THREADS, 0, c->stream>>>(a);
  CUDA_TRY(c, cudaGetLastError());
  CUDA_TRY(c, cudaEventRecord(e1, c->stream));
  c->n_launches += 1;
  std::vector<double> h(4 * (size_t)nb);
  CUDA_TRY(c, cudaMemcpyAsync(h.data(), c->d_rings, h.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  c->last_reduce_ms = ms;
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  const unsigned long long* hn = reinterpret_cast<const unsigned long long*>(h.data() + 3 * nb);
  // neutrons launched into this experiment: the caller's figure, else this context's own count (every experiment
  // of a context traces the same ids)
  const double launched = d->n_launched ? (double)d->n_launched : (double)(c->launched / c->n_exp);
  for (int b = 0; b < nb; ++b) {
    if (h_q) h_q[b] = d->q_lo + ((double)b + 0.5) * ((d->q_hi - d->q_lo) / (double)nb);
    const double norm = h[2 * nb + b] * launched;
    const bool any = hn[b] != 0 && norm > 0.0;
    if (h_I) h_I[b] = any ? h[b] / norm : 0.0;
    if (h_sigma) h_sigma[b] = any ? std::sqrt(h[nb + b]) / norm : 0.0;
    if (h_npix) h_npix[b] = hn[b];
  }
  return SAS_OK;
}

sas_status sas_get_reduce_time(sas_ctx* c, double* ms) {
  if (!c || !ms) return SAS_EINVAL;
  *ms = c->last_reduce_ms;
  return SAS_OK;
}

void sas_destroy(sas_ctx* c) { destroy_ctx(c); }

}  // extern "C"
