// sas_reduce_radial_static (include/sas.h): the ring average of a detector image (DESIGN.md R-R1)
// for callers that must not allocate: CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
// Same arithmetic as sas_reduce_radial (reduce_kernel.cuh + the host normalisation of sas_api.cu), but
//   - the ring scratch (sum P, sum P2, sum dOmega, pixel count per ring) is the file-scope device array
//     g_ring_scratch below, SAS_STATIC_MAX_RINGS rings = 16 KB, held by every GPU that loads the library until exit;
//   - inputs and outputs are the caller's DEVICE buffers; the normalisation runs in a second kernel;
//   - the call makes no cudaMalloc / cudaFree / event creation / synchronisation: one cudaMemsetAsync and two kernel
//     launches on the caller's stream.
// Every call on a device shares the array (it keeps the last call's contents: each call clears the part it uses
// first, in stream order): two calls that overlap on the GPU -- different streams, no dependency -- race.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <mutex>
#include <string>

#include <cuda_runtime.h>

#include "../../include/sas.h"

namespace sas {
void set_global_error(const std::string& msg);   // sas_api.cu: the message sas_last_error(NULL) returns

namespace {

constexpr int RS_THREADS = 256;
constexpr double RS_TWO_PI = 6.283185307179586;

// [0, n): sum P   [n, 2n): sum P2   [2n, 3n): sum dOmega   [3n, 4n): pixels (as unsigned long long), n = n_bins.
// In host code this name is only a handle for cudaGetSymbolAddress, never a device address.
static __device__ __align__(256) double g_ring_scratch[4 * SAS_STATIC_MAX_RINGS];

struct StaticReduceArgs {
  const double* sum_p;       // [ny][nx], device
  const double* sum_p2;
  double* scratch;           // device address of g_ring_scratch on the launching device
  double det_xw, det_yh, det_dist, px, py, a_pix_d;
  double two_k, q_lo, q_hi, scale;
  int32_t nx, ny, n_bins;
};

// the scratch-using kernel: reduce_radial_kernel's pass (one thread per pixel, per-block ring sums in shared
// memory, one pass of global reductions per block) accumulating into the static array
__global__ void __launch_bounds__(RS_THREADS) reduce_radial_static_kernel(const __grid_constant__ StaticReduceArgs a) {
  __shared__ double s_p[SAS_STATIC_MAX_RINGS], s_p2[SAS_STATIC_MAX_RINGS], s_om[SAS_STATIC_MAX_RINGS];
  __shared__ unsigned int s_n[SAS_STATIC_MAX_RINGS];
  for (int b = threadIdx.x; b < a.n_bins; b += RS_THREADS) { s_p[b] = 0.0; s_p2[b] = 0.0; s_om[b] = 0.0; s_n[b] = 0u; }
  __syncthreads();
  const int npix = a.nx * a.ny;
  for (int pix = blockIdx.x * RS_THREADS + threadIdx.x; pix < npix; pix += gridDim.x * RS_THREADS) {
    const int iy = pix / a.nx, ix = pix - iy * a.nx;
    // R-R1, operation by operation (compiled without FMA contraction, like the rest of the library)
    const double X = ((double)ix + 0.5) * a.px - 0.5 * a.det_xw;
    const double Y = ((double)iy + 0.5) * a.py - 0.5 * a.det_yh;
    const double r2 = X * X + Y * Y;
    const double two_theta = atan2(sqrt(r2), a.det_dist);
    const double q = a.two_k * sin(0.5 * two_theta);
    if (!(q >= a.q_lo && q < a.q_hi)) continue;
    const int b = (int)floor((q - a.q_lo) * a.scale);
    if (b < 0 || b >= a.n_bins) continue;
    const double d2 = a.det_dist * a.det_dist + r2;
    const double dOmega = a.a_pix_d / (d2 * sqrt(d2));
    atomicAdd(&s_p[b], a.sum_p[pix]);
    atomicAdd(&s_p2[b], a.sum_p2[pix]);
    atomicAdd(&s_om[b], dOmega);
    atomicAdd(&s_n[b], 1u);
  }
  __syncthreads();
  const int n = a.n_bins;
  for (int b = threadIdx.x; b < n; b += RS_THREADS) {
    if (s_n[b] == 0u) continue;
    atomicAdd(a.scratch + b, s_p[b]);
    atomicAdd(a.scratch + n + b, s_p2[b]);
    atomicAdd(a.scratch + 2 * n + b, s_om[b]);
    atomicAdd(reinterpret_cast<unsigned long long*>(a.scratch + 3 * n) + b, (unsigned long long)s_n[b]);
  }
}

// the normalisation sas_reduce_radial does on the host, ring by ring, into the caller's device buffers
__global__ void __launch_bounds__(RS_THREADS) finish_radial_static_kernel(const double* scratch, int n, double q_lo, double q_hi,
                                                                          double launched, double* q, double* I,
                                                                          double* sigma, unsigned long long* npix) {
  const int b = blockIdx.x * RS_THREADS + threadIdx.x;
  if (b >= n) return;
  const unsigned long long cnt = reinterpret_cast<const unsigned long long*>(scratch + 3 * n)[b];
  const double norm = scratch[2 * n + b] * launched;
  const bool any = cnt != 0ull && norm > 0.0;
  if (q) q[b] = q_lo + ((double)b + 0.5) * ((q_hi - q_lo) / (double)n);
  if (I) I[b] = any ? scratch[b] / norm : 0.0;
  if (sigma) sigma[b] = any ? sqrt(scratch[n + b]) / norm : 0.0;
  if (npix) npix[b] = cnt;
}

// set-up, once per device, with that device current: the device address of the array and the SM count
constexpr int RS_MAX_DEVICES = 64;
struct DeviceSlot { bool ready = false; double* scratch = nullptr; int n_sm = 0; };
DeviceSlot g_slots[RS_MAX_DEVICES];
std::mutex g_slots_mutex;

sas_status fail_static(sas_status st, const std::string& msg) {
  set_global_error(msg);
  return st;
}

sas_status slot_of_current_device(DeviceSlot** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail_static(SAS_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= RS_MAX_DEVICES) return fail_static(SAS_EUNSUPPORTED, "sas_reduce_radial_static: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_slots_mutex);
  DeviceSlot& s = g_slots[dev];
  if (!s.ready) {
    double* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_ring_scratch);   // of the CURRENT device's copy of the array
    if (e != cudaSuccess || !ptr) return fail_static(SAS_ECUDA, std::string("cudaGetSymbolAddress(g_ring_scratch): ") + cudaGetErrorString(e));
    int n_sm = 0;
    e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess || n_sm < 1) return fail_static(SAS_ECUDA, std::string("cudaDeviceGetAttribute: ") + cudaGetErrorString(e));
    s.scratch = ptr; s.n_sm = n_sm; s.ready = true;
  }
  *out = &s;
  return SAS_OK;
}

}  // namespace
}  // namespace sas

using namespace sas;

extern "C" sas_status sas_reduce_radial_static(const sas_instrument_desc* ins, const sas_radial_desc* d,
                                               const double* d_sum_p, const double* d_sum_p2, double* d_q, double* d_I,
                                               double* d_sigma, uint64_t* d_npix, void* stream) {
  if (!ins || ins->struct_size != sizeof(sas_instrument_desc)) return fail_static(SAS_EINVAL, "sas_instrument_desc.struct_size mismatch");
  if (!d || d->struct_size != sizeof(sas_radial_desc)) return fail_static(SAS_EINVAL, "sas_radial_desc.struct_size mismatch");
  if (!d_sum_p || !d_sum_p2) return fail_static(SAS_EINVAL, "sas_reduce_radial_static: d_sum_p and d_sum_p2 must be device buffers");
  if (d->n_bins < 1) return fail_static(SAS_EINVAL, "n_bins must be >= 1");
  if (d->n_bins > SAS_STATIC_MAX_RINGS)
    return fail_static(SAS_EINVAL, "sas_reduce_radial_static: n_bins = " + std::to_string(d->n_bins) + " exceeds SAS_STATIC_MAX_RINGS = " +
                                       std::to_string(SAS_STATIC_MAX_RINGS) + ", the size of the static ring scratch (use sas_reduce_radial)");
  if (!(d->q_hi > d->q_lo) || !(d->q_lo >= 0.0) || !std::isfinite(d->q_hi)) return fail_static(SAS_EINVAL, "need 0 <= q_lo < q_hi");
  if (!(d->lambda_ref > 0.0) || !std::isfinite(d->lambda_ref)) return fail_static(SAS_EINVAL, "lambda_ref must be > 0");
  if (d->n_launched == 0) return fail_static(SAS_EINVAL, "sas_reduce_radial_static: desc->n_launched must be given (there is no context to count for it)");
  if (ins->det_nx < 1 || ins->det_ny < 1 || (int64_t)ins->det_nx * ins->det_ny > (int64_t)1 << 30 || !(ins->det_xw > 0.0) || !(ins->det_yh > 0.0) ||
      !(ins->det_dist > 0.0) || !std::isfinite(ins->det_xw) || !std::isfinite(ins->det_yh) || !std::isfinite(ins->det_dist))
    return fail_static(SAS_EINVAL, "sas_reduce_radial_static: detector geometry of the instrument descriptor is not valid");
  DeviceSlot* slot = nullptr;
  { sas_status st = slot_of_current_device(&slot); if (st != SAS_OK) return st; }
  cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
  const int nb = d->n_bins;
  // the array keeps the previous call's sums: clear what this call accumulates into, in stream order
  cudaError_t e = cudaMemsetAsync(slot->scratch, 0, 4 * (size_t)nb * sizeof(double), s);
  if (e != cudaSuccess) return fail_static(SAS_ECUDA, std::string("cudaMemsetAsync: ") + cudaGetErrorString(e));
  StaticReduceArgs a;
  a.sum_p = d_sum_p; a.sum_p2 = d_sum_p2; a.scratch = slot->scratch;
  a.det_xw = ins->det_xw; a.det_yh = ins->det_yh; a.det_dist = ins->det_dist;
  a.px = ins->det_xw / (double)ins->det_nx; a.py = ins->det_yh / (double)ins->det_ny;
  a.a_pix_d = (a.px * a.py) * ins->det_dist;
  a.two_k = 2.0 * (RS_TWO_PI / d->lambda_ref);
  a.q_lo = d->q_lo; a.q_hi = d->q_hi; a.scale = (double)nb / (d->q_hi - d->q_lo);
  a.nx = ins->det_nx; a.ny = ins->det_ny; a.n_bins = nb;
  const int npix = ins->det_nx * ins->det_ny;
  const int grid = std::max(1, std::min(slot->n_sm * 4, (npix + RS_THREADS - 1) / RS_THREADS));
  reduce_radial_static_kernel<<<grid, RS_THREADS, 0, s>>>(a);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail_static(SAS_ECUDA, std::string("reduce_radial_static_kernel: ") + cudaGetErrorString(e));
  finish_radial_static_kernel<<<(nb + RS_THREADS - 1) / RS_THREADS, RS_THREADS, 0, s>>>(
      slot->scratch, nb, d->q_lo, d->q_hi, (double)d->n_launched, d_q, d_I, d_sigma, reinterpret_cast<unsigned long long*>(d_npix));
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail_static(SAS_ECUDA, std::string("finish_radial_static_kernel: ") + cudaGetErrorString(e));
  return SAS_OK;
}
