// Ring average of one detector image into I(q) with its standard error (DESIGN.md R-R1).
// One thread per pixel (grid-stride), per-block partial sums of the rings in shared memory, one pass of global
// reductions per block: the image is read once (24 B per pixel), the rings are a few KB.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace sas {

struct ReduceArgs {
  const double* sum_p;                 // [ny][nx] of the chosen experiment
  const double* sum_p2;
  double* ring_p;                      // [n_bins] sum P
  double* ring_p2;                     // [n_bins] sum P2
  double* ring_omega;                  // [n_bins] sum of pixel solid angles
  unsigned long long* ring_n;          // [n_bins] pixels
  double det_xw, det_yh, det_dist, px, py, a_pix_d;  // pixel pitches, A_pix * D
  double two_k, q_lo, q_hi, scale;     // 2 k = 4 pi / lambda_ref; scale = n_bins / (q_hi - q_lo)
  int32_t nx, ny, n_bins;
};

constexpr int REDUCE_THREADS = 256;
constexpr int REDUCE_MAX_BINS = 1024;  // four shared-memory arrays of that many entries: 32 KB

__global__ void __launch_bounds__(REDUCE_THREADS) reduce_radial_kernel(const __grid_constant__ ReduceArgs a) {
  __shared__ double s_p[REDUCE_MAX_BINS], s_p2[REDUCE_MAX_BINS], s_om[REDUCE_MAX_BINS];
  __shared__ unsigned int s_n[REDUCE_MAX_BINS];
  for (int b = threadIdx.x; b < a.n_bins; b += REDUCE_THREADS) { s_p[b] = 0.0; s_p2[b] = 0.0; s_om[b] = 0.0; s_n[b] = 0u; }
  __syncthreads();
  const int npix = a.nx * a.ny;
  for (int pix = blockIdx.x * REDUCE_THREADS + threadIdx.x; pix < npix; pix += gridDim.x * REDUCE_THREADS) {
    const int iy = pix / a.nx, ix = pix - iy * a.nx;
    // R-R1, operation by operation (this translation unit is compiled without FMA contraction)
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
  for (int b = threadIdx.x; b < a.n_bins; b += REDUCE_THREADS) {
    if (s_n[b] == 0u) continue;
    atomicAdd(a.ring_p + b, s_p[b]);
    atomicAdd(a.ring_p2 + b, s_p2[b]);
    atomicAdd(a.ring_omega + b, s_om[b]);
    atomicAdd(a.ring_n + b, (unsigned long long)s_n[b]);
  }
}

}  // namespace sas
