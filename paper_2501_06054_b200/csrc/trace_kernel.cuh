// The trace kernel: persistent blocks pull work items (experiment, id range) from a global counter;
// inside a block every warp is autonomous and runs a four-stage pipeline with warp-private ring
// queues in shared memory so that each stage executes with full warps although ~75 % of the neutrons
// die at slit 1 and ~80 % of the rest miss the detector:
//
//   stage A  Philox block 0 + slit-1 test on the raw 32-bit draws      (every launched neutron)
//   stage B0 Philox block 1 + conservative "certain to miss the         (slit-1 survivors)
//            detector" test on q lambda (geometry.cuh)
//   stage B  Philox block 0 again, fp64 geometry: slits, sample       (survivors that may hit)
//            chord, Q, detector pixel
//   stage C  model intensity I(Q) with the quadrature node loops,      (detected neutrons)
//            weight, histogram update
#pragma once
#include "geometry.cuh"
#include "models.cuh"

namespace sas {

#ifndef SAS_STAGE_A_ROWS
#define SAS_STAGE_A_ROWS 3
#endif
#ifndef SAS_B0_PER_LANE
#define SAS_B0_PER_LANE 2
#endif
#ifndef SAS_BLOCK_THREADS
#define SAS_BLOCK_THREADS 128
#endif
#ifndef SAS_MIN_BLOCKS
#define SAS_MIN_BLOCKS 5
#endif
// Threads per block by kernel variant, always 20 resident warps per SM (96 registers).  The sphere kernels run
// one warp per block: no barrier at the work fetch (measured: c1 +3.8 %, c0 +1.2 %); the variants with large
// quadrature tables share them among four warps (c3 loses 3 % with private copies).
constexpr int RESIDENT_THREADS_PER_SM = SAS_BLOCK_THREADS * SAS_MIN_BLOCKS;
__host__ __device__ constexpr int block_threads(int variant) { return variant == V_SPHERE ? 32 : SAS_BLOCK_THREADS; }
constexpr int RING = 64;     // entries per warp queue (power of two, >= 63)
constexpr int NB0 = SAS_B0_PER_LANE;  // queue-B entries a lane takes per stage-B0 step
constexpr int RING_B2 = NB0 > 1 ? 128 : 64;
constexpr int RING_B = (32 * NB0 - 1 + 32 * SAS_STAGE_A_ROWS) > 128 ? 256 : 128;  // queue B takes SAS_STAGE_A_ROWS rows of 32 per stage-A step on top of < 32 entries

// a stage runs only while its input queue is below one batch, so the capacities below can never be exceeded
static_assert(RING_B >= 32 * NB0 - 1 + 32 * SAS_STAGE_A_ROWS, "queue B: < one B0 batch + one stage-A step");
static_assert(RING_B2 >= 31 + 32 * NB0, "queue B2: < 32 entries + one B0 batch");
static_assert(RING >= 31 + 32, "queue C: < 32 entries + one stage-B batch");
static_assert((RING & (RING - 1)) == 0 && (RING_B & (RING_B - 1)) == 0 && (RING_B2 & (RING_B2 - 1)) == 0, "ring sizes are powers of two");

struct WarpQueues {
  // queue B: slit-1 survivors (their id offsets; stage B draws Philox block 0 again for the few it gets:
  // 40 integer instructions for 6 % of the neutrons instead of eight queue accesses for 25 %)
  uint32_t b_id[RING_B];
  // queue B2: survivors the classifier could not rule out (id offset and Philox block 1)
  uint32_t b2_id[RING_B2];
  uint32_t b2_w[4][RING_B2];
  // queue C: detected neutrons
  uint32_t c_id[RING];
  int32_t c_pixel[RING];
  double c_G[RING];
  double c_Q[3][RING];
  // outcome counts of this warp, one column per lane (no conflicts, no overflow): row 0 detected,
  // rows 1..5 = ST_*, row 6 = detector misses decided by the classifier
  uint32_t oc[7][32];
};

__host__ __device__ inline size_t round16(size_t x) { return (x + 15) & ~(size_t)15; }

template <typename Real>
__host__ __device__ inline size_t trace_smem_bytes(int tab_len_max, int warps_per_block) {
  return round16(sizeof(ExpParams)) + round16((size_t)tab_len_max * sizeof(Real)) +
         (size_t)warps_per_block * sizeof(WarpQueues);
}

// adds a warp's outcome counts to the global counters: detected (row 0) to slot 6, ST_* rows 1..5 to
// slots 1..5; the classifier's detector misses (row 6) to slot 5 and to slot 7
__device__ __forceinline__ void flush_outcomes(unsigned long long* counters, const uint32_t (*oc)[32]) {
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int f = 0; f < 7; ++f) {
    const unsigned tot = __reduce_add_sync(0xFFFFFFFFu, oc[f][lane]);
    if (lane == 0 && tot) {
      atomicAdd(counters + (f == 0 ? 6 : (f == 6 ? 5 : f)), (unsigned long long)tot);
      if (f == 6) atomicAdd(counters + 7, (unsigned long long)tot);
    }
  }
}

// EV: the experiments of this launch sample their sizes per scattering event (SAS_PD_GAUSS_MC); those
// kernels exist in fp64 only and evaluate Eq. 4 once per detected neutron (models.cuh)
template <typename Real, int V, bool EV>
__global__ void __launch_bounds__(block_threads(V), RESIDENT_THREADS_PER_SM / block_threads(V))
trace_kernel(const __grid_constant__ KernelArgs a) {
  constexpr int BLOCK_THREADS = block_threads(V);
  constexpr int WARPS_PER_BLOCK = BLOCK_THREADS / 32;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ unsigned int s_item;

  ExpParams& P = *reinterpret_cast<ExpParams*>(smem_raw);
  Real* tab = reinterpret_cast<Real*>(smem_raw + round16(sizeof(ExpParams)));
  WarpQueues& wq = reinterpret_cast<WarpQueues*>(smem_raw + round16(sizeof(ExpParams)) +
                                                 round16((size_t)a.tab_len_max * sizeof(Real)))[threadIdx.x >> 5];
  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;
  const unsigned FULL = 0xFFFFFFFFu;
  const bool DUMP = a.d_pixel != nullptr;  // parity hook: per-neutron outputs instead of the histogram
  const bool DUMP_Q = DUMP && a.d_q != nullptr;
  // the host never lets a launch cross a multiple of 2^32 ids: the high counter word is one number per launch
  const uint32_t first_lo = (uint32_t)a.first_id, id_hi = (uint32_t)(a.first_id >> 32);

  // warp-uniform pipeline state
  int headB = 0, cntB = 0, headB2 = 0, cntB2 = 0, headC = 0, cntC = 0;
#pragma unroll
  for (int f = 0; f < 7; ++f) wq.oc[f][lane] = 0;
  // programmatic dependent launch (sas_api.cu: launch): the previous kernel of the stream is complete from here on
  asm volatile("griddepcontrol.wait;" ::: "memory");

  int cur_exp = -1;
  bool replay = false, first = true;
  unsigned item = blockIdx.x;  // the first item of a block is its own index (the host launches grid <= n_items)

  for (;;) {
    if (!replay && !first) {
      if (a.n_items <= gridDim.x) {
        item = a.n_items;      // every block had its one item: nothing to fetch
      } else {
        __syncthreads();  // everyone is done with s_item and with the staged experiment of the last pass
        if (threadIdx.x == 0) s_item = gridDim.x + (atomicAdd(a.work_counter, 1u) - a.work_base);
        __syncthreads();
        item = s_item;
      }
    }
    first = false;
    const bool have = item < a.n_items;
    const int e = have ? (a.use_exp0 ? a.exp0.exp_index : (int)a.exp_ids[item / a.items_per_exp]) : -1;
    const bool drain = (e != cur_exp) && (cur_exp >= 0) && !replay;
    uint32_t row = 0, row_end = 0, off0 = 0, cnt_ids = 0;
    if (drain) {
      replay = true;  // come back for this item after the queues are empty
    } else {
      replay = false;
      if (!have) break;
      if (e != cur_exp) {
        // stage the experiment: parameters and tables (fp64 in HBM -> Real in shared memory)
        __syncthreads();  // every warp has drained the previous experiment
        const ExpParams* src = a.use_exp0 ? &a.exp0 : a.exps + e;   // kernel arguments or HBM
        const uint32_t* s32 = reinterpret_cast<const uint32_t*>(src);
        uint32_t* d32 = reinterpret_cast<uint32_t*>(&P);
        for (int i = threadIdx.x; i < (int)(sizeof(ExpParams) / 4); i += BLOCK_THREADS) d32[i] = s32[i];
        const int tl = src->tab_len;
        SAS_CHECK(tl >= 0 && tl <= a.tab_len_max);
        const double* tsrc = a.tab_pool + src->tab_off;
        for (int i = threadIdx.x; i < tl; i += BLOCK_THREADS) tab[i] = (Real)tsrc[i];
        cur_exp = e;
        __syncthreads();
      }
      const uint32_t kk = item % a.items_per_exp;
      off0 = kk * a.item_ids;
      cnt_ids = min(a.item_ids, a.n_per_exp - off0);
      SAS_CHECK(item < a.n_items && off0 < a.n_per_exp);
      row = warp;
      row_end = (cnt_ids + 31u) >> 5;
    }

    // ------------------------------------------------------------------ the pump
    for (;;) {
      SAS_CHECK(cntB >= 0 && cntB <= RING_B && cntB2 >= 0 && cntB2 <= RING_B2 && cntC >= 0 && cntC <= RING);
      const bool rows_left = row < row_end;
      // Philox counter word 3 of the staged experiment (one add from a kernel parameter: not kept live)
      const uint32_t exp_word = a.exp_base + (uint32_t)cur_exp;
      if (cntC >= 32 || (drain && cntB == 0 && cntB2 == 0 && cntC > 0)) {
        // ---------------- stage C: model + weight + histogram
        const int n = cntC < 32 ? cntC : 32;
        const bool act = lane < n;
        const int slot = (headC + lane) & (RING - 1);
        uint32_t idoff = 0; int32_t pixel = 0; double G = 0, Qx = 0, Qy = 0, Qz = 0;
        if (act) {
          idoff = wq.c_id[slot]; pixel = wq.c_pixel[slot]; G = wq.c_G[slot];
          Qx = wq.c_Q[0][slot]; Qy = wq.c_Q[1][slot]; Qz = wq.c_Q[2][slot];
        }
        __syncwarp();
        headC = (headC + n) & (RING - 1);
        cntC -= n;
        if (act) {
          const uint32_t id_lo = first_lo + idoff;
          Real I;
          if (EV)
            I = (Real)eval_intensity_event<V>(P, a.keys, id_lo, id_hi, exp_word, Qx, Qy, Qz);
          else
            I = eval_intensity<Real, V>(P, tab, a.keys, id_lo, id_hi, exp_word, Qx, Qy, Qz);
          const double p = G * (double)I;
          if (DUMP) {
            a.d_pixel[idoff] = pixel;
            a.d_weight[idoff] = p;
          } else {
            SAS_CHECK(pixel >= 0 && pixel < a.npix && cur_exp >= 0);
            const size_t ix = (size_t)cur_exp * (size_t)a.npix + (size_t)pixel;
            atomicAdd(a.counts + ix, 1ull);
            atomicAdd(a.sum_p + ix, p);
            atomicAdd(a.sum_p2 + ix, p * p);
          }
        }
        continue;
      }
      if (cntB2 >= 32 || (drain && cntB == 0 && cntB2 > 0)) {
        // ---------------- stage B: fp64 geometry
        const int n = cntB2 < 32 ? cntB2 : 32;
        const bool act = lane < n;
        const int slot = (headB2 + lane) & (RING_B2 - 1);
        uint32_t idoff = 0, w[4] = {0, 0, 0, 0}, w1[4] = {0, 0, 0, 0};
        if (act) {
          idoff = wq.b2_id[slot];
#pragma unroll
          for (int i = 0; i < 4; ++i) w1[i] = wq.b2_w[i][slot];
        }
        {
          philox4x32_10(a.keys, first_lo + idoff, id_hi, 0u, exp_word, w);
        }
        __syncwarp();
        headB2 = (headB2 + n) & (RING_B2 - 1);
        cntB2 -= n;
        int st = -1;
        Hit h;
        if (act) {
          st = P.geo_fast ? trace_geometry<true>(P, w, w1, h) : trace_geometry<false>(P, w, w1, h);
          if (DUMP_Q) a.d_q[idoff] = h.q;
          wq.oc[st][lane] += 1;
        }
        const unsigned m = __ballot_sync(FULL, st == ST_DETECTED);
        if (st == ST_DETECTED) {
          const int s2 = (headC + cntC + __popc(m & lt_mask)) & (RING - 1);
          wq.c_id[s2] = idoff; wq.c_pixel[s2] = h.pixel; wq.c_G[s2] = h.G;
          wq.c_Q[0][s2] = h.Qx; wq.c_Q[1][s2] = h.Qy; wq.c_Q[2][s2] = h.Qz;
        }
        cntC += __popc(m);
        __syncwarp();
        continue;
      }
      if (cntB >= 32 * NB0 || (drain && cntB > 0)) {
        // ---------------- stage B0: Philox block 1 + certain-miss classifier, NB0 entries per lane
        // (independent Philox chains in flight, as in stage A)
        const int n = cntB < 32 * NB0 ? cntB : 32 * NB0;
        uint32_t idoff[NB0], w1[NB0][4];
        bool act[NB0];
#pragma unroll
        for (int k = 0; k < NB0; ++k) {
          act[k] = lane + 32 * k < n;
          idoff[k] = act[k] ? wq.b_id[(headB + lane + 32 * k) & (RING_B - 1)] : 0u;
        }
        __syncwarp();
        headB = (headB + n) & (RING_B - 1);
        cntB -= n;
#pragma unroll
        for (int k = 0; k < NB0; ++k) {
          philox4x32_10(a.keys, first_lo + idoff[k], id_hi, 1u, exp_word, w1[k]);
        }
        int tail = headB2 + cntB2;
#pragma unroll
        for (int k = 0; k < NB0; ++k) {
          double q;
          const bool sure = surely_misses_detector(P, w1[k], q);
          if (act[k] && sure) {
            wq.oc[6][lane] += 1;
            if (DUMP_Q) a.d_q[idoff[k]] = q;
          }
          const bool keep = act[k] && !sure;
          const unsigned m = __ballot_sync(FULL, keep);
          if (keep) {
            const int s2 = (tail + __popc(m & lt_mask)) & (RING_B2 - 1);
            wq.b2_id[s2] = idoff[k];
#pragma unroll
            for (int i = 0; i < 4; ++i) wq.b2_w[i][s2] = w1[k][i];
          }
          tail += __popc(m);
        }
        cntB2 = tail - headB2;
        __syncwarp();
        continue;
      }
      if (rows_left) {
        // ---------------- stage A: Philox block 0 + slit 1 on the raw draws, until a full warp of
        // survivors is queued (tight loop: ~4 rows per stage-B round at a 25 % pass rate)
        const bool s1_int = P.s1_int_ok != 0;
        const uint32_t lo0 = P.s1_lo[0], hi0 = P.s1_hi[0], lo1 = P.s1_lo[1], hi1 = P.s1_hi[1];
        const uint32_t id0 = first_lo + off0 + lane;
#if SAS_STAGE_A_ROWS >= 2
        // several rows per step: independent Philox chains in flight, round keys loaded once
        do {
          constexpr int NR = SAS_STAGE_A_ROWS;
          uint32_t w[NR][4];
          bool pass[NR];
          unsigned m[NR];
#pragma unroll
          for (int k = 0; k < NR; ++k) {
            philox4x32_10(a.keys, id0 + ((row + k * WARPS_PER_BLOCK) << 5), id_hi, 0u, exp_word, w[k]);
          }
          int tail = headB + cntB;
#pragma unroll
          for (int k = 0; k < NR; ++k) {
            const uint32_t in_item = ((row + k * WARPS_PER_BLOCK) << 5) + lane;
            pass[k] = in_item < cnt_ids;  // a row past the item's end fails here as well
            if (s1_int) pass[k] = pass[k] && (w[k][0] - lo0 <= hi0 - lo0) && (w[k][1] - lo1 <= hi1 - lo1);
            m[k] = __ballot_sync(FULL, pass[k]);
            if (pass[k]) {
              const int s2 = (tail + __popc(m[k] & lt_mask)) & (RING_B - 1);
              wq.b_id[s2] = off0 + in_item;
            }
            tail += __popc(m[k]);
          }
          cntB = tail - headB;
          row += NR * WARPS_PER_BLOCK;
#else
        do {
          const uint32_t in_item = (row << 5) + lane;
          uint32_t w[4];
          philox4x32_10(a.keys, id0 + (row << 5), id_hi, 0u, exp_word, w);
          bool pass = in_item < cnt_ids;
          if (s1_int) pass = pass && (w[0] - lo0 <= hi0 - lo0) && (w[1] - lo1 <= hi1 - lo1);
          const unsigned m = __ballot_sync(FULL, pass);
          const int np = __popc(m);
          if (pass) {
            const int s2 = (headB + cntB + __popc(m & lt_mask)) & (RING_B - 1);
            wq.b_id[s2] = off0 + in_item;
          }
          cntB += np;
          row += WARPS_PER_BLOCK;
#endif
        } while (row < row_end && cntB < 32 * NB0);
        __syncwarp();
        continue;
      }
      break;
    }
  }

  // counters[0] (launched) is known to the host; counters[1] (died at slit 1) is what is left of it after
  // every other outcome (sas_get_counters): a neutron that the integer slit-1 test drops is never queued
  if (!DUMP) flush_outcomes(a.counters, wq.oc);
}

}  // namespace sas
