// lof_common.cuh — shared device-side definitions of the LOF CUDA path (sm_100a).
// Nothing here is shared with oracle/ (the oracle is written separately from PAPER.md).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/lof.h"

#define LOF_HIST_BINS 2048

// Per-stream device state: statistics, radix-select progress, thresholds.
struct LofStreamState {
  double   shift;                  // K = first sample; sums are of (x - K) (statistics)
  double   sum, sumsq;             // sum (x-K), sum (x-K)^2 over the stream, fixed reduction order
  double   mean, stddev;
  double   thr_d[LOF_MAX_LEVELS];  // threshold_I, fp64
  float    thr_f[LOF_MAX_LEVELS];  // same rounded to fp32: what the flag kernels compare against
  float    dead_f[LOF_MAX_LEVELS]; // early-exit levels of the frequency run (lof_dead_level), one per iteration
  float    dead_t[LOF_MAX_LEVELS]; // ... of the time run
  uint32_t nonfinite;
  uint32_t prefix;                 // radix select: key bits fixed so far
  uint32_t rank;                   // rank still to find among keys matching prefix
  float    median;
  // two-pass statistics of long streams (lof_stats_lr.cuh): histogram placement, the median's bin, candidates
  float    pl_scale, pl_off;       // bin(x) = round(clamp(x*pl_scale + pl_off)); shift is the centre K
  float    vmid, vhalf;            // |x - vmid| <= vhalf encloses the median's bin
  uint32_t bin, before, nb;        // that bin, the number of samples in lower bins, the number in the bin
  uint32_t ncand;                  // candidates gathered so far
  uint32_t fallback;               // 1: the histogram could not isolate the median; radix select over the stream
};

// Parameters every kernel needs, passed by value.
struct LofKParams {
  uint32_t S, C, T, W;             // W = ceil(T/32) flag words per row
  uint32_t n_levels;               // log2(max_window)+1
  uint32_t n_lev_f, n_lev_t;       // levels actually run along frequency / time (0 = direction off)
  uint32_t s0;                     // first stream of the group this launch works on
  double   factor[LOF_MAX_LEVELS]; // factor_I, fp64, host-computed
  double   sensitivity;
};

// Monotone map float -> uint32: ascending keys <=> ascending floats (radix select on bit patterns).
__device__ __forceinline__ uint32_t lof_key(float x) {
  uint32_t b = __float_as_uint(x);
  return b ^ ((b >> 31) ? 0xFFFFFFFFu : 0x80000000u);
}
__device__ __forceinline__ float lof_unkey(uint32_t k) {
  uint32_t b = (k >> 31) ? (k ^ 0x80000000u) : ~k;
  return __uint_as_float(b);
}
__device__ __forceinline__ bool lof_finite(float x) {
  return (__float_as_uint(x) & 0x7F800000u) != 0x7F800000u;
}

// Input adapters: float32 power, or complex int16 voltages turned into power on load
// (x = (float)(uint32)(re*re + im*im), integer-exact, S5).
struct InF32 {
  const float* p;
  __device__ __forceinline__ float ld(size_t i) const { return __ldg(p + i); }
  // four consecutive samples, i a multiple of 4 (the API requires 16-byte aligned input)
  __device__ __forceinline__ void ld4(size_t i, float (&x)[4]) const {
    const float4 v = __ldg(reinterpret_cast<const float4*>(p + i));
    x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w;
  }
  static constexpr int kBytes = 4;
  // a sample as it lies in memory (4 bytes) <-> the float32 power; `is_raw` = false: the word already holds the power
  __device__ __forceinline__ static uint32_t raw_of(float x) { return __float_as_uint(x); }
  __device__ __forceinline__ static float from_raw(uint32_t w, bool) { return __uint_as_float(w); }
};
struct InCI16 {
  const int16_t* p;
  __device__ __forceinline__ float ld(size_t i) const {
    const short2 v = __ldg(reinterpret_cast<const short2*>(p) + i);
    const int re = v.x, im = v.y;
    return __uint2float_rn((unsigned)(re * re) + (unsigned)(im * im));     // unsigned: (-32768, -32768) gives 2^31
  }
  __device__ __forceinline__ void ld4(size_t i, float (&x)[4]) const {
    const int4 v = __ldg(reinterpret_cast<const int4*>(p + 2 * i));
    const int w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int re = (int)(short)(w[k] & 0xFFFF), im = w[k] >> 16;
      x[k] = __uint2float_rn((unsigned)(re * re) + (unsigned)(im * im));
    }
  }
  static constexpr int kBytes = 4;
  // staging strips filled by asynchronous copies hold the voltage pair itself (is_raw), those filled through ld()
  // the power
  __device__ __forceinline__ static uint32_t raw_of(float x) { return __float_as_uint(x); }
  __device__ __forceinline__ static float from_raw(uint32_t w, bool is_raw) {
    if (!is_raw) return __uint_as_float(w);
    const int re = (int)(short)(w & 0xFFFFu), im = (int)w >> 16;
    return __uint2float_rn((unsigned)(re * re) + (unsigned)(im * im));
  }
};

// cycles of thread 0 per phase, summed over CTAs and streams, when built with -DLOF_FUSED_PROF (profiling builds
// only; process-global): [0] first load + statistics, [1] frequency pass, [2] plan of the next stream, [3] time
// pass with the next stream's row statistics, [4] end of the next stream's statistics
#ifdef LOF_FUSED_PROF
__device__ unsigned long long lof_fused_cycles_dev[8];
#endif
#ifdef LOF_FUSED_PROF
#define LOF_PROF_T(var) const long long var = clock64()
#define LOF_PROF_ADD(i, a, b) do { if (threadIdx.x == 0) atomicAdd(&lof_fused_cycles_dev[i], (unsigned long long)((b) - (a))); } while (0)
#define LOF_PROF_CNT(i) do { if ((threadIdx.x & 31) == 0) atomicAdd(&lof_fused_cycles_dev[i], 1ull); } while (0)
#else
#define LOF_PROF_T(var)
#define LOF_PROF_ADD(i, a, b)
#define LOF_PROF_CNT(i)
#endif

// Early exit of a SumThreshold run.  A window of 2^k samples is a disjoint union of windows
// of 2^j samples (j < k), and it fires only if the sum over its unflagged samples of (x - threshold_k) is
// positive (reading F7) — so at least one of those smaller windows has an unflagged mean above
// threshold_k.  Hence: if after iteration j NO window of 2^j samples has an unflagged mean above
// D_j = min over the iterations k still to come of threshold_k, none of them can flag anything and the run
// stops.  The test is exact; D_j is lowered by 2e-6 relative so that the fp32 rounding of the doubled sums
// (<= 10 additions, 6e-7 relative) and of the thresholds can never turn a skipped window into a firing one: the
// result is bit-identical to running every iteration.  A non-positive D_j disables the exit (-huge).
__device__ __forceinline__ float lof_dead_level(double median, double stddev, const double* factor, double sens,
                                                uint32_t j, uint32_t n_lev) {
  double tmin = 1e300;
  for (uint32_t k = j + 1; k < n_lev; ++k) tmin = fmin(tmin, median + stddev * factor[k] * sens);
  if (j + 1 >= n_lev) return 3.0e38f;                    // no iteration left: nothing can fire
  return tmin > 0.0 ? (float)(tmin * (1.0 - 2e-6)) : -1.0e34f;
}

// The same from the thresholds already rounded to fp32 (thr[k], each within 2^-24 relative of the fp64 value):
// 3e-6 relative below their minimum stays under the bound above.
__device__ __forceinline__ float lof_dead_level_f(const float* thr, uint32_t j, uint32_t n_lev) {
  if (j + 1 >= n_lev) return 3.0e38f;
  float tmin = thr[j + 1];
  for (uint32_t k = j + 2; k < n_lev; ++k) tmin = fminf(tmin, thr[k]);
  return tmin > 0.f ? tmin * (1.0f - 3e-6f) : -1.0e34f;
}

__device__ __forceinline__ float lof_max3(float a, float b, float c) {
  float d;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));   // FMNMX3: one issue slot, sm_100+
  return d;
}

// Deterministic block reduction of a double (fixed shuffle tree, then warp 0 in warp order).
__device__ __forceinline__ double lof_warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double lof_block_sum(double v, double* sh /* >= 32 doubles */) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  v = lof_warp_sum(v);
  __syncthreads();
  if (lane == 0) sh[w] = v;
  __syncthreads();
  double r = 0.0;
  if (w == 0) {
    r = lane < nw ? sh[lane] : 0.0;
    r = lof_warp_sum(r);
  }
  return r;   // valid in thread 0
}
