// lof_longrow.cuh — register-resident SumThreshold kernels for streams too long for one SM's shared
// memory (BASELINE.json configs 4 and 5: rows of 195 312 and 12 208 samples).  Same column / row cores as
// the fused kernel (lof_col_flag, lof_row_flag in lof_fused.cuh), fed from global memory (L2-resident: the
// host processes streams in groups that fit L2, after the statistics passes of lof_stats.cuh).
//   lof_k_freq_reg<C>: a warp per group of 32 time columns, a thread per column.
//   lof_k_time_seg   : a warp per row segment of 1024 samples = OUT output samples + a halo of H on
//                      each side, H >= the dependency cone sum_k (2^k - 1) of the time run, so segments
//                      are independent; lane l holds samples [32 l, 32 l + 32).
#pragma once
#include "lof_common.cuh"
#include "lof_fused.cuh"

#define LOF_LR_THREADS 256
#define LOF_LR_WARPS (LOF_LR_THREADS / 32)
#define LOF_LR_TILE 1024

template <int C, class In>
__global__ void __launch_bounds__(LOF_LR_THREADS)
lof_k_freq_reg(In in, LofKParams prm, const LofStreamState* __restrict__ state, uint32_t* __restrict__ fmask,
               uint32_t n_group_streams) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint64_t gid = (uint64_t)blockIdx.x * LOF_LR_WARPS + warp;
  const uint32_t W = prm.W, T = prm.T;
  if (gid >= (uint64_t)n_group_streams * W) return;       // whole warps leave together
  const uint32_t sl = (uint32_t)(gid / W), w = (uint32_t)(gid - (uint64_t)sl * W), s = prm.s0 + sl;
  const uint32_t t = w * 32 + lane;
  const bool valid = t < T;
  const uint64_t base = (uint64_t)s * C * T + (valid ? t : 0);
  const float* thr = state[s].thr_f;
  // a column beyond the row's end holds -inf: it never exceeds a threshold and any window sum with it is -inf
  const uint64_t fb = lof_col_flag<C>(
      [&](int c) { return valid ? in.ld(base + (uint64_t)c * T) : -INFINITY; }, thr, (int)prm.n_lev_f);
  uint32_t mine0, mine1;
  lof_col_words<C>(fb, lane, mine0, mine1);
  if (lane < C) fmask[((uint64_t)s * C + lane) * W + w] = mine0;
  if (C > 32 && lane + 32 < C) fmask[((uint64_t)s * C + lane + 32) * W + w] = mine1;
}

// element i of a warp's 1024-sample staging tile: float4 chunk g = i/4 stored at g ^ ((g/8) & 7), so the
// coalesced fill (lanes = consecutive i) and the per-lane reads of 32 consecutive floats are conflict-free
__device__ __forceinline__ int lof_lr_swz(int i) {
  const int g = i >> 2;
  return ((g ^ ((g >> 3) & 7)) << 2) | (i & 3);
}

template <class In>
__global__ void __launch_bounds__(LOF_LR_THREADS, 2)
lof_k_time_seg(In in, LofKParams prm, const LofStreamState* __restrict__ state, const uint32_t* __restrict__ fmask,
               uint32_t* __restrict__ flags, double* __restrict__ part_sum, uint32_t* __restrict__ part_cnt,
               lof_stream_stats* __restrict__ stats, uint32_t OUT, uint32_t H, uint32_t n_seg, uint32_t n_rows) {
  __shared__ __align__(16) float stage[LOF_LR_WARPS][LOF_LR_TILE];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint64_t unit = (uint64_t)blockIdx.x * LOF_LR_WARPS + warp;
  if (unit >= (uint64_t)n_rows * n_seg) return;
  const uint32_t rl = (uint32_t)(unit / n_seg), seg = (uint32_t)(unit - (uint64_t)rl * n_seg);
  const uint32_t W = prm.W, C = prm.C, T = prm.T;
  const uint64_t row = (uint64_t)prm.s0 * C + rl;
  const uint32_t s = (uint32_t)(row / C);
  const LofStreamState& st = state[s];
  const uint32_t o_lo = seg * OUT, o_hi = min(T, o_lo + OUT);
  const uint32_t t_lo = o_lo >= H ? o_lo - H : 0;        // multiple of 32
  float* sg = stage[warp];
  const uint64_t base = row * T;
#pragma unroll 4
  for (int q = 0; q < LOF_LR_TILE / 32; ++q) {
    const int i = q * 32 + lane;
    const uint32_t t = t_lo + i;
    sg[lof_lr_swz(i)] = t < T ? in.ld(base + t) : -INFINITY;   // beyond the row: never flagged, kills windows
  }
  __syncwarp();
  float x[32];
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    const float4 v = reinterpret_cast<const float4*>(sg)[(8 * lane + q) ^ (lane & 7)];
    x[4 * q] = v.x; x[4 * q + 1] = v.y; x[4 * q + 2] = v.z; x[4 * q + 3] = v.w;
  }
  const uint32_t t_w = t_lo + 32 * lane;                  // first sample of this lane's word
  const uint32_t valid = t_w >= T ? 0u : (T - t_w >= 32 ? 0xFFFFFFFFu : ((1u << (T - t_w)) - 1u));
  uint32_t fb = 0;
  if (prm.n_lev_f > 0 && valid) fb = fmask[row * W + (t_w >> 5)];   // start from the frequency run's mask (F10)
  if (st.nonfinite) fb = valid;                           // DESIGN.md S6: the whole stream is flagged
  else if (prm.n_lev_t > 0) lof_row_flag<32>(x, fb, st.thr_f, (int)prm.n_lev_t, lane, [] {});
  fb &= valid;
  const bool mine = t_w >= o_lo && t_w < o_hi;            // this lane's word belongs to the segment's output
  if (mine) flags[row * W + (t_w >> 5)] = fb;
  float p0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f;
  const uint32_t skip = fb | ~valid;
#pragma unroll
  for (int j = 0; j < 32; j += 4) {
    p0 += ((skip >> j) & 1u) ? 0.f : x[j];
    p1 += ((skip >> (j + 1)) & 1u) ? 0.f : x[j + 1];
    p2 += ((skip >> (j + 2)) & 1u) ? 0.f : x[j + 2];
    p3 += ((skip >> (j + 3)) & 1u) ? 0.f : x[j + 3];
  }
  double rs = mine ? (double)((p0 + p1) + (p2 + p3)) : 0.0;
  rs = lof_warp_sum(rs);
  uint32_t nf = mine ? __popc(fb) : 0u, nu = mine ? __popc(valid & ~fb) : 0u;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    nf += __shfl_down_sync(0xffffffffu, nf, o);
    nu += __shfl_down_sync(0xffffffffu, nu, o);
  }
  if (lane == 0) {
    part_sum[(uint64_t)rl * n_seg + seg] = rs;
    part_cnt[(uint64_t)rl * n_seg + seg] = nu;
    if (nf) atomicAdd(reinterpret_cast<unsigned long long*>(&stats[s].n_flagged), (unsigned long long)nf);
  }
}
