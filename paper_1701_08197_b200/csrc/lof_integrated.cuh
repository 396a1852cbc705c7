// lof_integrated.cuh — kernels of the fully integrated mode (Fig. 4): "integrate the time
// direction fully for frequency flagging, and ... the frequency direction fully for time domain flagging".
//   lof_k_integ_sums      ONE read of the block: per (stream, channel) the sum over time (tile partials, added in
//                         tile order later) and per (stream, time sample) the sum over ALL channels
//   lof_k_integ_spectrum  a[s][c] = (float)(sum / T)
//   (1-D SumThreshold over a: the ordinary time-run kernels on a block of S x 1 x C, host side)
//   lof_k_integ_series    b[s][t] = (float)((column sum - sum over the FLAGGED channels) / #unflagged channels):
//                         only the rows of flagged channels are read again
//   (1-D SumThreshold over b: the same kernels on S x 1 x T)
//   lof_k_integ_combine   flags[s][c][w] = channel flagged ? all ones : time mask word
// This path is bound by HBM: 4 B read per sample plus 1/8 B written, and a few instructions per sample.
#pragma once
#include "lof_common.cuh"

#define LOF_IG_THREADS 256
#define LOF_IG_TILE (4 * LOF_IG_THREADS)      // time samples per CTA: one float4 per thread and channel

// grid = (n_tiles, S).  Thread i of the CTA owns the four columns t0 + 4i .. t0 + 4i + 3 of the tile.
// Column sums: fp32 over groups of 8 channels, then fp64, channels in index order.  Row sums of the tile: fp32
// within the thread's four samples and across the warp (fixed shuffle tree), per-warp partials added in warp
// order as fp64: rowpart[s][c][tile].
__global__ void __launch_bounds__(LOF_IG_THREADS)
lof_k_integ_sums(const float* __restrict__ x, double* __restrict__ rowpart, double* __restrict__ colsum,
                 uint32_t C, uint32_t T, uint32_t n_tiles) {
  __shared__ float wpart[256][LOF_IG_THREADS / 32 + 1];   // [channel][warp]
  const uint32_t s = blockIdx.y, tile = blockIdx.x;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t t = tile * LOF_IG_TILE + 4u * tid;
  const float* xs = x + (size_t)s * C * T;
  const bool vec = (T & 3u) == 0 && t + 3 < T;            // rows start 16-byte aligned only when T % 4 == 0
  double c0 = 0.0, c1 = 0.0, c2 = 0.0, c3 = 0.0;
  float g0 = 0.f, g1 = 0.f, g2 = 0.f, g3 = 0.f;
  for (uint32_t cb = 0; cb < C; cb += 8) {
    float4 v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const uint32_t c = cb + k;
      v[k] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (c < C) {
        const float* p = xs + (size_t)c * T + t;
        if (vec) v[k] = __ldg(reinterpret_cast<const float4*>(p));
        else {
          if (t < T) v[k].x = __ldg(p);
          if (t + 1 < T) v[k].y = __ldg(p + 1);
          if (t + 2 < T) v[k].z = __ldg(p + 2);
          if (t + 3 < T) v[k].w = __ldg(p + 3);
        }
      }
    }
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      g0 += v[k].x; g1 += v[k].y; g2 += v[k].z; g3 += v[k].w;
      float r = (v[k].x + v[k].y) + (v[k].z + v[k].w);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
      if (lane == 0 && cb + k < C) wpart[cb + k][warp] = r;
    }
    c0 += (double)g0; c1 += (double)g1; c2 += (double)g2; c3 += (double)g3;
    g0 = g1 = g2 = g3 = 0.f;
  }
  double* cs = colsum + (size_t)s * T;
  if (t < T) cs[t] = c0;
  if (t + 1 < T) cs[t + 1] = c1;
  if (t + 2 < T) cs[t + 2] = c2;
  if (t + 3 < T) cs[t + 3] = c3;
  __syncthreads();
  for (uint32_t c = tid; c < C; c += LOF_IG_THREADS) {
    double a = 0.0;
#pragma unroll
    for (int w = 0; w < LOF_IG_THREADS / 32; ++w) a += (double)wpart[c][w];
    rowpart[((size_t)s * C + c) * n_tiles + tile] = a;
  }
}

// a[s][c] = (float)(sum over the tiles, in tile order, / T).  One thread per (s, c).
__global__ void lof_k_integ_spectrum(const double* __restrict__ rowpart, float* __restrict__ spec, uint64_t n_rows,
                                     uint32_t n_tiles, uint32_t T) {
  const uint64_t r = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n_rows) return;
  double a = 0.0;
  for (uint32_t j = 0; j < n_tiles; ++j) a += rowpart[r * n_tiles + j];
  spec[r] = (float)(a / (double)T);
}

// b[s][t]: mean over the unflagged channels.  cmask: [S][ceil(C/32)] words, bit c = channel c flagged.
// One thread per (s, t); the rows of flagged channels are read again (coalesced over t), channels in index order.
__global__ void lof_k_integ_series(const float* __restrict__ x, const double* __restrict__ colsum,
                                   const uint32_t* __restrict__ cmask, float* __restrict__ series, uint32_t S,
                                   uint32_t C, uint32_t T) {
  const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= (uint64_t)S * T) return;
  const uint32_t s = (uint32_t)(gid / T), t = (uint32_t)(gid - (uint64_t)s * T);
  const uint32_t CW = (C + 31) / 32;
  const float* xs = x + (size_t)s * C * T + t;
  double fsum = 0.0;
  uint32_t nfl = 0;
  for (uint32_t w = 0; w < CW; ++w) {
    uint32_t m = cmask[(size_t)s * CW + w];
    nfl += __popc(m);
    while (m) {
      const uint32_t c = w * 32u + (uint32_t)__ffs((int)m) - 1u;
      m &= m - 1u;
      fsum += (double)__ldg(xs + (size_t)c * T);
    }
  }
  const uint32_t n_unf = C - nfl;
  series[gid] = n_unf ? (float)((colsum[gid] - fsum) / (double)n_unf) : 0.f;
}

// flags[s][c][w] = channel c flagged ? all ones (padding bits 0) : tmask[s][w].  One thread per (s, c, w).
__global__ void lof_k_integ_combine(const uint32_t* __restrict__ cmask, const uint32_t* __restrict__ tmask,
                                    uint32_t* __restrict__ flags, uint32_t S, uint32_t C, uint32_t W, uint32_t T) {
  const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= (uint64_t)S * C * W) return;
  const uint32_t w = (uint32_t)(gid % W);
  const uint64_t r = gid / W;
  const uint32_t c = (uint32_t)(r % C), s = (uint32_t)(r / C);
  const uint32_t CW = (C + 31) / 32;
  const bool cf = (cmask[(size_t)s * CW + (c >> 5)] >> (c & 31)) & 1u;
  const uint32_t full = (w == W - 1 && (T & 31)) ? ((1u << (T & 31)) - 1u) : 0xFFFFFFFFu;
  flags[gid] = cf ? full : tmask[(size_t)s * W + w];
}
