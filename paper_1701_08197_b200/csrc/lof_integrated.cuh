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
#include "lof_flag_generic.cuh"
#include "lof_core.cuh"

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
// grid = (ceil(T / (256 * LOF_IG_SER)), S): a thread takes LOF_IG_SER time samples 256 apart; the rows of flagged
// channels are read again (coalesced over t), channels in index order.
#define LOF_IG_SER 4
__global__ void __launch_bounds__(256)
lof_k_integ_series(const float* __restrict__ x, const double* __restrict__ colsum,
                   const uint32_t* __restrict__ cmask, float* __restrict__ series, uint32_t C, uint32_t T) {
  __shared__ uint32_t cm[8];                              // C <= 256
  const uint32_t s = blockIdx.y;
  const uint32_t CW = (C + 31) / 32;
  if (threadIdx.x < CW) cm[threadIdx.x] = cmask[(size_t)s * CW + threadIdx.x];
  __syncthreads();
  uint32_t nfl = 0;
  for (uint32_t w = 0; w < CW; ++w) nfl += __popc(cm[w]);
  const uint32_t n_unf = C - nfl;
  const double inv = n_unf ? 1.0 / (double)n_unf : 0.0;
  (void)inv;
  const uint32_t t0 = blockIdx.x * (256u * LOF_IG_SER) + threadIdx.x;
  const float* xs = x + (size_t)s * C * T;
  double fsum[LOF_IG_SER];
#pragma unroll
  for (int k = 0; k < LOF_IG_SER; ++k) fsum[k] = 0.0;
  for (uint32_t w = 0; w < CW; ++w) {
    uint32_t m = cm[w];
    while (m) {                                           // (uniform over the CTA: every thread has the same mask)
      const uint32_t c = w * 32u + (uint32_t)__ffs((int)m) - 1u;
      m &= m - 1u;
#pragma unroll
      for (int k = 0; k < LOF_IG_SER; ++k) {
        const uint32_t t = t0 + 256u * k;
        if (t < T) fsum[k] += (double)__ldg(xs + (size_t)c * T + t);
      }
    }
  }
#pragma unroll
  for (int k = 0; k < LOF_IG_SER; ++k) {
    const uint32_t t = t0 + 256u * k;
    if (t < T) {
      const size_t g = (size_t)s * T + t;
      series[g] = n_unf ? (float)((colsum[g] - fsum[k]) / (double)n_unf) : 0.f;
    }
  }
}

// flags[s][c][w] = channel c flagged ? all ones (padding bits 0) : tmask[s][w].  One CTA per stream: the time
// mask's W words sit in shared memory (W <= LOF_IG_TM words, else they are read from global memory).
#define LOF_IG_TM 1024
__global__ void __launch_bounds__(256)
lof_k_integ_combine(const uint32_t* __restrict__ cmask, const uint32_t* __restrict__ tmask,
                    uint32_t* __restrict__ flags, uint32_t C, uint32_t W, uint32_t T) {
  __shared__ uint32_t cm[8];
  __shared__ uint32_t tm[LOF_IG_TM];
  const uint32_t s = blockIdx.x;
  const uint32_t CW = (C + 31) / 32;
  if (threadIdx.x < CW) cm[threadIdx.x] = cmask[(size_t)s * CW + threadIdx.x];
  const bool staged = W <= LOF_IG_TM;
  if (staged) for (uint32_t w = threadIdx.x; w < W; w += 256) tm[w] = tmask[(size_t)s * W + w];
  __syncthreads();
  const uint32_t last = (T & 31) ? ((1u << (T & 31)) - 1u) : 0xFFFFFFFFu;
  uint32_t* fo = flags + (size_t)s * C * W;
  for (uint32_t i = threadIdx.x; i < C * W; i += 256) {
    const uint32_t c = i / W, w = i - c * W;
    const bool cf = (cm[c >> 5] >> (c & 31)) & 1u;
    const uint32_t full = (w == W - 1) ? last : 0xFFFFFFFFu;
    fo[i] = cf ? full : (staged ? tm[w] : __ldg(tmask + (size_t)s * W + w));
  }
}

// ---- one SumThreshold run over a short vector (n <= LOF_VEC_MAX), statistics included: one CTA per vector.
// The integrated mode's two runs are over S vectors of C and of T samples; for the shapes of BASELINE.json's
// configs 1-3 (C <= 64, T <= 768) the multi-kernel statistics of lof_stats_lr.cuh would be a dozen launches of
// latency-bound work.  Here: load -> mean, stddev (two passes, fp64, fixed order: PAPER.md:41, readings S1-S3)
// -> exact median by a bitonic sort of a copy in shared memory -> thresholds -> lof_line_levels (the generic
// shared-memory SumThreshold of lof_flag_generic.cuh) -> packed mask + stats record.
#define LOF_VEC_MAX 4096

__global__ void __launch_bounds__(LOF_GEN_THREADS)
lof_k_vec_flag(const float* __restrict__ vec, uint32_t n, LofKParams prm, uint32_t n_lev, uint32_t* __restrict__ mask,
               lof_stream_stats* __restrict__ stats) {
  extern __shared__ __align__(16) unsigned char vraw[];
  __shared__ double red[32];
  __shared__ float thr[LOF_MAX_LEVELS];
  __shared__ uint32_t cnt[2];
  const uint32_t s = blockIdx.x, tid = threadIdx.x;
  const uint32_t Mpad = (n + 31) & ~31u;
  uint32_t npad = 32;
  while (npad < n) npad <<= 1;
  LofLineSmem sm(vraw, Mpad);
  float* ks = reinterpret_cast<float*>(vraw + (size_t)Mpad * LOF_GEN_BYTES_PER_ELEM + 16);
  ks = reinterpret_cast<float*>(((uintptr_t)ks + 15) & ~(uintptr_t)15);
  const float* v = vec + (size_t)s * n;
  if (tid < 2) cnt[tid] = 0;
  __syncthreads();
  uint32_t bad = 0;
  for (uint32_t i = tid; i < npad || i < Mpad; i += LOF_GEN_THREADS) {
    const float x = i < n ? v[i] : 0.f;
    if (i < Mpad) { sm.xs[i] = x; sm.fl[i] = 0; }
    if (i < npad) ks[i] = i < n ? x : INFINITY;
    if (i < n && !lof_finite(x)) ++bad;
  }
  if (bad) atomicAdd(&cnt[0], bad);
  __syncthreads();
  const uint32_t n_bad = cnt[0];
  // mean, then population stddev about it: thread i adds elements i, i + 256, ... ; fixed tree over the CTA
  double a = 0.0;
  for (uint32_t i = tid; i < n; i += LOF_GEN_THREADS) a += (double)sm.xs[i];
  a = lof_block_sum(a, red);
  if (tid == 0) red[0] = a / (double)n;
  __syncthreads();
  const double mean = red[0];
  __syncthreads();
  double q = 0.0;
  for (uint32_t i = tid; i < n; i += LOF_GEN_THREADS) { const double d = (double)sm.xs[i] - mean; q += d * d; }
  q = lof_block_sum(q, red);
  if (tid == 0) red[1] = sqrt(q / (double)n);
  // bitonic sort of the copy (ascending; the padding is +inf): median = element of rank floor(n/2)
  for (uint32_t k = 2; k <= npad; k <<= 1) {
    for (uint32_t j = k >> 1; j > 0; j >>= 1) {
      __syncthreads();
      for (uint32_t i = tid; i < npad; i += LOF_GEN_THREADS) {
        const uint32_t p = i ^ j;
        if (p > i) {
          const float x = ks[i], y = ks[p];
          const bool up = (i & k) == 0;
          if ((x > y) == up) { ks[i] = y; ks[p] = x; }
        }
      }
    }
  }
  __syncthreads();
  const float median = ks[n / 2];
  const double stddev = red[1];
  if (tid < n_lev) thr[tid] = (float)((double)median + stddev * prm.factor[tid] * prm.sensitivity);
  __syncthreads();
  if (n_bad) { for (uint32_t i = tid; i < Mpad; i += LOF_GEN_THREADS) sm.fl[i] = 1; __syncthreads(); }
  else lof_line_levels<1>(sm, n, n_lev, thr);
  const uint32_t W = (n + 31) / 32;
  uint32_t nf = 0;
  for (uint32_t i = tid; i < Mpad; i += LOF_GEN_THREADS) {
    const bool f = i < n && sm.fl[i] != 0;
    const uint32_t word = __ballot_sync(0xffffffffu, f);
    if ((tid & 31) == 0) { mask[(size_t)s * W + (i >> 5)] = word; nf += __popc(word); }
  }
  if (nf) atomicAdd(&cnt[1], nf);
  __syncthreads();
  if (tid == 0) {
    lof_stream_stats o;
    o.median = median; o.n_nonfinite = n_bad; o.mean = mean; o.stddev = stddev; o.n_flagged = cnt[1];
    stats[s] = o;
  }
}

// ---- the same for vectors of at most 1024 samples, one WARP per vector and no block barrier: lane l holds the
// samples [l*L, l*L + L) (beyond n: -inf, which no window survives); mean / stddev by fp64 shuffle trees in a
// fixed order, the exact median by a bitwise radix select on the monotone keys (32 votes), then the row core of
// lof_core.cuh (the one the time run of the fused kernel uses), and the mask words gathered by shuffles.
// Two neighbours of the integrated mode can ride on this kernel instead of being launches of their own
// (LofVecFuse, all pointers optional): the spectrum a[s][c] = (float)(sum over tiles / T) formed from the row
// partials when the vector is loaded (what lof_k_integ_spectrum does), and the final flags[s][c][w] written from
// the mask words while they are in the warp's registers (what lof_k_integ_combine does); for the series run also
// the series itself, b[s][t] = (column sum - sum over the flagged channels) / #unflagged, same operations in the
// same order as lof_k_integ_series.
struct LofVecFuse {
  const double* rowpart; uint32_t n_tiles, T; float* spec_out;      // vec[s][i] = (float)(sum_j rowpart[(s n + i) n_tiles + j] / T)
  const uint32_t* cmask; uint32_t* flags; uint32_t C;               // flags[s][c][w] = channel c flagged ? ones : mask word w
  const float* block; const double* colsum; float* series_out;      // vec[s][t] = series b[s][t] from the block [S][C][n]
};
template <int L>
__global__ void __launch_bounds__(256)
lof_k_vec_warp(const float* __restrict__ vec, uint32_t n, uint32_t S, LofKParams prm, uint32_t n_lev,
               uint32_t* __restrict__ mask, lof_stream_stats* __restrict__ stats, LofVecFuse fz) {
  __shared__ float wthr[8][32];                           // per warp: [0..16) thresholds, [16..32) early-exit levels
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t s = blockIdx.x * 8u + (uint32_t)warp;
  if (s >= S) return;                                     // whole warps leave together
  const float* v = vec + (size_t)s * n;
  const uint32_t i0 = (uint32_t)lane * L;
  const uint32_t nv = i0 >= n ? 0u : (n - i0 >= (uint32_t)L ? (uint32_t)L : n - i0);      // valid samples of this lane
  const uint32_t valid = nv >= 32 ? 0xFFFFFFFFu : ((1u << nv) - 1u);
  float x[L];
  if (fz.rowpart) {
#pragma unroll
    for (int j = 0; j < L; ++j) {
      x[j] = -INFINITY;
      if ((uint32_t)j < nv) {
        const uint64_t r = (uint64_t)s * n + i0 + j;
        double a = 0.0;
        for (uint32_t k = 0; k < fz.n_tiles; ++k) a += fz.rowpart[r * fz.n_tiles + k];
        x[j] = (float)(a / (double)fz.T);
        fz.spec_out[r] = x[j];
      }
    }
  } else if (fz.colsum) {
    const uint32_t CW = (fz.C + 31) / 32;
    const uint32_t cmw = (uint32_t)lane < CW ? fz.cmask[(size_t)s * CW + lane] : 0u;
    const uint32_t n_unf = fz.C - __reduce_add_sync(0xffffffffu, (uint32_t)__popc(cmw));
    const float* xs = fz.block + (size_t)s * fz.C * n;
    double fs[L];
#pragma unroll
    for (int j = 0; j < L; ++j) fs[j] = 0.0;
    for (uint32_t w = 0; w < CW; ++w) {
      uint32_t m = __shfl_sync(0xffffffffu, cmw, (int)w);   // the same for every lane: uniform loops
      while (m) {
        const uint32_t c = w * 32u + (uint32_t)__ffs((int)m) - 1u;
        m &= m - 1u;
#pragma unroll
        for (int j = 0; j < L; ++j) if ((uint32_t)j < nv) fs[j] += (double)__ldg(xs + (size_t)c * n + i0 + j);
      }
    }
#pragma unroll
    for (int j = 0; j < L; ++j) {
      x[j] = -INFINITY;
      if ((uint32_t)j < nv) {
        const size_t g = (size_t)s * n + i0 + j;
        x[j] = n_unf ? (float)((fz.colsum[g] - fs[j]) / (double)n_unf) : 0.f;
        fz.series_out[g] = x[j];
      }
    }
  } else {
#pragma unroll
    for (int j = 0; j < L; ++j) x[j] = (uint32_t)j < nv ? __ldg(v + i0 + j) : -INFINITY;
  }
  uint32_t bad = 0;
  double a = 0.0;
#pragma unroll
  for (int j = 0; j < L; ++j) if ((uint32_t)j < nv) { bad += lof_finite(x[j]) ? 0u : 1u; a += (double)x[j]; }
  const uint32_t n_bad = __reduce_add_sync(0xffffffffu, bad);
  a = lof_warp_sum(a);
  const double mean = __shfl_sync(0xffffffffu, a, 0) / (double)n;
  double q = 0.0;
#pragma unroll
  for (int j = 0; j < L; ++j) if ((uint32_t)j < nv) { const double d = (double)x[j] - mean; q += d * d; }
  q = lof_warp_sum(q);
  const double stddev = sqrt(__shfl_sync(0xffffffffu, q, 0) / (double)n);
  // exact median: the key of rank floor(n/2), one bit per vote from the top
  uint32_t cand = valid, rank = n / 2, prefix = 0;
  uint32_t key[L];
#pragma unroll
  for (int j = 0; j < L; ++j) key[j] = lof_key(x[j]);
  uint32_t left = n;                                       // candidates left (warp-uniform)
#pragma unroll 1
  for (int b = 31; b >= 0 && left > 1; --b) {
    uint32_t ones = 0;
#pragma unroll
    for (int j = 0; j < L; ++j) ones |= ((key[j] >> b) & 1u) << j;
    const uint32_t zeros = cand & ~ones;
    const uint32_t c0 = __reduce_add_sync(0xffffffffu, (uint32_t)__popc(zeros));
    if (rank < c0) { cand = zeros; left = c0; }
    else { rank -= c0; cand &= ones; left -= c0; prefix |= 1u << b; }
  }
  if (left == 1) {                                         // a single candidate: its key is the answer (usually after
    uint32_t k = 0;                                        // about 20 of the 32 votes)
#pragma unroll
    for (int j = 0; j < L; ++j) if ((cand >> j) & 1u) k = key[j];
    prefix = __shfl_sync(0xffffffffu, k, __ffs((int)__ballot_sync(0xffffffffu, cand != 0u)) - 1);
  }
  const float median = lof_unkey(prefix);
  if ((uint32_t)lane < n_lev) {
    wthr[warp][lane] = (float)((double)median + stddev * prm.factor[lane] * prm.sensitivity);
    wthr[warp][16 + lane] = lof_dead_level((double)median, stddev, prm.factor, prm.sensitivity, lane, n_lev);
  }
  __syncwarp();
  uint32_t fb = 0;
  float lane_sum = 0.f;
  if (n_bad) fb = valid;                                  // S6
  else {
    auto load = [&](float2 (&x2)[L / 2], bool) {
#pragma unroll
      for (int m = 0; m < L / 2; ++m) x2[m] = make_float2(x[2 * m], x[2 * m + 1]);
    };
    lof_row_flag<L, 9>(load, fb, wthr[warp], wthr[warp] + 16, (int)n_lev, lane, lane_sum);
    fb &= valid;
  }
  // word w of the vector = bits [32w, 32w+32) gathered from the lanes' L-bit masks
  {
    const uint32_t W = (n + 31) / 32;
    const int q0 = (32 * lane) / L, r0 = 32 * lane - L * q0;
    uint32_t word = 0;
    constexpr int NI = (31 + L) / L + 1;
#pragma unroll
    for (int i = 0; i < NI; ++i) {
      const int src = q0 + i;
      uint32_t w = __shfl_sync(0xffffffffu, fb, src & 31);
      if (src > 31) w = 0;
      const int sh = i * L - r0;
      if (sh < 32) word |= sh >= 0 ? (w << sh) : (w >> (-sh));
    }
    if ((uint32_t)lane < W) mask[(size_t)s * W + lane] = word;
    if (fz.flags) {
      const uint32_t CW = (fz.C + 31) / 32, tot = fz.C * W;
      const uint32_t cmw = (uint32_t)lane < CW ? fz.cmask[(size_t)s * CW + lane] : 0u;     // C <= 256: 8 words
      const uint32_t last = (n & 31) ? ((1u << (n & 31)) - 1u) : 0xFFFFFFFFu;
      uint32_t* fo = fz.flags + (size_t)s * tot;
      const uint32_t d32 = 32u / W, r32 = 32u - d32 * W;  // i -> i + 32: c += d32, w += r32 (with carry)
      uint32_t cq = (uint32_t)lane / W, w = (uint32_t)lane - cq * W;
      for (uint32_t i0w = 0; i0w < tot; i0w += 32) {       // warp-uniform trip count: shuffles inside
        const uint32_t i = i0w + (uint32_t)lane;
        const uint32_t c = cq < fz.C ? cq : fz.C - 1;
        const uint32_t cmv = __shfl_sync(0xffffffffu, cmw, (int)(c >> 5));
        const uint32_t tv = __shfl_sync(0xffffffffu, word, (int)w);
        if (i < tot) fo[i] = ((cmv >> (c & 31)) & 1u) ? (w == W - 1 ? last : 0xFFFFFFFFu) : tv;
        cq += d32; w += r32;
        if (w >= W) { w -= W; ++cq; }
      }
    }
  }
  const uint32_t nf = __reduce_add_sync(0xffffffffu, (uint32_t)__popc(fb));
  if (lane == 0) {
    lof_stream_stats o;
    o.median = median; o.n_nonfinite = n_bad; o.mean = mean; o.stddev = stddev; o.n_flagged = nf;
    stats[s] = o;
  }
}
