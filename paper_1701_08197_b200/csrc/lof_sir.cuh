// lof_sir.cuh — the scale-invariant rank operator as PAPER.md:49-57 states it: "all ranges of consecutive
// flagged samples are extended by flagging 20% more samples, before and after the original range".  It "operates
// on the flag masks only, and not on the actual data": two kernels on the bit-packed mask
// uint32[S][C][W], frequency direction first, then time on the result (readings SIR-1..6):
//   every maximal run of flagged samples of the INPUT mask of a pass, of length n, gets floor(eta * n) more
//   samples flagged on each side, clipped at the ends of the line; run lengths are those of the input.
// Both kernels read `in` and write `out` (different buffers), and add the bits they set to the stream's n_flagged.
#pragma once
#include "lof_common.cuh"

__device__ __forceinline__ uint32_t lof_sir_ext(float eta, uint32_t n) {
  return (uint32_t)floor((double)eta * (double)n);       // the oracle's expression, same IEEE operations
}

// first position q in [p, pend) whose bit equals `want` (pend if none); w = the row's words
__device__ __forceinline__ uint32_t lof_sir_next(const uint32_t* __restrict__ w, uint32_t p, uint32_t pend, bool want) {
  while (p < pend) {
    uint32_t word = w[p >> 5];
    if (!want) word = ~word;
    word &= 0xFFFFFFFFu << (p & 31);
    if (word) { const uint32_t q = (p & ~31u) + (uint32_t)__ffs((int)word) - 1u; return q < pend ? q : pend; }
    p = (p & ~31u) + 32u;
  }
  return pend;
}
// number of consecutive set bits ending just before pend, looking back no further than p0
__device__ __forceinline__ uint32_t lof_sir_trail(const uint32_t* __restrict__ w, uint32_t p0, uint32_t pend) {
  uint32_t p = pend;
  while (p > p0) {
    const uint32_t wi = (p - 1) >> 5, hi = ((p - 1) & 31) + 1;            // bits [0, hi) of word wi are in range
    uint32_t word = ~w[wi];
    if (hi < 32) word &= (1u << hi) - 1u;
    const uint32_t lo_pos = wi << 5;
    if (lo_pos < p0) word &= 0xFFFFFFFFu << (p0 - lo_pos);
    if (word) { const uint32_t z = lo_pos + 31u - (uint32_t)__clz((int)word); return pend - (z + 1u); }
    if (lo_pos <= p0) break;
    p = lo_pos;
  }
  return pend - p0;
}
// set bits [lo, hi) of the row's words
__device__ __forceinline__ void lof_sir_set(uint32_t* __restrict__ w, uint32_t lo, uint32_t hi) {
  while (lo < hi) {
    const uint32_t wi = lo >> 5, b = lo & 31, e = min(hi - (wi << 5), 32u);
    const uint32_t m = (e >= 32 ? 0xFFFFFFFFu : ((1u << e) - 1u)) & (0xFFFFFFFFu << b);
    w[wi] |= m;
    lo = (wi << 5) + 32u;
  }
}

// Time direction.  G lanes (a power of two <= 32) share one row of T bits; lane j owns the words [j*B, j*B+B).
// 1. per lane: is the block all ones, how many ones lead / trail it; scans across the G lanes give the length of
//    the run that ends just left of the block (carry_in) and of the one that starts just right of it (carry_out);
// 2. per lane: every run of the block with its full length (carries added); the lane in which a run really ends
//    emits the right reach end + floor(eta n), the lane in which it really starts the left reach start - floor(..);
//    an exclusive prefix maximum / suffix minimum over the lanes carries the reaches into the other blocks;
// 3. per lane: out = in | own extensions | [block start, reach from the left) | [reach from the right, block end).
// The row operator for one row: lane j of a group of G lanes (gmask = the group's lanes within the warp) owns the
// words [j*B, j*B+B) of the row wi[0..W) (B = ceil(W/G)); the output words go to wo (a different buffer).  Every
// lane of the group must call it; `live` = false makes the group compute and write nothing.  Returns the number
// of bits this lane's words gained.
// m_min = the shortest run that grows at all (floor(eta * m_min) >= 1): shorter runs — most of them, single
// noise flags — skip the fp64 product, and a lane whose block has nothing to extend copies its words.
template <int G>
__device__ __forceinline__ uint32_t lof_sir_time_row(const uint32_t* wi, uint32_t* wo, int j, unsigned gmask,
                                                     uint32_t W, uint32_t T, float eta, uint32_t m_min, bool live) {
  const uint32_t B = (W + G - 1) / G;
  const uint32_t p0 = min((uint32_t)j * B * 32u, T), p1 = min(((uint32_t)j + 1u) * B * 32u, T), len = p1 - p0;
  // 1. block summary and the carries
  const uint32_t lead = lof_sir_next(wi, p0, p1, false) - p0;
  const bool all = lead == len;
  const uint32_t trail = all ? len : lof_sir_trail(wi, p0, p1);
  uint32_t cin = 0, cout = 0;
  if (G > 1) {
    // inclusive scan of (all, trailing ones) from the left, then shifted by one lane; mirrored from the right
    uint32_t t = trail; bool a = all;
    uint32_t l = lead; bool b = all;
#pragma unroll
    for (int o = 1; o < G; o <<= 1) {
      const uint32_t tl = __shfl_up_sync(gmask, t, o, G); const bool al = __shfl_up_sync(gmask, (int)a, o, G);
      if (j >= o) { if (a) t += tl; a = a && al; }
      const uint32_t lr = __shfl_down_sync(gmask, l, o, G); const bool br = __shfl_down_sync(gmask, (int)b, o, G);
      if (j + o < G) { if (b) l += lr; b = b && br; }
    }
    cin = __shfl_up_sync(gmask, t, 1, G); if (j == 0) cin = 0;
    cout = __shfl_down_sync(gmask, l, 1, G); if (j == G - 1) cout = 0;
  }
  // 2. runs of the block, reaches
  int rmax = -1;                                          // exclusive end of the farthest right extension emitted here
  int lmin = 0x7FFFFFFF;                                  // start of the farthest left extension emitted here
  bool grows = false;                                     // some run of this block has an extension
  for (uint32_t p = p0; p < p1;) {
    const uint32_t a = lof_sir_next(wi, p, p1, true);
    if (a >= p1) break;
    const uint32_t b = lof_sir_next(wi, a, p1, false);
    const bool starts = a > p0 || cin == 0, ends = b < p1 || cout == 0;
    const uint32_t n = (b - a) + (a == p0 ? cin : 0u) + (b == p1 ? cout : 0u);
    const uint32_t e = n >= m_min ? lof_sir_ext(eta, n) : 0u;
    grows = grows || e != 0u;
    if (ends) rmax = max(rmax, (int)min(b + e, T));
    if (starts) lmin = min(lmin, (int)(a > e ? a - e : 0u));
    p = b;
  }
  int rin = -1, lin = 0x7FFFFFFF;
  if (G > 1) {
    int r = rmax, l = lmin;
#pragma unroll
    for (int o = 1; o < G; o <<= 1) {
      const int rl = __shfl_up_sync(gmask, r, o, G); if (j >= o) r = max(r, rl);
      const int lr = __shfl_down_sync(gmask, l, o, G); if (j + o < G) l = min(l, lr);
    }
    rin = __shfl_up_sync(gmask, r, 1, G); if (j == 0) rin = -1;
    lin = __shfl_down_sync(gmask, l, 1, G); if (j == G - 1) lin = 0x7FFFFFFF;
  }
  if (!live) return 0;
  // 3. output words of the block
  const uint32_t w0 = (uint32_t)j * B, w1 = min(w0 + B, W);
  uint32_t before = 0, after = 0;
  for (uint32_t w = w0; w < w1; ++w) { const uint32_t v = wi[w]; wo[w] = v; before += __popc(v); }
  if (grows) for (uint32_t p = p0; p < p1;) {
    const uint32_t a = lof_sir_next(wi, p, p1, true);
    if (a >= p1) break;
    const uint32_t b = lof_sir_next(wi, a, p1, false);
    const bool starts = a > p0 || cin == 0, ends = b < p1 || cout == 0;
    const uint32_t n = (b - a) + (a == p0 ? cin : 0u) + (b == p1 ? cout : 0u);
    const uint32_t e = n >= m_min ? lof_sir_ext(eta, n) : 0u;
    if (ends && e) lof_sir_set(wo, b, min(b + e, p1));
    if (starts && e) lof_sir_set(wo, max(a > e ? a - e : 0u, p0), a);
    p = b;
  }
  if (rin > (int)p0) lof_sir_set(wo, p0, min((uint32_t)rin, p1));
  if (lin < (int)p1) lof_sir_set(wo, max((uint32_t)max(lin, 0), p0), p1);
  for (uint32_t w = w0; w < w1; ++w) after += __popc(wo[w]);
  return after - before;
}

// STAGE: the CTA's 256/G rows are short enough to sit in shared memory (in and out copies, filled and drained
// with coalesced accesses), so that the bit scans run at shared-memory latency.
template <int G, bool STAGE>
__global__ void __launch_bounds__(256)
lof_k_sir_time(const uint32_t* __restrict__ in, uint32_t* __restrict__ out, lof_stream_stats* __restrict__ stats,
               uint64_t n_rows, uint32_t C, uint32_t W, uint32_t T, float eta, uint32_t m_min) {
  extern __shared__ uint32_t sir_sh[];                    // STAGE: [2][256/G][W]
  const uint64_t gid = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) / G;
  const int j = threadIdx.x % G;
  const bool live = gid < n_rows;
  const uint64_t row = live ? gid : n_rows - 1;           // idle groups shadow the last row and write nothing
  const uint32_t* wi = in + row * W;
  uint32_t* wo = out + row * W;
  constexpr int RPB = 256 / G;                            // rows per CTA
  const uint64_t row0 = (uint64_t)blockIdx.x * RPB;
  const uint32_t n_here = (uint32_t)min((uint64_t)RPB, n_rows > row0 ? n_rows - row0 : 0);
  if (STAGE) {
    for (uint32_t i = threadIdx.x; i < n_here * W; i += 256) sir_sh[i] = in[row0 * W + i];
    __syncthreads();
    const uint32_t lr = live ? (uint32_t)(gid - row0) : (n_here ? n_here - 1 : 0);
    wi = sir_sh + lr * W;
    wo = sir_sh + (RPB + lr) * W;
  }
  const unsigned gmask = (G == 32) ? 0xFFFFFFFFu : (((1u << G) - 1u) << ((threadIdx.x & 31) / G * G));
  const uint32_t added = lof_sir_time_row<G>(wi, wo, j, gmask, W, T, eta, m_min, live);
  if (added) atomicAdd(reinterpret_cast<unsigned long long*>(&stats[row / C].n_flagged), (unsigned long long)added);
  if (STAGE) {
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < n_here * W; i += 256) out[row0 * W + i] = sir_sh[RPB * W + i];
  }
}

// The frequency operator on one word column held as a C-bit mask per lane (lane = time sample of the word):
// returns the bits to add (runs of the input mask, each grown by floor(eta * length) on both sides, clipped).
template <int C>
__device__ __forceinline__ unsigned long long lof_sir_col_ext(unsigned long long col, float eta) {
  unsigned long long ext = 0, rest = col;
  while (rest) {
    const int a0 = __ffsll((long long)rest) - 1;
    const unsigned long long from = rest >> a0;                           // the run starts at bit 0 of `from`
    const int len = (~from == 0ull) ? 64 - a0 : __ffsll((long long)~from) - 1;
    const int e = (int)lof_sir_ext(eta, (uint32_t)len);
    const int lo = max(a0 - e, 0), hi = min(a0 + len + e, C);
    ext |= (hi >= 64 ? ~0ull : ((1ull << hi) - 1ull)) & ~((1ull << lo) - 1ull);
    rest = (a0 + len >= 64) ? 0ull : (rest & ~((1ull << (a0 + len)) - 1ull));
  }
  return ext & ~col;
}

// 32 x 32 bit-matrix transpose across a warp: lane r holds row r (bit i = column i); afterwards lane i holds column
// i (bit r = row r).  Five exchange steps (blocks of 16, 8, 4, 2, 1); its own inverse.
__device__ __forceinline__ uint32_t lof_bit_transpose32(uint32_t x, int lane) {
  uint32_t m = 0x0000FFFFu;
#pragma unroll
  for (int j = 16; j > 0; j >>= 1) {
    const uint32_t p = __shfl_xor_sync(0xffffffffu, x, j);
    if ((lane & j) == 0) x ^= (((x >> j) ^ p) & m) << j;
    else x ^= ((p >> j) ^ x) & m;
    m ^= m << (j >> 1);
  }
  return x;
}

// Frequency direction, C = 16, 32 or 64 channels: a WARP per (stream, word column).  Lane c loads the word of
// channel c (and c + 32): 32 time samples each.  Two bit-matrix transposes turn them into one C-bit column mask
// per lane = time sample; a run can only grow if it is at least m_min = ceil(1/eta) channels long, which a few
// shifts and ANDs of the mask decide; the lanes with such a run extend theirs (lof_sir_col_ext); if any lane added
// a bit, two more transposes bring the new bits back to the channel words.  (The first version was a thread per word
// column with the C words in registers and a loop over the time samples with long runs: the lanes of a warp waited
// for the one whose word lay inside a burst — 32 samples x 400 instructions — and the kernel took 150 us for the
// 38 MB mask of config 2 x 64 subbands.)  grid = (S, ceil(W / 8)), 256 threads: a CTA takes 8 consecutive word
// columns of one stream (one 32-byte sector per channel row).
template <int C>
__global__ void __launch_bounds__(256)
lof_k_sir_freq_reg(const uint32_t* __restrict__ in, uint32_t* __restrict__ out, lof_stream_stats* __restrict__ stats,
                   uint32_t W, float eta, uint32_t m_min) {
  const int lane = threadIdx.x & 31;
  const uint32_t s = blockIdx.x, w = blockIdx.y * 8u + (threadIdx.x >> 5);
  if (w >= W) return;                                     // whole warps leave together
  const uint32_t* ci = in + (size_t)s * C * W + w;
  uint32_t* co = out + (size_t)s * C * W + w;
  uint32_t lo = lane < C ? __ldg(ci + (size_t)lane * W) : 0u;
  uint32_t hi = C > 32 ? __ldg(ci + (size_t)(lane + 32) * W) : 0u;
  const uint32_t tl = lof_bit_transpose32(lo, lane);
  const uint32_t th = C > 32 ? lof_bit_transpose32(hi, lane) : 0u;
  const unsigned long long col = (unsigned long long)tl | ((unsigned long long)th << 32);
  // does this time sample's column hold a run of at least m_min channels?  r = AND of col >> 0 .. m_min-1
  unsigned long long r = col;
  if (m_min > (uint32_t)C) r = 0;
  else {
    uint32_t k = 1;
    while (2 * k <= m_min) { r &= r >> k; k *= 2; }
    if (m_min > k) r &= r >> (m_min - k);
  }
  const unsigned long long nw = r ? lof_sir_col_ext<C>(col, eta) : 0ull;
  if (__any_sync(0xffffffffu, nw != 0ull)) {
    lo |= lof_bit_transpose32((uint32_t)nw, lane);
    if (C > 32) hi |= lof_bit_transpose32((uint32_t)(nw >> 32), lane);
    const uint32_t added = __reduce_add_sync(0xffffffffu, (uint32_t)__popcll(nw));
    if (lane == 0) atomicAdd(reinterpret_cast<unsigned long long*>(&stats[s].n_flagged), (unsigned long long)added);
  }
  if (lane < C) co[(size_t)lane * W] = lo;
  if (C > 32) co[(size_t)(lane + 32) * W] = hi;
}

// Frequency direction, any channel count.  One thread per (stream, word column): the C words in[c][w] carry 32 time samples each.
// A run can only grow if it is at least m = ceil(1/eta) channels long: a bit-parallel screen (AND of m consecutive
// words, OR over c) names the time samples that have such a run; only those columns are walked channel by channel.
__global__ void __launch_bounds__(256)
lof_k_sir_freq(const uint32_t* __restrict__ in, uint32_t* __restrict__ out, lof_stream_stats* __restrict__ stats,
               uint64_t n_cols /* S*W */, uint32_t C, uint32_t W, float eta, uint32_t m_min) {
  const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= n_cols) return;
  const uint64_t s = gid / W;
  const uint32_t w = (uint32_t)(gid - s * W);
  const uint32_t* ci = in + s * C * W + w;
  uint32_t* co = out + s * C * W + w;
  // copy, and screen: longrun = OR over c of the AND of the m_min words ending at channel c
  uint32_t longrun = 0;
  for (uint32_t c = 0; c < C; ++c) {
    const uint32_t v = ci[(uint64_t)c * W];
    co[(uint64_t)c * W] = v;
    if (c + 1 >= m_min) {
      uint32_t a = v;
      for (uint32_t k = 1; k < m_min && a; ++k) a &= ci[(uint64_t)(c - k) * W];
      longrun |= a;
    }
  }
  if (m_min > C) longrun = 0;
  uint32_t added = 0;
  while (longrun) {
    const uint32_t b = (uint32_t)__ffs((int)longrun) - 1u;
    longrun &= longrun - 1u;
    const uint32_t bit = 1u << b;
    for (uint32_t c = 0; c < C;) {
      if (!(ci[(uint64_t)c * W] & bit)) { ++c; continue; }
      uint32_t e_ = c;
      while (e_ < C && (ci[(uint64_t)e_ * W] & bit)) ++e_;                 // run [c, e_)
      const uint32_t ext = lof_sir_ext(eta, e_ - c);
      const uint32_t lo = c > ext ? c - ext : 0u, hi = min(e_ + ext, C);
      for (uint32_t q = lo; q < c; ++q) { const uint32_t o = co[(uint64_t)q * W]; if (!(o & bit)) { co[(uint64_t)q * W] = o | bit; ++added; } }
      for (uint32_t q = e_; q < hi; ++q) { const uint32_t o = co[(uint64_t)q * W]; if (!(o & bit)) { co[(uint64_t)q * W] = o | bit; ++added; } }
      c = e_;
    }
  }
  if (added) atomicAdd(reinterpret_cast<unsigned long long*>(&stats[s].n_flagged), (unsigned long long)added);
}
