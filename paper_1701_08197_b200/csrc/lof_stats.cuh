// lof_stats.cuh — generic (any stream size) statistics path: fp64 shifted sums in a fixed
// reduction order, and the exact median by a 3-pass radix select (11 + 11 + 10 bits) on the
// float bit pattern (PAPER.md:41 uses median and stddev; :120 "efficient O(N) implementation").
// Streams that fit one CTA's shared memory take the fused kernel in lof_fused.cuh instead.
#pragma once
#include "lof_common.cuh"

#define LOF_STATS_THREADS 256
#define LOF_STATS_PER_THREAD 32
#define LOF_STATS_CHUNK (LOF_STATS_THREADS * LOF_STATS_PER_THREAD)

// Pass p of the radix select over one chunk of one stream.  Pass 0 also accumulates the sums.
// grid.x = n_chunks * group_streams.  hist: [group_streams][2048].  partial: [group_streams][n_chunks][2].
template <class In, int PASS>
__global__ void __launch_bounds__(LOF_STATS_THREADS)
lof_k_hist(In in, LofKParams prm, LofStreamState* __restrict__ state, uint32_t* __restrict__ hist,
           double* __restrict__ partial, uint32_t n_chunks) {
  __shared__ uint32_t sh_hist[LOF_HIST_BINS];
  __shared__ double sh_red[32];
  const uint32_t sl = blockIdx.x / n_chunks;            // stream within the group
  const uint32_t chunk = blockIdx.x - sl * n_chunks;
  const uint32_t s = prm.s0 + sl;
  const uint64_t N = (uint64_t)prm.C * prm.T;
  const uint64_t base = (uint64_t)s * N;
  const uint64_t lo = (uint64_t)chunk * LOF_STATS_CHUNK;
  const uint64_t hi = min(N, lo + (uint64_t)LOF_STATS_CHUNK);
  for (int b = threadIdx.x; b < LOF_HIST_BINS; b += LOF_STATS_THREADS) sh_hist[b] = 0;
  __syncthreads();

  uint32_t prefix = 0;
  if (PASS > 0) prefix = state[s].prefix;
  double sum = 0.0, sumsq = 0.0;
  uint32_t bad = 0;
  double K = 0.0;
  if (PASS == 0) K = (double)in.ld(base);               // shift: the stream's first sample
  for (uint64_t i = lo + threadIdx.x; i < hi; i += LOF_STATS_THREADS) {
    const float x = in.ld(base + i);
    const uint32_t key = lof_key(x);
    if (PASS == 0) {
      const double d = (double)x - K;
      sum += d;
      sumsq = fma(d, d, sumsq);
      bad += lof_finite(x) ? 0u : 1u;
      atomicAdd(&sh_hist[key >> 21], 1u);
    } else if (PASS == 1) {
      if ((key >> 21) == prefix) atomicAdd(&sh_hist[(key >> 10) & 2047u], 1u);
    } else {
      if ((key >> 10) == prefix) atomicAdd(&sh_hist[key & 1023u], 1u);
    }
  }
  __syncthreads();
  uint32_t* gh = hist + (size_t)sl * LOF_HIST_BINS;
  for (int b = threadIdx.x; b < LOF_HIST_BINS; b += LOF_STATS_THREADS) {
    const uint32_t v = sh_hist[b];
    if (v) atomicAdd(&gh[b], v);
  }
  if (PASS == 0) {
    const double rs = lof_block_sum(sum, sh_red);
    const double rq = lof_block_sum(sumsq, sh_red);
    if (threadIdx.x == 0) {
      partial[((size_t)sl * n_chunks + chunk) * 2 + 0] = rs;
      partial[((size_t)sl * n_chunks + chunk) * 2 + 1] = rq;
    }
    if (bad) atomicAdd(&state[s].nonfinite, bad);
  }
}

// Thresholds threshold_I = median + stddev * factor_I * sensitivity, fp64.
__device__ __forceinline__ void lof_write_thresholds(LofStreamState& st, const LofKParams& prm) {
  for (uint32_t k = 0; k < prm.n_levels; ++k) {
    const double t = (double)st.median + st.stddev * prm.factor[k] * prm.sensitivity;
    st.thr_d[k] = t;
    st.thr_f[k] = (float)t;
    st.dead_f[k] = lof_dead_level((double)st.median, st.stddev, prm.factor, prm.sensitivity, k, prm.n_lev_f);
    st.dead_t[k] = lof_dead_level((double)st.median, st.stddev, prm.factor, prm.sensitivity, k, prm.n_lev_t);
  }
}

// One CTA per stream of the group: locate the histogram bin holding the wanted rank, narrow the
// prefix, clear the histogram for the next pass.  Pass 0 first reduces the chunk partials in
// chunk order (deterministic) into mean and stddev; pass 2 ends with median and thresholds.
template <class In, int PASS>
__global__ void __launch_bounds__(256)
lof_k_scan(In in, LofKParams prm, LofStreamState* __restrict__ state, uint32_t* __restrict__ hist,
           const double* __restrict__ partial, uint32_t n_chunks, lof_stream_stats* __restrict__ stats) {
  __shared__ uint32_t sh_cnt[256];
  __shared__ uint32_t sh_sel[2];
  const uint32_t sl = blockIdx.x, s = prm.s0 + sl;
  const uint64_t N = (uint64_t)prm.C * prm.T;
  LofStreamState& st = state[s];
  uint32_t* gh = hist + (size_t)sl * LOF_HIST_BINS;
  const int tid = threadIdx.x;
  uint32_t rank;
  if (PASS == 0) {
    rank = (uint32_t)(N / 2);                           // rank floor(N/2), 0-based (S3)
    // chunk partials reduced in a fixed order: each thread a contiguous run of chunks, then a fixed tree
    __shared__ double sh_red2[32];
    const uint32_t per = (n_chunks + 255) / 256;
    double a = 0.0, q = 0.0;
    for (uint32_t c = tid * per; c < min(n_chunks, (tid + 1) * per); ++c) {
      a += partial[((size_t)sl * n_chunks + c) * 2 + 0];
      q += partial[((size_t)sl * n_chunks + c) * 2 + 1];
    }
    a = lof_block_sum(a, sh_red2);
    q = lof_block_sum(q, sh_red2);
    if (tid == 0) {
      const double K = (double)in.ld((uint64_t)s * N);
      const double n = (double)N;
      double var = (q - a * a / n) / n;
      if (!(var > 0.0)) var = 0.0;
      st.shift = K; st.sum = a; st.sumsq = q;
      st.mean = K + a / n;
      st.stddev = sqrt(var);
    }
  } else {
    rank = st.rank;
  }
  // 2048 bins, 8 per thread; warp 0 scans the 256 per-thread totals
  uint32_t loc[8], tot = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) { loc[j] = gh[tid * 8 + j]; tot += loc[j]; }
  sh_cnt[tid] = tot;
  __syncthreads();
  if (tid < 32) {
    uint32_t p[8], sum = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { p[j] = sh_cnt[tid * 8 + j]; sum += p[j]; }
    uint32_t inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o); if (tid >= o) inc += v; }
    const uint32_t exc = inc - sum;
    if ((rank >= exc && rank < inc) || (tid == 31 && rank >= inc)) {
      uint32_t acc = exc; int j = 0;
      for (; j < 7; ++j) { if (acc + p[j] > rank) break; acc += p[j]; }
      sh_sel[0] = tid * 8 + j; sh_sel[1] = acc;
    }
  }
  __syncthreads();
  if (tid == (int)sh_sel[0]) {
    uint32_t acc = sh_sel[1];
    int j = 0;
    for (; j < 7; ++j) { if (acc + loc[j] > rank) break; acc += loc[j]; }
    const uint32_t bin = tid * 8 + j;
    if (PASS == 0) { st.prefix = bin; st.rank = rank - acc; }
    else if (PASS == 1) { st.prefix = (st.prefix << 11) | bin; st.rank = rank - acc; }
    else {
      const uint32_t key = (st.prefix << 10) | bin;
      st.median = lof_unkey(key);
      lof_write_thresholds(st, prm);
      lof_stream_stats o;
      o.median = st.median; o.n_nonfinite = st.nonfinite; o.mean = st.mean; o.stddev = st.stddev;
      o.n_flagged = 0;
      stats[s] = o;
    }
  }
#pragma unroll
  for (int j = 0; j < 8; ++j) gh[tid * 8 + j] = 0;      // ready for the next pass / next block
}

// Clears the per-stream counters that kernels accumulate into with atomics.
__global__ void lof_k_clear_state(LofStreamState* state, uint32_t s0, uint32_t n) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { state[s0 + i].nonfinite = 0; state[s0 + i].prefix = 0; state[s0 + i].rank = 0; }
}


// ---- robust scale ("the MAD"; lof_params.stats_mode = LOF_STATS_MAD, R1)
// Input adapter: d_i = |x_i - median(stream of i)| as float32 (one rounding of the exact difference, like the
// oracle's); the radix-select kernels above then find its rank floor(N/2) element into a second state array.
template <class In>
struct InAbsDev {
  In in;
  const LofStreamState* state;   // of the primary statistics: median per stream
  uint64_t N;                    // samples per stream
  const void* p;                 // (unused; keeps the shape of an input adapter)
  __device__ __forceinline__ float ld(size_t i) const { return fabsf(in.ld(i) - state[i / N].median); }
  static constexpr int kBytes = 4;
};

// stddev := 1.4826 * MAD; thresholds and early-exit levels once more; the stats record reports the scale used.
__global__ void lof_k_mad_apply(LofStreamState* __restrict__ state, const LofStreamState* __restrict__ dev_state,
                                LofKParams prm, lof_stream_stats* __restrict__ stats, uint32_t s0, uint32_t n) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  LofStreamState& st = state[s0 + i];
  if (st.nonfinite) return;
  st.stddev = 1.4826 * (double)dev_state[s0 + i].median;
  lof_write_thresholds(st, prm);
  stats[s0 + i].stddev = st.stddev;
}
