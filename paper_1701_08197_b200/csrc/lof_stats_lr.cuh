// lof_stats_lr.cuh — statistics of long streams (configs 4, 5: a stream does not fit one SM) in two passes
// over the group's input instead of the three radix passes of lof_stats.cuh, three launches:
//   lof_k_lr_hist     a CTA over consecutive 8192-sample chunks of one stream.  First the plan, recomputed by
//                     every CTA of the stream (same inputs, same result): a strided sample of 256, sorted per
//                     warp -> centre K and scale of a 4096-bin value histogram (rank statistics, so RFI does
//                     not widen the bins).  Then per chunk the shifted sums (fp32 over 8, then fp64, fixed
//                     order) and the value histogram (shared memory, merged into the group slot's by atomics).
//   lof_k_lr_gather   same decomposition.  First, again per CTA, the bin that holds rank floor(N/2) from the
//                     slot's histogram and value bounds that enclose it; then two compares per sample against
//                     those bounds: the bin's samples are appended to the slot's candidate list.
//   lof_k_lr_select2  per stream: mean, stddev from the chunk partials in chunk order; exact rank select among
//                     the candidates (radix select on the float keys, from shared memory); median, thresholds,
//                     stats record; leaves the slot's histogram and counters zeroed for the next group.  If the
//                     histogram could not isolate the median (bin at an end of the range, list overflow,
//                     non-finite sums) the same CTA runs the radix select over the whole stream: slower, same
//                     result.
// The bin function is the fused kernel's (monotone in x, so bins are value-ordered and selection is exact).
#pragma once
#include "lof_common.cuh"
#include "lof_stats.cuh"

#define LOF_LR_NBINS 4096
#define LOF_LR_CAND 32768          // candidate list entries per stream
#define LOF_LR_CTA_LIST 1024       // candidates a gather CTA collects before it reserves list space
#define LOF_LR_STAGE 8192          // ... of which this many can be selected from shared memory

// Byte offset of x's bin in a histogram of LOF_LR_NBINS words: FFMA.SAT, FFMA, LOP (the fused kernel's
// lof_stat_binoff).  t = x*scale + off in bin units, clamped to [0, NBINS-1]; adding 1.5*2^23 leaves round(4 t) in
// the low mantissa bits, whose two lowest are masked off: bin b holds t in [b - 1/8, b + 7/8).  s1, o1 = scale, off
// divided by NBINS - 1.  Monotone in x: bins are value-ordered.
__device__ __forceinline__ uint32_t lof_lr_binoff(float x, float s1, float o1) {
  const float y = __saturatef(fmaf(x, s1, o1));
  return __float_as_uint(fmaf(y, 4.0f * (float)(LOF_LR_NBINS - 1), 12582912.0f)) & (uint32_t)(4 * LOF_LR_NBINS - 4);
}
__device__ __forceinline__ uint32_t lof_lr_bin(float x, float scale, float off) {
  return lof_lr_binoff(x, scale * (1.0f / (float)(LOF_LR_NBINS - 1)), off * (1.0f / (float)(LOF_LR_NBINS - 1))) >> 2;
}

// The histogram placement of stream s, by all 256 threads of a CTA; K, scale, off valid in every thread.
// Contains __syncthreads.
template <class In>
__device__ __forceinline__ void lof_lr_plan(const In& in, uint64_t base, uint64_t N, float* red /*17 floats*/,
                                            float& K, float& scale, float& off) {
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const uint64_t step = N / 256 > 0 ? N / 256 : 1;
  uint64_t idx = (uint64_t)tid * step + ((uint64_t)tid * 7) % step;
  if (idx >= N) idx = N - 1;
  float v = in.ld(base + idx);
  if (!lof_finite(v)) v = 0.f;
#pragma unroll
  for (int k = 2; k <= 32; k <<= 1) {
#pragma unroll
    for (int j = k >> 1; j > 0; j >>= 1) {
      const float o = __shfl_xor_sync(0xffffffffu, v, j);
      const bool up = ((lane & k) == 0) == ((lane & j) == 0);
      v = up ? fminf(v, o) : fmaxf(v, o);
    }
  }
  const float q1 = __shfl_sync(0xffffffffu, v, 8), m0 = __shfl_sync(0xffffffffu, v, 15),
              m1 = __shfl_sync(0xffffffffu, v, 16), q3 = __shfl_sync(0xffffffffu, v, 24);
  if (lane == 0) { red[w] = 0.5f * (m0 + m1); red[8 + w] = q3 - q1; }
  __syncthreads();
  float Ks = 0.f, iqr = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) { Ks += red[i]; iqr += red[8 + i]; }
  Ks *= 0.125f; iqr *= 0.125f;
  float h = 2.5f * iqr;
  if (!(h > 0.f) || !lof_finite(h)) h = fmaxf(fabsf(Ks) * 1e-6f, 1e-30f);
  K = Ks;
  scale = (float)(LOF_LR_NBINS - 2) / (2.0f * h);
  off = fmaf(-(Ks - h), scale, 1.0f);
}

// grid.x = group_streams * n_blk; a CTA takes `cpb` consecutive chunks of one stream (n_blk = ceil(n_chunks /
// cpb)), keeps their histogram in shared memory and merges it into the stream's once: with one chunk per CTA
// the merge would cost as many global atomics as half the samples.  Sums stay per chunk (fixed order).
template <class In>
__global__ void __launch_bounds__(LOF_STATS_THREADS)
lof_k_lr_hist(In in, LofKParams prm, LofStreamState* __restrict__ state, uint32_t* __restrict__ hist,
              uint32_t* __restrict__ ctr, double* __restrict__ partial, uint32_t n_chunks, uint32_t cpb,
              uint32_t n_blk) {
  __shared__ uint32_t sh_hist[LOF_LR_NBINS];
  __shared__ double sh_red[32];
  __shared__ float sh_plan[17];
  const uint32_t sl = blockIdx.x / n_blk;
  const uint32_t blk = blockIdx.x - sl * n_blk;
  const uint32_t s = prm.s0 + sl;
  const uint64_t N = (uint64_t)prm.C * prm.T;
  const uint64_t base = (uint64_t)s * N;
  for (int b = threadIdx.x; b < LOF_LR_NBINS; b += LOF_STATS_THREADS) sh_hist[b] = 0;
  float K, scale, off;
  lof_lr_plan(in, base, N, sh_plan, K, scale, off);
  if (blk == 0 && threadIdx.x == 0) {
    LofStreamState& st = state[s];
    st.shift = (double)K; st.pl_scale = scale; st.pl_off = off;
    st.prefix = 0; st.rank = 0;
  }
  __syncthreads();
  uint32_t bad = 0;
  const uint32_t c_end = min(n_chunks, (blk + 1) * cpb);
  const float s1 = scale * (1.0f / (float)(LOF_LR_NBINS - 1)), o1 = off * (1.0f / (float)(LOF_LR_NBINS - 1));
  unsigned char* hb = reinterpret_cast<unsigned char*>(sh_hist);
  const float2 nK = make_float2(-K, -K);
  // the thread's sums over ALL of the CTA's chunks (fp32 over 8 samples per half of a pair, then fp64), reduced
  // over the CTA once: a block reduction per chunk had cost two of the kernel's twenty instructions per sample
  double sum = 0.0, sumsq = 0.0;
  for (uint32_t chunk = blk * cpb; chunk < c_end; ++chunk) {
    const uint64_t lo = (uint64_t)chunk * LOF_STATS_CHUNK;
    const uint64_t hi = min(N, lo + (uint64_t)LOF_STATS_CHUNK);
    if (((N | lo) & 3) == 0 && hi - lo == LOF_STATS_CHUNK) {
      // full chunk, 16-byte aligned: 4 x 16-byte loads per thread in flight; packed fp32 pairs: .x and .y each take
      // 8 of the 16 samples
#pragma unroll 1
      for (int it = 0; it < LOF_STATS_PER_THREAD / 16; ++it) {
        float xv[16];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          float t4[4];
          in.ld4(base + lo + ((uint64_t)(it * 4 + r) * LOF_STATS_THREADS + threadIdx.x) * 4, t4);
          xv[4 * r] = t4[0]; xv[4 * r + 1] = t4[1]; xv[4 * r + 2] = t4[2]; xv[4 * r + 3] = t4[3];
        }
        float2 ga = make_float2(0.f, 0.f), gq = make_float2(0.f, 0.f);
#pragma unroll
        for (int r = 0; r < 8; ++r) {
          const float2 d = __fadd2_rn(make_float2(xv[2 * r], xv[2 * r + 1]), nK);
          ga = __fadd2_rn(ga, d); gq = __ffma2_rn(d, d, gq);
          atomicAdd(reinterpret_cast<uint32_t*>(hb + lof_lr_binoff(xv[2 * r], s1, o1)), 1u);
          atomicAdd(reinterpret_cast<uint32_t*>(hb + lof_lr_binoff(xv[2 * r + 1], s1, o1)), 1u);
        }
        const float gas = ga.x + ga.y, gqs = gq.x + gq.y;
        // a non-finite sample makes its group's sums non-finite: count exactly only then
        if (!lof_finite(gas) || !lof_finite(gqs)) {
#pragma unroll
          for (int r = 0; r < 16; ++r) bad += lof_finite(xv[r]) ? 0u : 1u;
        }
        sum += (double)ga.x + (double)ga.y; sumsq += (double)gq.x + (double)gq.y;
      }
    } else {
      for (uint64_t i0 = lo + threadIdx.x; i0 < hi; i0 += 8 * LOF_STATS_THREADS) {
        float ga = 0.f, gq = 0.f;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
          const uint64_t i = i0 + (uint64_t)r * LOF_STATS_THREADS;
          if (i < hi) {
            const float x = in.ld(base + i), d = x - K;
            ga += d; gq = fmaf(d, d, gq);
            bad += lof_finite(x) ? 0u : 1u;
            atomicAdd(&sh_hist[lof_lr_bin(x, scale, off)], 1u);
          }
        }
        sum += (double)ga; sumsq += (double)gq;
      }
    }
  }
  {
    // the CTA's sums go to the slot of its first chunk, zeros to its other chunks (lof_k_lr_select2 adds the chunk
    // slots of a stream in chunk order)
    const double rs = lof_block_sum(sum, sh_red);
    const double rq = lof_block_sum(sumsq, sh_red);
    const uint32_t c0 = blk * cpb;
    for (uint32_t chunk = c0 + threadIdx.x; chunk < c_end; chunk += LOF_STATS_THREADS) {
      partial[((size_t)sl * n_chunks + chunk) * 2 + 0] = chunk == c0 ? rs : 0.0;
      partial[((size_t)sl * n_chunks + chunk) * 2 + 1] = chunk == c0 ? rq : 0.0;
    }
  }
  __syncthreads();
  uint32_t* gh = hist + (size_t)sl * LOF_LR_NBINS;
  for (int b = threadIdx.x; b < LOF_LR_NBINS; b += LOF_STATS_THREADS) {
    const uint32_t v = sh_hist[b];
    if (v) atomicAdd(&gh[b], v);
  }
  if (bad) atomicAdd(&ctr[2 * sl], bad);
}

// The bin of the slot's histogram that holds `rank`, by the 256 threads of a CTA: sh[0] = bin, sh[1] = number
// of samples in lower bins (rank beyond the total gives the last bin).  Contains __syncthreads.
__device__ __forceinline__ void lof_lr_find_bin(const uint32_t* __restrict__ gh, uint32_t rank, uint32_t* sh_cnt /*256*/,
                                                uint32_t* sh /*2*/) {
  constexpr int PER = LOF_LR_NBINS / 256;
  const int tid = threadIdx.x;
  uint32_t tot = 0;
#pragma unroll
  for (int j = 0; j < PER; ++j) tot += gh[tid * PER + j];
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
      int b = 0;
      const int g = tid * 8 + j;
      for (; b < PER - 1; ++b) { const uint32_t hv = gh[g * PER + b]; if (acc + hv > rank) break; acc += hv; }
      sh[0] = g * PER + b; sh[1] = acc;
    }
  }
  __syncthreads();
}

template <class In>
__global__ void __launch_bounds__(LOF_STATS_THREADS)
lof_k_lr_gather(In in, LofKParams prm, LofStreamState* __restrict__ state, const uint32_t* __restrict__ hist,
                uint32_t* __restrict__ ctr, float* __restrict__ cand, uint32_t n_chunks, uint32_t cpb, uint32_t n_blk) {
  __shared__ uint32_t sh_cnt[256];
  __shared__ uint32_t sh_sel[2];
  const uint32_t sl = blockIdx.x / n_blk;
  const uint32_t blk = blockIdx.x - sl * n_blk;
  const uint32_t s = prm.s0 + sl;
  LofStreamState& st = state[s];
  const uint64_t N = (uint64_t)prm.C * prm.T;
  const uint64_t base = (uint64_t)s * N;
  const uint32_t* gh = hist + (size_t)sl * LOF_LR_NBINS;
  // every CTA of the stream finds the median's bin itself (same histogram, same result)
  lof_lr_find_bin(gh, (uint32_t)(N / 2), sh_cnt, sh_sel);
  const uint32_t bin = sh_sel[0], before = sh_sel[1], n_b = gh[bin], n_bad = ctr[2 * sl];
  const float scale = st.pl_scale, off = st.pl_off, inv = 1.0f / scale;
  const float v0 = ((float)bin - 0.5f - off) * inv, v1 = ((float)bin + 1.0f - off) * inv;   // (lof_lr_binoff: [b-1/8, b+7/8))
  const float eps = 8e-7f * (fabsf(v0) + fabsf(v1) + fabsf(off) * inv) + 8e-4f * inv;
  const float vmid = 0.5f * (v0 + v1), vhalf = 0.5f * (v1 - v0) + eps;
  const bool fallback = bin == 0 || bin >= LOF_LR_NBINS - 1 || n_b > LOF_LR_CAND || n_bad != 0;
  if (blk == 0 && threadIdx.x == 0) {
    st.bin = bin; st.before = before; st.nb = n_b; st.vmid = vmid; st.vhalf = vhalf;
    st.nonfinite = n_bad; st.fallback = fallback ? 1u : 0u;
  }
  if (fallback) return;
  const uint64_t lo = (uint64_t)blk * cpb * LOF_STATS_CHUNK;
  const uint64_t hi = min(N, lo + (uint64_t)cpb * LOF_STATS_CHUNK);
  uint32_t* ncand = ctr + 2 * sl + 1;

  float* cl = cand + (size_t)sl * LOF_LR_CAND;
  // candidates are collected per CTA in shared memory and appended with one reservation per CTA: thousands of
  // atomics on the one list counter of a stream serialise in L2 (measured: 37 us instead of 10)
  __shared__ float sh_list[LOF_LR_CTA_LIST];
  __shared__ uint32_t sh_n, sh_base;
  if (threadIdx.x == 0) sh_n = 0;
  __syncthreads();
  auto take = [&](float x) {
    if (fabsf(x - vmid) <= vhalf && lof_lr_bin(x, scale, off) == bin) {
      const uint32_t slot = atomicAdd(&sh_n, 1u);
      if (slot < LOF_LR_CTA_LIST) sh_list[slot] = x;
      else {                                              // CTA list full: straight to the stream's list
        const uint32_t g = atomicAdd(ncand, 1u);
        if (g < LOF_LR_CAND) cl[g] = x;
      }
    }
  };
  uint64_t i = lo;
  if (((N | lo) & 3) == 0) {
    const uint64_t hi4 = lo + ((hi - lo) & ~(uint64_t)3);
    // four 16-byte loads in flight per thread, then the compares
    constexpr uint64_t STEP = 4 * LOF_STATS_THREADS;
    uint64_t j = lo + (uint64_t)threadIdx.x * 4;
    for (; j + 3 * STEP < hi4; j += 4 * STEP) {
      float x[4][4];
#pragma unroll
      for (int r = 0; r < 4; ++r) in.ld4(base + j + r * STEP, x[r]);
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const float dmin = fminf(fminf(fabsf(x[r][0] - vmid), fabsf(x[r][1] - vmid)),
                                 fminf(fabsf(x[r][2] - vmid), fabsf(x[r][3] - vmid)));
        if (dmin <= vhalf) { take(x[r][0]); take(x[r][1]); take(x[r][2]); take(x[r][3]); }
      }
    }
    for (; j < hi4; j += STEP) {
      float x[4];
      in.ld4(base + j, x);
      const float dmin = fminf(fminf(fabsf(x[0] - vmid), fabsf(x[1] - vmid)), fminf(fabsf(x[2] - vmid), fabsf(x[3] - vmid)));
      if (dmin <= vhalf) { take(x[0]); take(x[1]); take(x[2]); take(x[3]); }
    }
    i = hi4;
  }
  for (uint64_t j = i + threadIdx.x; j < hi; j += LOF_STATS_THREADS) take(in.ld(base + j));
  __syncthreads();
  const uint32_t n_loc = min(sh_n, (uint32_t)LOF_LR_CTA_LIST);
  if (threadIdx.x == 0 && n_loc) sh_base = atomicAdd(ncand, n_loc);
  __syncthreads();
  for (uint32_t k = threadIdx.x; k < n_loc; k += LOF_STATS_THREADS)
    if (sh_base + k < LOF_LR_CAND) cl[sh_base + k] = sh_list[k];
}

// Exact rank-`rank` element of n values by a 3-pass radix select (11 + 11 + 10 bits of the key), one CTA of
// 256 threads; ld(i) returns value i.  Result valid in every thread.
template <class Ld>
__device__ float lof_lr_radix_select(Ld ld, uint64_t n, uint32_t rank, uint32_t* sh_hist /*2048*/, uint32_t* sh_cnt /*256*/,
                                     uint32_t* sh_sel /*2*/) {
  const int tid = threadIdx.x;
  uint32_t prefix = 0;
  for (int pass = 0; pass < 3; ++pass) {
    for (int b = tid; b < 2048; b += 256) sh_hist[b] = 0;
    __syncthreads();
#pragma unroll 8
    for (uint64_t i = tid; i < n; i += 256) {
      const uint32_t key = lof_key(ld(i));
      if (pass == 0) atomicAdd(&sh_hist[key >> 21], 1u);
      else if (pass == 1) { if ((key >> 21) == prefix) atomicAdd(&sh_hist[(key >> 10) & 2047u], 1u); }
      else { if ((key >> 10) == prefix) atomicAdd(&sh_hist[key & 1023u], 1u); }
    }
    __syncthreads();
    uint32_t loc[8], tot = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { loc[j] = sh_hist[tid * 8 + j]; tot += loc[j]; }
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
        int b = 0;
        const int g = tid * 8 + j;
        for (; b < 7; ++b) { const uint32_t hv = sh_hist[g * 8 + b]; if (acc + hv > rank) break; acc += hv; }
        sh_sel[0] = g * 8 + b; sh_sel[1] = acc;
      }
    }
    __syncthreads();
    const uint32_t bin = sh_sel[0];
    rank -= sh_sel[1];
    prefix = pass == 0 ? bin : (pass == 1 ? ((prefix << 11) | bin) : ((prefix << 10) | bin));
    __syncthreads();
  }
  return lof_unkey(prefix);
}

template <class In>
__global__ void __launch_bounds__(256)
lof_k_lr_select2(In in, LofKParams prm, LofStreamState* __restrict__ state, uint32_t* __restrict__ hist,
                 uint32_t* __restrict__ ctr, const double* __restrict__ partial, uint32_t n_chunks,
                 const float* __restrict__ cand, lof_stream_stats* __restrict__ stats) {
  __shared__ uint32_t sh_hist[2048];
  __shared__ uint32_t sh_cnt[256];
  __shared__ uint32_t sh_sel[2];
  __shared__ double sh_red[32];
  __shared__ float sh_c[LOF_LR_STAGE];
  const uint32_t sl = blockIdx.x, s = prm.s0 + sl;
  const uint64_t N = (uint64_t)prm.C * prm.T;
  const uint64_t base = (uint64_t)s * N;
  LofStreamState& st = state[s];
  const int tid = threadIdx.x;
  // chunk partials reduced in a fixed order: each thread a contiguous run of chunks, then a fixed tree
  {
    const uint32_t per = (n_chunks + 255) / 256;
    double a = 0.0, q = 0.0;
    for (uint32_t c = tid * per; c < min(n_chunks, (tid + 1) * per); ++c) {
      a += partial[((size_t)sl * n_chunks + c) * 2 + 0];
      q += partial[((size_t)sl * n_chunks + c) * 2 + 1];
    }
    a = lof_block_sum(a, sh_red);
    q = lof_block_sum(q, sh_red);
    if (tid == 0) {
      const double n = (double)N;
      double var = (q - a * a / n) / n;
      if (!(var > 0.0)) var = 0.0;
      st.sum = a; st.sumsq = q;
      st.mean = st.shift + a / n;
      st.stddev = sqrt(var);
      sh_sel[0] = (isfinite(a) && isfinite(q)) ? 0u : 1u;
    }
    __syncthreads();
  }
  const bool sums_bad = sh_sel[0] != 0;
  const uint32_t rank = (uint32_t)(N / 2);
  const uint32_t nc = ctr[2 * sl + 1], before = st.before, nb = st.nb, fb = st.fallback;
  __syncthreads();
  // leave the slot's histogram and counters zeroed for the next group that uses it
  {
    uint32_t* gh = hist + (size_t)sl * LOF_LR_NBINS;
    for (int b = tid; b < LOF_LR_NBINS; b += 256) gh[b] = 0;
    if (tid < 2) ctr[2 * sl + tid] = 0;
  }
  const bool direct = fb != 0 || sums_bad || nc != nb || nc > LOF_LR_CAND || before > rank || rank - before >= nc;
  float median;
  if (!direct) {
    const float* cl = cand + (size_t)sl * LOF_LR_CAND;
    if (nc <= LOF_LR_STAGE) {
      // the usual case: the list fits shared memory; one round of global loads, then three passes on chip
#pragma unroll 8
      for (uint32_t i = threadIdx.x; i < nc; i += 256) sh_c[i] = __ldg(cl + i);
      __syncthreads();
      median = lof_lr_radix_select([&](uint64_t i) { return sh_c[i]; }, nc, rank - before, sh_hist, sh_cnt, sh_sel);
    } else {
      median = lof_lr_radix_select([cl](uint64_t i) { return cl[i]; }, nc, rank - before, sh_hist, sh_cnt, sh_sel);
    }
  } else {
    median = lof_lr_radix_select([&](uint64_t i) { return in.ld(base + i); }, N, rank, sh_hist, sh_cnt, sh_sel);
    if (st.nonfinite == 0 && (!isfinite(st.sum) || !isfinite(st.sumsq))) {
      // the fp32 group sums overflowed on finite data: redo them in fp64
      double a = 0.0, q = 0.0;
      for (uint64_t i = threadIdx.x; i < N; i += 256) {
        const double d = (double)in.ld(base + i) - st.shift; a += d; q = fma(d, d, q);
      }
      a = lof_block_sum(a, sh_red);
      q = lof_block_sum(q, sh_red);
      if (threadIdx.x == 0) {
        const double n = (double)N;
        double var = (q - a * a / n) / n;
        if (!(var > 0.0)) var = 0.0;
        st.sum = a; st.sumsq = q; st.mean = st.shift + a / n; st.stddev = sqrt(var);
      }
    }
  }
  __syncthreads();
  if (threadIdx.x < LOF_MAX_LEVELS) {
    // one threshold per thread: threshold_I = median + stddev * factor_I * sensitivity, fp64
    const double sd = st.stddev;
    const uint32_t k = threadIdx.x;
    if (k < prm.n_levels) {
      const double t = (double)median + sd * prm.factor[k] * prm.sensitivity;
      st.thr_d[k] = t;
      st.thr_f[k] = (float)t;
      st.dead_f[k] = lof_dead_level((double)median, sd, prm.factor, prm.sensitivity, k, prm.n_lev_f);
      st.dead_t[k] = lof_dead_level((double)median, sd, prm.factor, prm.sensitivity, k, prm.n_lev_t);
    }
    if (k == 0) {
      st.median = median;
      lof_stream_stats o;
      o.median = median; o.n_nonfinite = st.nonfinite; o.mean = st.mean; o.stddev = sd;
      o.n_flagged = 0;
      stats[s] = o;
    }
  }
}
