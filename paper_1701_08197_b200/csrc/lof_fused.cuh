// lof_fused.cuh — the fused LOF kernel for streams that fit one SM's shared memory
// (BASELINE.json configs 1-3: 16x256, 64x768, 16x768 float32 = 16 / 192 / 48 KB per stream).
//
// One CTA owns one stream at a time (persistent over streams) and does the whole hot path with a
// single HBM read of the stream and a single write of its flag words:
//   load stream -> shared memory                                    (4 B/sample from HBM)
//   S: statistics: shifted fp32 group sums folded into fp64;
//      exact median by a 4096-bin value histogram around the estimated centre, then an exact
//      rank count among the few samples of the median's bin (radix select as the fallback)
//   F: SumThreshold along frequency: a thread per time column, the
//      column's C window sums in registers, doubled in place level by level
//   T: SumThreshold along time, starting from F's mask: a warp per channel row, each lane holding
//      L = T/32 consecutive samples in registers, neighbours' partial sums by warp shuffle
//   bit-pack + row sums of unflagged samples          (1/8 B/sample to HBM)
// The window test is the paper's "sum with flagged samples replaced by threshold_I > I*threshold_I"
// written as  u > e * threshold_I  with u = sum of the unflagged samples of the window and
// e = their number, both obtained by doubling: X_2I[t] = X_I[t] + X_I[t+I].
// Flags are frozen during an iteration (F8): u and e are rebuilt from level 0 whenever
// an iteration set a new flag.
#pragma once
#include <cuda_fp16.h>

#include "lof_common.cuh"
#include "lof_core.cuh"

// iterations of the time run compiled into the fused kernel: windows up to 2^6 = 64 ("7 iterations", the low end of
// PAPER.md:45's 7-10; BASELINE's configs 1-3 use 32 and 64).  Larger windows on these shapes take the row kernels of
// lof_longrow.cuh: the unrolled levels 7-9 alone were a third of the kernel's code, and two CTAs per SM in different
// phases already miss the instruction cache (no_instruction stalls: 11 % on config 3).
#define LOF_FUSED_KMAX 6
#define LOF_F_NBINS 4096
#define LOF_F_CAP 1024
#define LOF_F_MAGIC 12582912.0f   // 1.5 * 2^23: adding it leaves round-to-nearest(x) in the low mantissa bits

template <int C, int L>
struct LofFusedCfg {
  static constexpr int T = 32 * L, N = C * T, W = L;
  // threads per CTA: the 64-channel column (64 sums + 32 packed counts in registers) allows 12 warps at
  // 168 registers; 24 column groups and 64 rows then split evenly enough over 12 warps
#ifdef LOF_FUSED_NT
  static constexpr int NT = LOF_FUSED_NT;
#else
  static constexpr int NT = (C >= 64) ? 512 : 256;
#endif
#ifdef LOF_FUSED_MINB
  static constexpr int MINB = LOF_FUSED_MINB;
#else
  static constexpr int MINB = (C >= 64) ? 1 : 2;
#endif
  // the next stream's statistics pass runs inside the time pass when the SM holds a single CTA; with two
  // CTAs per SM their phases interleave anyway and the plain order measured faster
#ifdef LOF_STAT_OVERLAP
  static constexpr bool OVL = LOF_STAT_OVERLAP != 0;
#else
  static constexpr bool OVL = MINB == 1;
#endif
  static constexpr size_t smem_bytes =
      (size_t)N * 4 + LOF_F_NBINS * 4 + LOF_F_CAP * 4 + 64 * 8 + (size_t)3 * C * 8 + (64 + 48) * 4 + 256 * 4;
};

struct LofFusedSmem {
  float* xs; uint32_t* hist; float* cand; double* red; double* rowpart; unsigned long long* rowbar; float* thr;
  uint32_t* ctl; uint32_t* part;
  template <int C, int L>
  __device__ static LofFusedSmem make(unsigned char* base) {
    LofFusedSmem s;
    constexpr int N = C * 32 * L;
    s.xs = reinterpret_cast<float*>(base);
    s.hist = reinterpret_cast<uint32_t*>(s.xs + N);
    s.cand = reinterpret_cast<float*>(s.hist + LOF_F_NBINS);
    s.red = reinterpret_cast<double*>(s.cand + LOF_F_CAP);
    s.rowpart = s.red + 64;
    s.rowbar = reinterpret_cast<unsigned long long*>(s.rowpart + 2 * C);
    s.thr = reinterpret_cast<float*>(s.rowbar + C);
    // thr[0..16) thresholds, [16..32) / [32..48) early-exit levels of the two runs, [48] = FLT_MAX (time run off)
    s.ctl = reinterpret_cast<uint32_t*>(s.thr + 64);
    s.part = s.ctl + 48;
    return s;
  }
};
// ctl slots
enum { CT_COLGRP = 12, CT_ROW = 11, CT_NCAND = 0, CT_BIN, CT_BEFORE, CT_MEDBITS, CT_NFLAG, CT_BAD, CT_SELP, CT_SELACC, CT_PREFIX, CT_RANK, CT_FOUND, CT_SROW = 13, CT_TICKET = 14 /* and 15 */ };

// Diagnostics live in a context-owned array `diag` (LOF_DIAG_WORDS words, lof_fused_counters): how the median of
// each stream was found: [0] rank count among the samples of the median's bin, [1] radix select among them (a
// crowded bin), [2] radix select over the whole stream, [3] stream with non-finite samples.
#define LOF_DIAG_WORDS 16
#define LOF_DIAG_TICKET 6         // work queue of the persistent CTAs: streams handed out beyond the fixed first two
// Find the bin holding `rank` in hist[NB] (NB a multiple of 1024, any blockDim that is a multiple of 32).
// Results in ctl[CT_BIN] (bin) and ctl[CT_BEFORE] (number of entries in lower bins); rank beyond the total
// gives the last bin.  Groups of 32 bins are summed by warps (one bin per lane: no bank conflicts), warp 0
// scans the group sums and then the 32 bins of the group it lands in.
template <int NB>
__device__ __forceinline__ void lof_find_bin_sums(const uint32_t* hist, uint32_t* part /*>= NB/32*/) {
  constexpr int NG = NB / 32;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int g = w; g < NG; g += nw) {
    const uint32_t s = __reduce_add_sync(0xffffffffu, hist[g * 32 + lane]);
    if (lane == 0) part[g] = s;
  }
}
// the scan over the group sums and then over the 32 bins of the group that holds `rank`; one warp (all 32 lanes)
template <int NB>
__device__ __forceinline__ void lof_find_bin_scan(const uint32_t* hist, uint32_t rank, const uint32_t* part, uint32_t* ctl) {
  constexpr int NG = NB / 32, PERL = NG / 32;
  const int lane = threadIdx.x & 31;
  uint32_t p[PERL], s = 0;
#pragma unroll
  for (int j = 0; j < PERL; ++j) { p[j] = part[lane * PERL + j]; s += p[j]; }
  uint32_t inc = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
  const uint32_t exc = inc - s;
  const bool mine = (rank >= exc && rank < inc) || (lane == 31 && rank >= inc);
  uint32_t acc = exc; int j = 0;
#pragma unroll
  for (int jj = 0; jj < PERL - 1; ++jj) { if (j == jj && acc + p[jj] <= rank) { acc += p[jj]; j = jj + 1; } }
  const int src = __ffs(__ballot_sync(0xffffffffu, mine)) - 1;
  const int g = __shfl_sync(0xffffffffu, lane * PERL + j, src);
  acc = __shfl_sync(0xffffffffu, acc, src);
  const uint32_t hv = hist[g * 32 + lane];
  uint32_t binc = hv;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, binc, o); if (lane >= o) binc += v; }
  const uint32_t hit = __ballot_sync(0xffffffffu, acc + binc > rank);
  const int bl = hit ? __ffs(hit) - 1 : 31;
  const uint32_t before = acc + __shfl_sync(0xffffffffu, binc - hv, bl);
  if (lane == 0) { ctl[CT_BIN] = g * 32 + bl; ctl[CT_BEFORE] = before; }
}
template <int NB>
__device__ void lof_find_bin(const uint32_t* hist, uint32_t rank, uint32_t* part /*>= NB/32*/, uint32_t* ctl) {
  lof_find_bin_sums<NB>(hist, part);
  __syncthreads();
  if (threadIdx.x < 32) lof_find_bin_scan<NB>(hist, rank, part, ctl);
  __syncthreads();
}

// Exact rank-`rank` element of xs[0..N) by a 3-pass radix select (11+11+10 bits of the key) with a
// shared-memory histogram: the fallback when the value histogram cannot isolate the median.
template <int NT>
__device__ float lof_radix_select_smem(const float* xs, int N, uint32_t rank, uint32_t* hist, uint32_t* part,
                                       uint32_t* ctl) {
  uint32_t prefix = 0;
  for (int pass = 0; pass < 3; ++pass) {
    for (int b = threadIdx.x; b < 2048; b += NT) hist[b] = 0;
    __syncthreads();
    for (int i = threadIdx.x; i < N; i += NT) {
      const uint32_t key = lof_key(xs[i]);
      if (pass == 0) atomicAdd(&hist[key >> 21], 1u);
      else if (pass == 1) { if ((key >> 21) == prefix) atomicAdd(&hist[(key >> 10) & 2047u], 1u); }
      else { if ((key >> 10) == prefix) atomicAdd(&hist[key & 1023u], 1u); }
    }
    __syncthreads();
    lof_find_bin<2048>(hist, rank, part, ctl);
    const uint32_t bin = ctl[CT_BIN];
    rank -= ctl[CT_BEFORE];
    prefix = pass == 0 ? bin : (pass == 1 ? ((prefix << 11) | bin) : ((prefix << 10) | bin));
    __syncthreads();
  }
  return lof_unkey(prefix);
}

// Block reduction of two doubles at once (fixed order); result valid in every thread.
template <int NT>
__device__ __forceinline__ void lof_block_sum2(double& a, double& b, double* red /*64*/) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  constexpr int NW = NT / 32;
  a = lof_warp_sum(a); b = lof_warp_sum(b);
  __syncthreads();
  if (lane == 0) { red[w] = a; red[32 + w] = b; }
  __syncthreads();
  double ra = 0.0, rb = 0.0;
#pragma unroll
  for (int i = 0; i < NW; ++i) { ra += red[i]; rb += red[32 + i]; }
  a = ra; b = rb;
  __syncthreads();
}

// ---- S: statistics, organised by channel row so that the pass over a row can run
// anywhere: for the first stream of a CTA right after the load, for every later stream inside the time
// pass of the stream before it, on rows whose prefetch has landed.
//
// LofStatPlan places the value histogram of one stream; every thread holds the same values.
struct LofStatPlan {
  float K, scale, off, s1, o1;
};
__device__ __forceinline__ uint32_t lof_stat_binoff(float x, float s1, float o1) {
  const float y = __saturatef(fmaf(x, s1, o1));
  return __float_as_uint(fmaf(y, 4.0f * (float)(LOF_F_NBINS - 1), LOF_F_MAGIC)) & (uint32_t)(4 * LOF_F_NBINS - 4);
}
__device__ __forceinline__ uint32_t lof_stat_bin(float x, const LofStatPlan& pl) { return lof_stat_binoff(x, pl.s1, pl.o1) >> 2; }

// Plan from one strided sample per thread: each warp sorts its 32 samples (bitonic, shuffles) and reads off
// their median and interquartile range; the plan centres the histogram on the mean of the warp medians with
// a half-width of 2.5 mean interquartile ranges.  Rank statistics, because RFI of 100 sigma in a few per cent
// of the samples inflates a plain standard deviation tenfold and the bins with it.  Any K and any range give
// the same exact results; they only decide how fast the median is found.  Contains one __syncthreads; call it
// right after a block barrier, and put another one before anything else writes `red`.
template <int NT>
__device__ __forceinline__ LofStatPlan lof_stat_plan(float v, float* red /* >= 2*NT/32 floats */) {
  constexpr int NW = NT / 32;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (!lof_finite(v)) v = 0.f;
#pragma unroll
  for (int k = 2; k <= 32; k <<= 1) {
#pragma unroll
    for (int j = k >> 1; j > 0; j >>= 1) {
      const float o = __shfl_xor_sync(0xffffffffu, v, j);
      const bool up = ((lane & k) == 0) == ((lane & j) == 0);     // keep the smaller of the pair
      v = up ? fminf(v, o) : fmaxf(v, o);
    }
  }
  const float q1 = __shfl_sync(0xffffffffu, v, 8), m0 = __shfl_sync(0xffffffffu, v, 15),
              m1 = __shfl_sync(0xffffffffu, v, 16), q3 = __shfl_sync(0xffffffffu, v, 24);
  // (no barrier here: every caller comes from one, and nothing writes `red` between that and this point)
  if (lane == 0) { red[w] = 0.5f * (m0 + m1); red[NW + w] = q3 - q1; }
  __syncthreads();
  float K = 0.f, iqr = 0.f;
#pragma unroll
  for (int i = 0; i < NW; ++i) { K += red[i]; iqr += red[NW + i]; }
  K *= 1.0f / NW; iqr *= 1.0f / NW;
  // (none here either: the next writer of `red`, lof_stat_finalize, is behind the callers' next barrier)
  float h = 2.5f * iqr;                                   // Gaussian: +-3.4 sigma; exponential: 96 % of the samples
  if (!(h > 0.f) || !lof_finite(h)) h = fmaxf(fabsf(K) * 1e-6f, 1e-30f);
  LofStatPlan pl;
  pl.K = K;
  pl.scale = (float)(LOF_F_NBINS - 2) / (2.0f * h);
  pl.off = fmaf(-(K - h), pl.scale, 1.0f);               // x = K-h -> 1, x = K+h -> NBINS-1
  pl.s1 = pl.scale * (1.0f / (float)(LOF_F_NBINS - 1));
  pl.o1 = pl.off * (1.0f / (float)(LOF_F_NBINS - 1));
  return pl;
}

// One channel row of the stream in shared memory, by one warp: partial sums of d = x-K and d^2 (fp32 over
// groups of 8, then fp64, fixed order) and the row's samples into the value histogram.  Row partials land
// in rowpart[2c], [2c+1].
template <int C, int L>
__device__ __forceinline__ void lof_stat_row(const LofFusedSmem& sm, int c, const LofStatPlan& pl, int lane) {
  constexpr int T = 32 * L;
  const float4* rp = reinterpret_cast<const float4*>(sm.xs + c * T);
  const float s1 = pl.s1, o1 = pl.o1;
  const float2 nK = make_float2(-pl.K, -pl.K);
  unsigned char* hist = reinterpret_cast<unsigned char*>(sm.hist);
  double da = 0.0, dq = 0.0;
  float2 ga = make_float2(0.f, 0.f), gq = make_float2(0.f, 0.f);   // packed: .x and .y each take 8 samples a group
#pragma unroll
  for (int q = 0; q < L / 4; ++q) {
    const float4 v = rp[q * 32 + lane];
    const float2 d0 = __fadd2_rn(make_float2(v.x, v.y), nK), d1 = __fadd2_rn(make_float2(v.z, v.w), nK);
    ga = __fadd2_rn(__fadd2_rn(ga, d0), d1);
    gq = __ffma2_rn(d1, d1, __ffma2_rn(d0, d0, gq));
    atomicAdd(reinterpret_cast<uint32_t*>(hist + lof_stat_binoff(v.x, s1, o1)), 1u);
    atomicAdd(reinterpret_cast<uint32_t*>(hist + lof_stat_binoff(v.y, s1, o1)), 1u);
    atomicAdd(reinterpret_cast<uint32_t*>(hist + lof_stat_binoff(v.z, s1, o1)), 1u);
    atomicAdd(reinterpret_cast<uint32_t*>(hist + lof_stat_binoff(v.w, s1, o1)), 1u);
    if ((q & 3) == 3 || q == L / 4 - 1) {
      da += (double)ga.x + (double)ga.y; dq += (double)gq.x + (double)gq.y;
      ga = make_float2(0.f, 0.f); gq = make_float2(0.f, 0.f);
    }
  }
  da = lof_warp_sum(da); dq = lof_warp_sum(dq);
  if (lane == 0) { sm.rowpart[2 * c] = da; sm.rowpart[2 * c + 1] = dq; }
}

// After every row of the stream went through lof_stat_row (and a __syncthreads): mean and stddev from the
// row partials in row order, the exact median (rank floor(N/2), S3) from the histogram and the
// gathered samples, thresholds, the stats record.  Leaves the histogram zeroed and the work counters reset for
// the passes that follow.  Returns the number of non-finite samples (then everything else is unspecified,
// DESIGN.md S6); `median_out` is valid in every thread.
template <int C, int L>
__device__ uint32_t lof_stat_finalize(const LofFusedSmem& sm, const LofKParams& prm, const LofStatPlan& pl,
                                      lof_stream_stats* out, float& median_out, unsigned long long* diag,
                                      uint64_t* nflag_prev = nullptr /* n_flagged of the stream just flagged */) {
  using Cfg = LofFusedCfg<C, L>;
  constexpr int N = Cfg::N, NT = Cfg::NT, NW = NT / 32;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t* part = sm.part;
  const float4* x4 = reinterpret_cast<const float4*>(sm.xs);
  // The steps below are latency chains between block barriers (12 k cycles per stream when each had its own): they
  // are paired so that one barrier serves two of them.  Here: the row partials added by the last warp (which also
  // resets the work counters of the passes that follow: nothing reads them inside this function), and the group
  // sums of the histogram for the bin search by every warp.
  if (warp == NW - 1) {
    double a = 0.0, q = 0.0;
#pragma unroll
    for (int c = lane; c < C; c += 32) { a += sm.rowpart[2 * c]; q += sm.rowpart[2 * c + 1]; }
    a = lof_warp_sum(a); q = lof_warp_sum(q);
    if (lane == 0) {
      sm.red[0] = a; sm.red[1] = q;
      if (nflag_prev) *nflag_prev = sm.ctl[CT_NFLAG];     // (before the counter is reset for the next stream)
      sm.ctl[CT_NCAND] = 0; sm.ctl[CT_BAD] = 0; sm.ctl[CT_FOUND] = 0;
      sm.ctl[CT_NFLAG] = 0; sm.ctl[CT_ROW] = 0; sm.ctl[CT_COLGRP] = 0; sm.ctl[CT_SROW] = 0;
    }
  }
  lof_find_bin_sums<LOF_F_NBINS>(sm.hist, part);
  __syncthreads();
  double da = sm.red[0], dq = sm.red[1];
  uint32_t n_bad = 0;
  if (!isfinite(da) || !isfinite(dq)) {
    // rare: a non-finite sample, or d^2 overflowed fp32: count exactly and redo the sums in fp64
    uint32_t bad = 0; double a2 = 0.0, q2 = 0.0;
    for (int i = tid; i < N; i += NT) {
      const float x = sm.xs[i];
      bad += lof_finite(x) ? 0u : 1u;
      const double d = (double)x - (double)pl.K; a2 += d; q2 = fma(d, d, q2);
    }
    if (bad) atomicAdd(&sm.ctl[CT_BAD], bad);
    lof_block_sum2<NT>(a2, q2, sm.red);
    da = a2; dq = q2;
    n_bad = sm.ctl[CT_BAD];
  }
  LOF_PROF_T(ta);
  const uint32_t rank = N / 2;
  float median = 0.f;
  int how = 3;
  bool dp_done = false, fast = false;
  if (n_bad == 0) {
    if (tid < 32) lof_find_bin_scan<LOF_F_NBINS>(sm.hist, rank, part, sm.ctl);
    __syncthreads();
    LOF_PROF_T(tb);
    const uint32_t bin = sm.ctl[CT_BIN], before = sm.ctl[CT_BEFORE];
    const uint32_t n_b = sm.hist[bin];
    bool ok = bin > 0 && bin < LOF_F_NBINS - 1 && n_b <= LOF_F_CAP;
    if (ok) {
      // gather the samples of the median's bin: two compares per sample against value bounds that enclose
      // the bin (a few ulps wide of it), then the exact bin function on the few that pass.  The last warp
      // does the fp64 end of mean and stddev meanwhile (a long dependent chain that would otherwise sit
      // on one thread between two barriers).
      if (tid >= NT - 32) {
        double sd = 0.0;
        if (lane == 0) {
          const double n = (double)N;
          double var = (dq - da * da / n) / n;
          if (!(var > 0.0)) var = 0.0;
          sd = sqrt(var);
          sm.red[2] = (double)pl.K + da / n; sm.red[3] = sd;
        }
        // ... and the part of each threshold that does not need the median: stddev * factor_I
        sd = __shfl_sync(0xffffffffu, sd, 0);
        if ((uint32_t)lane < prm.n_levels) sm.red[8 + lane] = sd * prm.factor[lane];
      } else {
        const float inv = 1.0f / pl.scale;
        const float v0 = ((float)bin - 0.5f - pl.off) * inv, v1 = ((float)bin + 1.0f - pl.off) * inv;
        const float eps = 8e-7f * (fabsf(v0) + fabsf(v1) + fabsf(pl.off) * inv) + 8e-4f * inv;
        const float vmid = 0.5f * (v0 + v1), vhalf = 0.5f * (v1 - v0) + eps;
        // the four samples of a chunk near the bin: membership without branches (range and exact bin function),
        // then one reservation in the candidate list for the chunk's members (there are a few dozen per stream)
        auto take4 = [&](const float4& v) {
          const float xq[4] = {v.x, v.y, v.z, v.w};
          uint32_t mk = 0;
#pragma unroll
          for (int k = 0; k < 4; ++k)
            mk |= ((uint32_t)(fabsf(xq[k] - vmid) <= vhalf) & (uint32_t)(lof_stat_bin(xq[k], pl) == bin)) << k;
          if (mk) {
            uint32_t slot = atomicAdd(&sm.ctl[CT_NCAND], (uint32_t)__popc(mk));
#pragma unroll
            for (int k = 0; k < 4; ++k)
              if ((mk >> k) & 1u) { if (slot < LOF_F_CAP) sm.cand[slot] = xq[k]; ++slot; }
          }
        };
        // pass 1, no branches: which of the thread's chunks have a sample within the bounds (one bit per chunk;
        // a thread takes N/4/(NT-32) <= 64 chunks).  pass 2: the few chunks that have (about one in 250).
        constexpr int STR = NT - 32;
        static_assert((N / 4 + STR - 1) / STR <= 64, "one hit bit per chunk of a thread");
        unsigned long long hits = 0;
        constexpr int NCH = (N / 4 + STR - 1) / STR;        // chunks per thread (the last one may not exist)
#pragma unroll
        for (int k0 = 0; k0 < NCH; k0 += 8) {               // eight 16-byte loads in flight, no branch
          float4 v[8];
#pragma unroll
          for (int r = 0; r < 8; ++r) if (k0 + r < NCH) v[r] = x4[min(tid + (k0 + r) * STR, N / 4 - 1)];
#pragma unroll
          for (int r = 0; r < 8; ++r) if (k0 + r < NCH) {
            const float dmin = fminf(fminf(fabsf(v[r].x - vmid), fabsf(v[r].y - vmid)),
                                     fminf(fabsf(v[r].z - vmid), fabsf(v[r].w - vmid)));
            hits |= ((dmin <= vhalf) & (tid + (k0 + r) * STR < N / 4) ? 1ull : 0ull) << (k0 + r);
          }
        }
        while (hits) {
          const int k = __ffsll((long long)hits) - 1;
          hits &= hits - 1;
          take4(x4[tid + k * STR]);
        }
      }
      dp_done = true;
      __syncthreads();
      LOF_PROF_T(tg);
      LOF_PROF_ADD(5, tb, tg);
      // the candidate with exactly (rank - before) candidates ordered before it
      const uint32_t want = rank - before, nc = sm.ctl[CT_NCAND];
      if (nc != n_b) ok = false;                         // bounds too tight (cannot happen): stay exact anyway
      else if (nc <= 256) {
        how = 0;
        // G threads per candidate i (there are a few dozen candidates; G = 8 or 4 then), each over every G-th
        // candidate j: less = #{j : c_j < c_i, or equal and j < i}, added over the group by shuffles.  The
        // histogram is zeroed for the next stream under the same barrier (its last read was hist[bin] above).
        {
          uint32_t lg = 0;
          while (lg < 5 && (nc << (lg + 1)) <= (uint32_t)NT) ++lg;
          const uint32_t G = 1u << lg, i = (uint32_t)tid >> lg, sub = (uint32_t)tid & (G - 1);
          const float v = sm.cand[i < nc ? i : 0];
          uint32_t less = 0;
          if (i < nc) {
#pragma unroll 4
            for (uint32_t j = sub; j < nc; j += G) {
              const float w = sm.cand[j];
              less += (w < v || (w == v && j < i)) ? 1u : 0u;
            }
          }
          for (uint32_t o = G >> 1; o > 0; o >>= 1) less += __shfl_xor_sync(0xffffffffu, less, o);
          if (i < nc && sub == 0 && less == want) { sm.ctl[CT_MEDBITS] = __float_as_uint(v); sm.ctl[CT_FOUND] = 1; }
        }
        for (int b = tid; b < LOF_F_NBINS; b += NT) sm.hist[b] = 0;
        __syncthreads();
        ok = sm.ctl[CT_FOUND] != 0;
        median = __uint_as_float(sm.ctl[CT_MEDBITS]);
        fast = ok;
      } else {
        how = 1;
        median = lof_radix_select_smem<NT>(sm.cand, (int)nc, want, sm.hist, part, sm.ctl);
      }
    }
    if (!ok) { how = 2; median = lof_radix_select_smem<NT>(sm.xs, N, rank, sm.hist, part, sm.ctl); }
  }
  LOF_PROF_T(tc);
  if (fast) {
    // the usual case: every warp forms the thresholds and early-exit levels itself (same inputs, same bits) and
    // goes on to the frequency pass without another block barrier
    float t = INFINITY;
    if ((uint32_t)lane < prm.n_levels) {
      t = (float)((double)median + sm.red[8 + lane] * prm.sensitivity);
      sm.thr[lane] = t;
    }
    // early-exit levels (lof_dead_level_f: the minimum over the later thresholds of the run) by suffix minima
    // over the lanes
    float mf = (uint32_t)lane < prm.n_lev_f ? t : INFINITY, mt = (uint32_t)lane < prm.n_lev_t ? t : INFINITY;
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
      const float a = __shfl_down_sync(0xffffffffu, mf, o), b = __shfl_down_sync(0xffffffffu, mt, o);
      if (lane + o < 32) { mf = fminf(mf, a); mt = fminf(mt, b); }
    }
    mf = __shfl_down_sync(0xffffffffu, mf, 1); mt = __shfl_down_sync(0xffffffffu, mt, 1);
    if ((uint32_t)lane < prm.n_levels) {
      sm.thr[16 + lane] = (uint32_t)lane + 1 >= prm.n_lev_f ? 3.0e38f : (mf > 0.f ? mf * (1.0f - 3e-6f) : -1.0e34f);
      sm.thr[32 + lane] = (uint32_t)lane + 1 >= prm.n_lev_t ? 3.0e38f : (mt > 0.f ? mt * (1.0f - 3e-6f) : -1.0e34f);
    }
    if (lane == 0) sm.thr[48] = LOF_BELOW_MARK;
    if (tid == 0) {
      lof_stream_stats o;
      o.median = median; o.n_nonfinite = 0; o.mean = sm.red[2]; o.stddev = sm.red[3];
      o.n_flagged = 0;
      *out = o;
      atomicAdd(&diag[0], 1ull);
    }
    __syncwarp();
    LOF_PROF_T(te);
    median_out = median;
    return 0;
  }
  for (int b = tid; b < LOF_F_NBINS; b += NT) sm.hist[b] = 0;
  if (tid < 32) {
    double mean, stddev;
    if (dp_done) { mean = sm.red[2]; stddev = sm.red[3]; }
    else {
      const double n = (double)N;
      double var = (dq - da * da / n) / n;
      if (!(var > 0.0)) var = 0.0;
      mean = (double)pl.K + da / n; stddev = sqrt(var);
    }
    if ((uint32_t)lane < prm.n_levels)                   // threshold_I, one per lane
      sm.thr[lane] = (float)((double)median + stddev * prm.factor[lane] * prm.sensitivity);
    __syncwarp();
    if ((uint32_t)lane < prm.n_levels) {                 // early-exit levels (lof_dead_level_f), from the fp32 thresholds
      sm.thr[16 + lane] = lof_dead_level_f(sm.thr, lane, prm.n_lev_f);
      sm.thr[32 + lane] = lof_dead_level_f(sm.thr, lane, prm.n_lev_t);
    }
    if (lane == 0) sm.thr[48] = LOF_BELOW_MARK;            // "threshold" of a run that is switched off
    if (lane == 0) {
      lof_stream_stats o;
      o.median = median; o.n_nonfinite = n_bad; o.mean = mean; o.stddev = stddev;
      o.n_flagged = n_bad ? (uint64_t)N : 0;
      *out = o;
      sm.ctl[CT_NFLAG] = 0; sm.ctl[CT_ROW] = 0; sm.ctl[CT_COLGRP] = 0; sm.ctl[CT_SROW] = 0;
      atomicAdd(&diag[how], 1ull);
    }
  }
  __syncthreads();
  LOF_PROF_T(td);
  median_out = median;
  return n_bad;
}

// Statistics of a stream that is completely in shared memory (first stream of a CTA): plan from a strided
// sample, every row through lof_stat_row, then lof_stat_finalize.
template <int C, int L>
__device__ uint32_t lof_stat_whole(const LofFusedSmem& sm, const LofKParams& prm, float sample,
                                   lof_stream_stats* out, float& median_out, unsigned long long* diag,
                                   uint64_t* nflag_prev = nullptr) {
  using Cfg = LofFusedCfg<C, L>;
  constexpr int NT = Cfg::NT, NW = NT / 32;
  const LofStatPlan pl = lof_stat_plan<NT>(sample, reinterpret_cast<float*>(sm.red));
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int c = warp; c < C; c += NW) lof_stat_row<C, L>(sm, c, pl, lane);
  __syncthreads();
  return lof_stat_finalize<C, L>(sm, prm, pl, out, median_out, diag, nflag_prev);
}

// Shared-memory layout of a row: float4 chunk g is stored at g ^ ((g >> 3) & 1): adjacent float4 pairs swapped in
// every odd group of 32 floats.  Column access (32 consecutive t) stays conflict-free, and the time pass's
// per-lane runs of L consecutive floats (lane stride 96 B for L = 24) become conflict-free LDS.128 as well.
__device__ __forceinline__ int lof_swz_chunk(int g) { return g ^ ((g >> 3) & 1); }
__device__ __forceinline__ int lof_swz_elem(int t) { return t ^ (((t >> 5) & 1) << 2); }

// 16-byte asynchronous global -> shared copy (LDGSTS); completion via lof_cp_async_wait_all().
__device__ __forceinline__ void lof_cp_async16(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void lof_cp_async_wait_all() {
  asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}

// mbarrier per channel row: the 32 lanes that prefetch a row of the next stream make the row's barrier track
// their copies; any warp can then wait for the row (cp.async.wait_group would only serve the issuing thread).
__device__ __forceinline__ void lof_mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void lof_mbar_arrive_on_copies(unsigned long long* bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void lof_mbar_wait(unsigned long long* bar, unsigned parity) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile(
      "{\n.reg .pred p;\nLOF_MBAR_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@!p bra LOF_MBAR_WAIT_%=;\n}" ::"r"(a), "r"(parity) : "memory");
}

// ---- F: SumThreshold along frequency ("We first flag in the frequency direction"): the column
// cores of lof_core.cuh on the stream in shared memory.  A flagged sample is marked IN the shared-memory copy
// of the stream (LOF_MARK): that is how the time run, which starts from this run's mask (reading F10), sees it.
template <int C, int L>
__device__ void lof_fused_freq(const LofFusedSmem& sm, uint32_t n_lev_f) {
  using Cfg = LofFusedCfg<C, L>;
  constexpr int T = Cfg::T;
  const int lane = threadIdx.x & 31;
#pragma unroll 1
  for (;;) {
    // groups of 32 columns are handed out dynamically (restarts and early exits make their cost uneven)
    int g = 0;
    if (lane == 0) g = (int)atomicAdd(&sm.ctl[CT_COLGRP], 1u);
    g = __shfl_sync(0xffffffffu, g, 0);
    if (g >= T / 32) break;
    const int col = g * 32 + lane;
    float* cp = sm.xs + lof_swz_elem(col);
    uint64_t fb = lof_col_flag<C>([cp](int c) { return cp[c * T]; }, sm.thr, sm.thr + 16, (int)n_lev_f);
    while (fb) { const int c = __ffsll((long long)fb) - 1; cp[c * T] = LOF_MARK; fb &= fb - 1; }
  }
}

// 64 channels: two lanes per column (lof_pcol_flag), 16 columns per task.
template <int C, int L>
__device__ void lof_fused_freq_pair(const LofFusedSmem& sm, uint32_t n_lev_f) {
  static_assert(C == 64, "two lanes per column: 64 channels");
  using Cfg = LofFusedCfg<C, L>;
  constexpr int T = Cfg::T;
  const int lane = threadIdx.x & 31, h = lane >> 4, p = lane & 15;
#pragma unroll 1
  for (;;) {
    int g = 0;
    if (lane == 0) g = (int)atomicAdd(&sm.ctl[CT_COLGRP], 1u);
    g = __shfl_sync(0xffffffffu, g, 0);
    if (g >= T / 16) break;
    const int col = g * 16 + p;
    float* cp = sm.xs + (32 * h) * T + lof_swz_elem(col);
    uint32_t fb = lof_pcol_flag([cp](int j) { return cp[j * T]; }, sm.thr, sm.thr + 16, (int)n_lev_f, h);
    while (fb) { const int j = __ffs((int)fb) - 1; cp[j * T] = LOF_MARK; fb &= fb - 1; }
  }
}

// ---- T: SumThreshold along time (lof_row_flag): one warp per channel row, then bit-pack and row sums.
template <int C, int L>
__device__ void lof_fused_time(const LofFusedSmem& sm, const LofKParams& prm, uint32_t s,
                               uint32_t* __restrict__ flags, double* __restrict__ rowsum,
                               uint32_t* __restrict__ rowcnt, const float* __restrict__ this_stream,
                               const float* __restrict__ next_stream,
                               const LofStatPlan& plan_next, unsigned bar_parity) {
  using Cfg = LofFusedCfg<C, L>;
  constexpr int T = Cfg::T, NT = Cfg::NT, W = Cfg::W, NW = NT / 32;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t nlt = prm.n_lev_t;
  uint32_t n_flag_acc = 0;
  (void)warp; (void)NW;
#pragma unroll 1
  for (;;) {
    // rows are handed out dynamically: their cost varies with the number of restarts
    int c = 0;
    if (lane == 0) c = (int)atomicAdd(&sm.ctl[CT_ROW], 1u);
    c = __shfl_sync(0xffffffffu, c, 0);
    if (c >= C) break;
    // the row from shared memory (samples the frequency run flagged hold LOF_MARK there: the run starts from its
    // mask, F10); as soon as it is in registers its slot takes the next stream's row.  A restart re-reads the raw
    // row from global memory (every flag so far, the frequency run's included, is then in fb).
    const float4* rp = reinterpret_cast<const float4*>(sm.xs + c * T);
    const float4* gp = reinterpret_cast<const float4*>(this_stream + c * T);
    auto load = [&](float2 (&x2)[L / 2], bool again) {
#pragma unroll
      for (int q = 0; q < L / 4; ++q) {
        const float4 v = again ? __ldg(gp + lane * (L / 4) + q) : rp[lof_swz_chunk(lane * (L / 4) + q)];
        x2[2 * q] = make_float2(v.x, v.y); x2[2 * q + 1] = make_float2(v.z, v.w);
      }
      if (!again && next_stream) {
        float4* dst = reinterpret_cast<float4*>(sm.xs + c * T);
        const float4* src = reinterpret_cast<const float4*>(next_stream + c * T);
#pragma unroll
        for (int q = 0; q < L / 4; ++q) lof_cp_async16(dst + lof_swz_chunk(q * 32 + lane), src + q * 32 + lane);
        lof_mbar_arrive_on_copies(sm.rowbar + c);
      }
    };
    // With the time direction off (n_lev_t = 0) level 0 alone runs, with a threshold only the marks exceed: it
    // turns them into the mask and sums the rest.
    uint32_t fb = 0;
    float lane_sum = 0.f;
    lof_row_flag<L, LOF_FUSED_KMAX>(load, fb, nlt > 0 ? sm.thr : sm.thr + 48, sm.thr + 32, nlt > 0 ? (int)nlt : 1, lane, lane_sum);
    // bit-pack: word w of the row = bits [32w, 32w+32) gathered from the lanes' L-bit masks
    {
      const int q0 = (32 * lane) / L, r0 = 32 * lane - L * q0;
      uint32_t word = 0;
      constexpr int NI = (31 + L) / L + 1;
#pragma unroll
      for (int i = 0; i < NI; ++i) {
        const int src = q0 + i;
        uint32_t v = __shfl_sync(0xffffffffu, fb, src & 31);
        if (src > 31) v = 0;
        const int sh = i * L - r0;
        if (sh < 32) word |= sh >= 0 ? (v << sh) : (v >> (-sh));
      }
      if (lane < W) flags[((size_t)s * C + c) * W + lane] = word;
    }
    // row sum of unflagged samples: fp32 within the lane (lof_row_flag), fp64 across lanes
    double rs = (double)lane_sum;
    rs = lof_warp_sum(rs);
    uint32_t nf = __popc(fb);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nf += __shfl_down_sync(0xffffffffu, nf, o);
    if (lane == 0) {
      rowsum[(size_t)s * C + c] = rs;
      rowcnt[(size_t)s * C + c] = T - nf;
      n_flag_acc += nf;
    }
  }
  // statistics pass of the next stream: warps that run out of rows above take the prefetched rows in the
  // order they were asked for and wait on the row's barrier; the slower warps find little left to do
  if (Cfg::OVL && next_stream) {
#pragma unroll 1
    for (;;) {
      int c = 0;
      if (lane == 0) c = (int)atomicAdd(&sm.ctl[CT_SROW], 1u);
      c = __shfl_sync(0xffffffffu, c, 0);
      if (c >= C) break;
      lof_mbar_wait(sm.rowbar + c, bar_parity);
      lof_stat_row<C, L>(sm, c, plan_next, lane);
    }
  }
  if (lane == 0 && n_flag_acc) atomicAdd(&sm.ctl[CT_NFLAG], n_flag_acc);
}


// The kernel: persistent CTAs, one stream at a time.  Steady state per stream: frequency pass, time pass
// (which also brings in the next stream row by row and runs that stream's statistics pass on the rows that
// have landed), then the short serial end of the next stream's statistics (median, thresholds).
template <int C, int L>
__global__ void __launch_bounds__(LofFusedCfg<C, L>::NT, LofFusedCfg<C, L>::MINB)
lof_k_fused(const float* __restrict__ power, uint32_t* __restrict__ flags, lof_stream_stats* __restrict__ stats,
            double* __restrict__ rowsum, uint32_t* __restrict__ rowcnt, LofKParams prm,
            unsigned long long* __restrict__ diag) {
  using Cfg = LofFusedCfg<C, L>;
  constexpr int N = Cfg::N, NT = Cfg::NT, W = Cfg::W;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const LofFusedSmem sm = LofFusedSmem::make<C, L>(smem_raw);
  const int tid = threadIdx.x;
  // position of this thread's sample for the plan (one strided sample per thread)
  const int samp_idx0 = (int)(((long long)tid * N) / NT) + (tid * 7) % (N / NT > 0 ? N / NT : 1);
  const int samp_idx = samp_idx0 < N ? samp_idx0 : N - 1;
  bool ready = false;          // shared memory holds stream s and its statistics are done
  float median = 0.f;
  uint32_t n_bad = 0;
  unsigned bar_parity = 0;     // phase of the row barriers the next prefetch completes
  if (tid < C) lof_mbar_init(sm.rowbar + tid, 32);
  __syncthreads();
  // Streams are handed out dynamically after the first two of a CTA (blockIdx.x and blockIdx.x + gridDim.x): a
  // stream's cost depends on its content (restarts), and with ~42 streams per CTA in a fixed order the kernel waited
  // for the unluckiest CTA.  Tickets come from diag[LOF_DIAG_TICKET]; a stream must be known one stream ahead (its
  // rows are prefetched during the time pass of the one before), so the ticket for the stream AFTER NEXT is drawn at
  // the top of an iteration and read after that iteration's first barrier (two slots by parity).  The host zeroes
  // the counter before every launch.
  // (Measured: + 2 % with one CTA per SM, config 2; - 2.5 % with two CTAs per SM, config 3, whose CTAs then stay in
  // a fixed order: DYN.)
  constexpr bool DYN = Cfg::MINB == 1;
  uint32_t s_nx = blockIdx.x + gridDim.x, it = 0;
#pragma unroll 1
  for (uint32_t s = blockIdx.x; s < prm.S; ++it) {
    LOF_PROF_T(t0);
    // (drawn here, put into shared memory only before the barrier that publishes it: the atomic's round trip to L2
    // hides behind the frequency pass instead of holding warp 0 at the top of the iteration)
    uint32_t ticket = 0;
    if (DYN && tid == 0) ticket = 2u * gridDim.x + (uint32_t)atomicAdd(&diag[LOF_DIAG_TICKET], 1ull);
    if (!ready) {                                         // first stream of this CTA (or after a skipped one)
      const float* gs = power + (size_t)s * N;
      const float4* g4 = reinterpret_cast<const float4*>(gs);
      float4* s4 = reinterpret_cast<float4*>(sm.xs);
      for (int i = tid; i < N / 4; i += NT) lof_cp_async16(s4 + lof_swz_chunk(i), g4 + i);
      const float sample = __ldg(gs + samp_idx);
      for (int b = tid; b < LOF_F_NBINS; b += NT) sm.hist[b] = 0;
      lof_cp_async_wait_all();
      __syncthreads();
      n_bad = lof_stat_whole<C, L>(sm, prm, sample, stats + s, median, diag);
    }
    ready = false;
    if (n_bad) {
      // DESIGN.md S6: the whole stream is flagged
      for (int i = tid; i < C * W; i += NT) flags[(size_t)s * C * W + i] = 0xFFFFFFFFu;
      for (int i = tid; i < C; i += NT) { rowsum[(size_t)s * C + i] = 0.0; rowcnt[(size_t)s * C + i] = 0; }
      if (tid == 0) { atomicAdd(&diag[3], 1ull); sm.ctl[CT_TICKET + (it & 1u)] = ticket; }
      __syncthreads();
      { const uint32_t nx2 = DYN ? sm.ctl[CT_TICKET + (it & 1u)] : s_nx + gridDim.x; s = s_nx; s_nx = nx2; }
      continue;
    }
    const uint32_t s_next = s_nx;
    const bool more = s_next < prm.S;
    const float* next = more ? power + (size_t)s_next * N : nullptr;
    // issued here, consumed after the frequency pass: no select on the loaded value, or the wait moves up here
    const float sample_next = __ldg((more ? next : power + (size_t)s * N) + samp_idx);
    const bool have_f = prm.n_lev_f > 0;
    LOF_PROF_T(t1);
    if (have_f) {
      if constexpr (C == 64) lof_fused_freq_pair<C, L>(sm, prm.n_lev_f);
      else lof_fused_freq<C, L>(sm, prm.n_lev_f);
    }
    if (tid == 0) sm.ctl[CT_TICKET + (it & 1u)] = ticket;
    __syncthreads();
    const uint32_t s_nx2 = DYN ? sm.ctl[CT_TICKET + (it & 1u)] : s_nx + gridDim.x;
    LOF_PROF_T(t2);
    LofStatPlan plan_next;
    if (Cfg::OVL) plan_next = lof_stat_plan<NT>(sample_next, reinterpret_cast<float*>(sm.red));
    LOF_PROF_T(t3);
    lof_fused_time<C, L>(sm, prm, s, flags, rowsum, rowcnt, power + (size_t)s * N, next, plan_next, bar_parity);
    if (more) bar_parity ^= 1u;
    lof_cp_async_wait_all();
    __syncthreads();
    LOF_PROF_T(t4);
    // the stream's flag count: stored by the thread that resets the counter for the next stream (no barrier of its own)
    if (more) {
      if (Cfg::OVL) n_bad = lof_stat_finalize<C, L>(sm, prm, plan_next, stats + s_next, median, diag, &stats[s].n_flagged);
      else n_bad = lof_stat_whole<C, L>(sm, prm, sample_next, stats + s_next, median, diag, &stats[s].n_flagged);
      ready = true;
    } else if (tid == 0) stats[s].n_flagged = sm.ctl[CT_NFLAG];
    LOF_PROF_T(t5);
    LOF_PROF_ADD(0, t0, t1); LOF_PROF_ADD(1, t1, t2); LOF_PROF_ADD(2, t2, t3); LOF_PROF_ADD(3, t3, t4);
    LOF_PROF_ADD(4, t4, t5);
    s = s_nx; s_nx = s_nx2;
  }
  lof_cp_async_wait_all();
}
