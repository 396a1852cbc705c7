// lof_flag_generic.cuh — generic SumThreshold kernels (any C <= 256, any T, any max_window).
// One routine runs the iterations of PAPER.md:37-47 on a set of lines held in shared memory;
// the frequency kernel feeds it 32 time columns of a stream (lines along channels), the time
// kernel one row tile with a halo as wide as the dependency cone (lines along time).
// Shape-specialised fused kernels (lof_fused.cuh) replace these where the shape allows; the
// results are the same and tests compare both with the oracle.
#pragma once
#include "lof_common.cuh"

#define LOF_GEN_THREADS 256
#define LOF_GEN_BYTES_PER_ELEM 17   // xs 4 + a 2x4 + cn 2x2 + fl 1

// Shared-memory carve-up for M elements (M a multiple of 32).
struct LofLineSmem {
  float* xs; float* a[2]; uint16_t* cn[2]; uint8_t* fl;
  __device__ LofLineSmem(unsigned char* base, uint32_t M) {
    xs = reinterpret_cast<float*>(base);
    a[0] = xs + M; a[1] = a[0] + M;
    cn[0] = reinterpret_cast<uint16_t*>(a[1] + M); cn[1] = cn[0] + M;
    fl = reinterpret_cast<uint8_t*>(cn[1] + M);
  }
};

// SumThreshold iterations on NLINE interleaved lines of n samples each (element (i, line) at
// index i*NLINE + line).  Window I = 2^k is flagged when the sum of its unflagged samples
// exceeds (I - #flagged) * threshold_I — the paper's test "window sum with flagged samples
// replaced by threshold_I > I * threshold_I" (F4, F7) — with flags frozen at the
// start of each iteration (F8).  Window sums come from a doubling tree in fp32 (error
// <= log2(I) ulp), rebuilt from level 0 whenever the previous iteration set a flag.
template <int NLINE>
__device__ void lof_line_levels(const LofLineSmem& sm, uint32_t n, uint32_t n_lev, const float* thr) {
  const uint32_t M = n * NLINE;
  const int tid = threadIdx.x;
  int cur = 0;
  int dirty = 1;
  for (uint32_t k = 0; k < n_lev; ++k) {
    const uint32_t I = 1u << k;
    if (I > n) break;
    uint32_t j0 = k;
    if (dirty) {
      for (uint32_t e = tid; e < M; e += LOF_GEN_THREADS) {
        const uint8_t f = sm.fl[e];
        sm.a[0][e] = f ? 0.f : sm.xs[e];
        sm.cn[0][e] = f;
      }
      cur = 0; j0 = 1;
      __syncthreads();
    }
    for (uint32_t j = j0; j <= k; ++j) {               // level j-1 -> level j
      const uint32_t d = (1u << (j - 1)) * NLINE, lim = (n - (1u << j) + 1) * NLINE;
      const float* as = sm.a[cur]; float* ad = sm.a[cur ^ 1];
      const uint16_t* cs = sm.cn[cur]; uint16_t* cd = sm.cn[cur ^ 1];
      for (uint32_t e = tid; e < lim; e += LOF_GEN_THREADS) {
        ad[e] = as[e] + as[e + d];
        cd[e] = (uint16_t)(cs[e] + cs[e + d]);
      }
      cur ^= 1;
      __syncthreads();
    }
    const float T = thr[k];
    const uint32_t lim = (n - I + 1) * NLINE;
    int trig = 0;
    for (uint32_t e = tid; e < lim; e += LOF_GEN_THREADS) {
      const float room = (float)(I - sm.cn[cur][e]) * T;
      if (sm.a[cur][e] > room) {
        trig = 1;
        for (uint32_t j = 0; j < I; ++j) sm.fl[e + j * NLINE] = 1;
      }
    }
    dirty = __syncthreads_or(trig);
  }
}

// Frequency direction ("We first flag in the frequency direction").
// grid.x = group_streams * ceil(T/32); CTA = 32 time columns x all C channels.
template <class In>
__global__ void __launch_bounds__(LOF_GEN_THREADS)
lof_k_freq_generic(In in, LofKParams prm, const LofStreamState* __restrict__ state,
                   uint32_t* __restrict__ fmask) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t W = prm.W, C = prm.C, T = prm.T;
  const uint32_t sl = blockIdx.x / W, tb = blockIdx.x - sl * W, s = prm.s0 + sl;
  const uint32_t M = C * 32;
  LofLineSmem sm(smem_raw, M);
  const LofStreamState& st = state[s];
  const uint64_t base = (uint64_t)s * C * T;
  const uint32_t t = tb * 32 + (threadIdx.x & 31);
  for (uint32_t e = threadIdx.x; e < M; e += LOF_GEN_THREADS) {
    const uint32_t c = e >> 5;
    sm.xs[e] = t < T ? in.ld(base + (uint64_t)c * T + t) : 0.f;
    sm.fl[e] = 0;
  }
  __syncthreads();
  lof_line_levels<32>(sm, C, prm.n_lev_f, st.thr_f);
  const uint32_t valid = (T - tb * 32 >= 32) ? 0xFFFFFFFFu : ((1u << (T - tb * 32)) - 1u);
  for (uint32_t e = threadIdx.x; e < M; e += LOF_GEN_THREADS) {
    const uint32_t word = __ballot_sync(0xffffffffu, sm.fl[e] != 0) & valid;
    if ((threadIdx.x & 31) == 0) fmask[((uint64_t)s * C + (e >> 5)) * W + tb] = word;
  }
}

// Time direction, starting from the frequency run's mask (F10), plus the bit-pack and
// the per-row sums of unflagged samples.  grid.x = group_rows * n_tiles.  A tile
// covers [t0 - halo, t0 + TT + halo) of one row and writes the words of [t0, t0 + TT).
// part_sum/part_cnt: [rows][n_tiles].
template <class In>
__global__ void __launch_bounds__(LOF_GEN_THREADS)
lof_k_time_generic(In in, LofKParams prm, const LofStreamState* __restrict__ state,
                   const uint32_t* __restrict__ fmask, uint32_t* __restrict__ flags,
                   double* __restrict__ part_sum, uint32_t* __restrict__ part_cnt,
                   lof_stream_stats* __restrict__ stats, uint32_t TT, uint32_t halo, uint32_t n_tiles) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double sh_red[32];
  __shared__ uint32_t sh_cnt[2];
  const uint32_t W = prm.W, C = prm.C, T = prm.T;
  const uint32_t rl = blockIdx.x / n_tiles, tile = blockIdx.x - rl * n_tiles;
  const uint64_t row = (uint64_t)prm.s0 * C + rl;
  const uint32_t s = (uint32_t)(row / C);
  const uint32_t t0 = tile * TT;
  const uint32_t t_lo = t0 >= halo ? t0 - halo : 0;
  const uint32_t t_hi = min(T, t0 + TT + halo);
  const uint32_t n = t_hi - t_lo;
  const uint32_t Mpad = (n + 31) & ~31u;
  LofLineSmem sm(smem_raw, (TT + 2 * halo + 31) & ~31u);
  const LofStreamState& st = state[s];
  const bool bad = st.nonfinite != 0;
  const uint64_t base = row * T;
  const uint32_t* fm = fmask + row * W;
  const bool have_f = prm.n_lev_f > 0;
  for (uint32_t e = threadIdx.x; e < Mpad; e += LOF_GEN_THREADS) {
    const uint32_t t = t_lo + e;
    float x = 0.f; uint8_t f = 0;
    if (t < t_hi) {
      x = in.ld(base + t);
      if (have_f) f = (fm[t >> 5] >> (t & 31)) & 1u;
      if (bad) f = 1;                                   // DESIGN.md S6: the whole stream is flagged
    }
    sm.xs[e] = x; sm.fl[e] = f;
  }
  if (threadIdx.x == 0) { sh_cnt[0] = 0; sh_cnt[1] = 0; }
  __syncthreads();
  if (!bad) lof_line_levels<1>(sm, n, prm.n_lev_t, st.thr_f);
  // bit-pack the central words, sum the unflagged samples (fp64, fixed order)
  const uint32_t c_lo = t0 - t_lo;                      // multiple of 32
  const uint32_t c_hi = min(T, t0 + TT) - t_lo;
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double acc = 0.0; uint32_t n_un = 0, n_fl = 0;
  for (uint32_t w0 = c_lo + warp * 32; w0 < c_hi; w0 += (LOF_GEN_THREADS / 32) * 32) {
    const uint32_t e = w0 + lane;
    const bool in_row = e < c_hi;
    const bool f = in_row && sm.fl[e] != 0;
    const uint32_t word = __ballot_sync(0xffffffffu, f);
    if (lane == 0) flags[row * W + ((t_lo + w0) >> 5)] = word;
    if (in_row && !f) { acc += (double)sm.xs[e]; ++n_un; }
    n_fl += f ? 1u : 0u;
  }
  const double tot = lof_block_sum(acc, sh_red);
  atomicAdd(&sh_cnt[0], n_un);
  atomicAdd(&sh_cnt[1], n_fl);
  __syncthreads();
  if (threadIdx.x == 0) {
    part_sum[(uint64_t)rl * n_tiles + tile] = tot;
    part_cnt[(uint64_t)rl * n_tiles + tile] = sh_cnt[0];
    if (sh_cnt[1]) atomicAdd(reinterpret_cast<unsigned long long*>(&stats[s].n_flagged),
                             (unsigned long long)sh_cnt[1]);
  }
}

// Row sums: tile partials added in tile order (deterministic).  One thread per row of the group.
__global__ void lof_k_rowsum_final(const double* __restrict__ part_sum, const uint32_t* __restrict__ part_cnt,
                                   double* __restrict__ rowsum, uint32_t* __restrict__ rowcnt,
                                   uint64_t row0, uint32_t n_rows, uint32_t n_tiles) {
  const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n_rows) return;
  double a = 0.0; uint32_t c = 0;
  for (uint32_t j = 0; j < n_tiles; ++j) { a += part_sum[(uint64_t)r * n_tiles + j]; c += part_cnt[(uint64_t)r * n_tiles + j]; }
  rowsum[row0 + r] = a; rowcnt[row0 + r] = c;
}
