// lof_longrow.cuh — register-resident SumThreshold kernels for streams too long for one SM's shared
// memory (BASELINE.json configs 4 and 5: rows of 195 312 and 12 208 samples).  Same column / row cores as
// the fused kernel (lof_col_flag, lof_row_flag in lof_fused.cuh), fed from global memory after the
// statistics passes of lof_stats_lr.cuh (one group of streams per launch sequence).
//   lof_k_freq_reg<C> / lof_k_freq_stg<C>: a warp per group of 32 time columns, a thread per column;
//                      the second one persistent with the next unit staged by LDGSTS (32 and 64 channels).
//   lof_k_time_seg   : a warp per row segment of 1024 samples = OUT output samples + a halo of H on
//                      each side, H >= the dependency cone sum_k (2^k - 1) of the time run, so segments
//                      are independent; lane l holds samples [32 l, 32 l + 32).
#pragma once
#include "lof_common.cuh"
#include "lof_core.cuh"

#define LOF_LR_THREADS 256
#define LOF_LR_WARPS (LOF_LR_THREADS / 32)
#define LOF_LR_TILE 1024
#define LOF_SEG_SMEM (2 * LOF_LR_WARPS * LOF_LR_TILE * 4)

// One launch of a warp per unit, loads straight into registers: the form kept for 16 channels, which is bound by
// instruction issue (70 % of the issue slots) and measured 8 % slower in the staged form below.
template <int C, class In>
__global__ void __launch_bounds__(LOF_LR_THREADS, (C <= 32 ? 2 : 1))
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
      [&](int c) { return valid ? in.ld(base + (uint64_t)c * T) : -INFINITY; }, thr, state[s].dead_f, (int)prm.n_lev_f);
  uint32_t mine0, mine1;
  lof_col_words<C>(fb, lane, mine0, mine1);
  if (lane < C) fmask[((uint64_t)s * C + lane) * W + w] = mine0;
  if (C > 32 && lane + 32 < C) fmask[((uint64_t)s * C + lane + 32) * W + w] = mine1;
}

// 16-byte asynchronous global -> shared copy (LDGSTS), and "all of this thread's copy groups but the newest n"
__device__ __forceinline__ void lof_lr_cp16(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void lof_lr_cp4(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void lof_lr_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void lof_lr_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Persistent: a warp walks over units (stream, group of 32 columns).  With 16-byte aligned rows (T % 4 == 0) the
// C x 32 samples of the NEXT unit are on their way into the warp's second staging strip (LDGSTS, C x 128 bytes,
// raw 4-byte samples) while the current columns are processed: one load phase and one compute phase per warp had
// left the SM waiting on memory with 8-16 warps resident (20 % of the warp slots, 4.6 warps per issued
// instruction on the long scoreboard).  Shared memory: LOF_FREQ_SMEM(C) = 2 strips x 8 warps x C x 128 bytes.
#define LOF_FREQ_SMEM(C) (2 * LOF_LR_WARPS * (C) * 128)
template <int C, class In>
__global__ void __launch_bounds__(LOF_LR_THREADS, (C <= 32 ? 2 : 1))
lof_k_freq_stg(In in, LofKParams prm, const LofStreamState* __restrict__ state, uint32_t* __restrict__ fmask,
               uint32_t n_group_streams) {
  extern __shared__ __align__(16) unsigned char fr_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t W = prm.W, T = prm.T;
  const uint64_t n_units = (uint64_t)n_group_streams * W, n_warps = (uint64_t)gridDim.x * LOF_LR_WARPS;
  const bool async = (T & 3) == 0;
  const unsigned char* raw = reinterpret_cast<const unsigned char*>(in.p);
  auto strip = [&](int buf) { return reinterpret_cast<uint32_t*>(fr_raw) + (size_t)(buf * LOF_LR_WARPS + warp) * C * 32; };
  auto issue = [&](uint64_t u, int buf) {
    const uint32_t sl = (uint32_t)(u / W), w = (uint32_t)(u - (uint64_t)sl * W), s = prm.s0 + sl;
    uint32_t* sg = strip(buf);
#pragma unroll
    for (int q = 0; q < C / 4; ++q) {
      const int i = q * 32 + lane, c = i >> 3, ch = i & 7;
      const uint32_t t = w * 32 + ch * 4;
      if (t < T) lof_lr_cp16(sg + c * 32 + ch * 4, raw + (((uint64_t)s * C + c) * T + t) * 4);
    }
    lof_lr_commit();
  };
  uint64_t unit = (uint64_t)blockIdx.x * LOF_LR_WARPS + warp;
  int buf = 0;
  if (async && unit < n_units) issue(unit, 0);
#pragma unroll 1
  for (; unit < n_units; unit += n_warps, buf ^= 1) {
    const uint32_t sl = (uint32_t)(unit / W), w = (uint32_t)(unit - (uint64_t)sl * W), s = prm.s0 + sl;
    const uint32_t t = w * 32 + lane;
    const bool valid = t < T;
    const uint64_t base = (uint64_t)s * C * T + (valid ? t : 0);
    const uint32_t* sg = strip(buf);
    if (async) {
      if (unit + n_warps < n_units) { issue(unit + n_warps, buf ^ 1); lof_lr_wait<1>(); }
      else lof_lr_wait<0>();
      __syncwarp();
    }
    const float* thr = state[s].thr_f;
    // a column beyond the row's end holds -inf: it never exceeds a threshold and any window sum with it is -inf
    const uint64_t fb = lof_col_flag<C>(
        [&](int c) {
          if (!valid) return -INFINITY;
          return async ? In::from_raw(sg[c * 32 + lane], true) : in.ld(base + (uint64_t)c * T);
        },
        thr, state[s].dead_f, (int)prm.n_lev_f);
    uint32_t mine0, mine1;
    lof_col_words<C>(fb, lane, mine0, mine1);
    if (lane < C) fmask[((uint64_t)s * C + lane) * W + w] = mine0;
    if (C > 32 && lane + 32 < C) fmask[((uint64_t)s * C + lane + 32) * W + w] = mine1;
    __syncwarp();                                         // the strip is free for the copy after next
  }
}

// element i of a warp's 1024-sample staging tile: float4 chunk g = i/4 stored at g ^ ((g/8) & 7), so the
// coalesced fill (lanes = consecutive i) and the per-lane reads of 32 consecutive floats are conflict-free
__device__ __forceinline__ int lof_lr_swz(int i) {
  const int g = i >> 2;
  return ((g ^ ((g >> 3) & 7)) << 2) | (i & 3);
}

// sum of the samples of a lane's word that are not in `skip` (the lane's share of PAPER.md:102's row mean)
__device__ __forceinline__ float lof_sum_unflagged(const float2 (&x2)[16], uint32_t skip) {
  float p0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f;
#pragma unroll
  for (int m = 0; m < 16; m += 2) {
    p0 += ((skip >> (2 * m)) & 1u) ? 0.f : x2[m].x;
    p1 += ((skip >> (2 * m + 1)) & 1u) ? 0.f : x2[m].y;
    p2 += ((skip >> (2 * m + 2)) & 1u) ? 0.f : x2[m + 1].x;
    p3 += ((skip >> (2 * m + 3)) & 1u) ? 0.f : x2[m + 1].y;
  }
  return (p0 + p1) + (p2 + p3);
}

// Persistent: a warp walks over units (row segments) gw, gw + #warps, ...  When the rows are 16-byte aligned
// (T % 4 == 0) the strip of the NEXT unit is on its way into the warp's second staging strip (LDGSTS, raw 4-byte
// samples: float32, or complex int16 turned into power when the registers are filled) while the current one is
// processed: the kernel had been stalled on its own loads (3.1 warps per issued instruction waiting on global
// memory, 16 warps per SM).  Otherwise the strip is filled synchronously as before.
template <class In>
__global__ void __launch_bounds__(LOF_LR_THREADS, 2)
lof_k_time_seg(In in, LofKParams prm, const LofStreamState* __restrict__ state, const uint32_t* __restrict__ fmask,
               uint32_t* __restrict__ flags, double* __restrict__ part_sum, uint32_t* __restrict__ part_cnt,
               lof_stream_stats* __restrict__ stats, uint32_t OUT, uint32_t H, uint32_t n_seg, uint32_t n_rows) {
  extern __shared__ __align__(16) unsigned char seg_raw[];          // LOF_SEG_SMEM bytes: [2][warps][tile] words
  uint32_t (*stage)[LOF_LR_WARPS][LOF_LR_TILE] = reinterpret_cast<uint32_t (*)[LOF_LR_WARPS][LOF_LR_TILE]>(seg_raw);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t W = prm.W, C = prm.C, T = prm.T;
  const uint64_t n_units = (uint64_t)n_rows * n_seg, n_warps = (uint64_t)gridDim.x * LOF_LR_WARPS;
  const bool async = (T & 3) == 0;
  const unsigned char* raw = reinterpret_cast<const unsigned char*>(in.p);
  // strip of unit u -> staging strip `buf` (chunks beyond the row's end are left alone: masked when read)
  auto issue = [&](uint64_t u, int buf) {
    const uint32_t rl = (uint32_t)(u / n_seg), seg = (uint32_t)(u - (uint64_t)rl * n_seg);
    const uint64_t row = (uint64_t)prm.s0 * C + rl;
    const uint32_t o_lo = seg * OUT, t_lo = o_lo >= H ? o_lo - H : 0;
    uint4* sg4 = reinterpret_cast<uint4*>(stage[buf][warp]);
#pragma unroll
    for (int q = 0; q < LOF_LR_TILE / 128; ++q) {
      const int g = q * 32 + lane;
      const uint32_t t = t_lo + 4 * g;
      if (t < T) lof_lr_cp16(sg4 + (g ^ ((g >> 3) & 7)), raw + (row * T + t) * 4);
    }
    lof_lr_commit();
  };
  uint64_t unit = (uint64_t)blockIdx.x * LOF_LR_WARPS + warp;
  int buf = 0;
  if (async && unit < n_units) issue(unit, 0);
#pragma unroll 1
  for (; unit < n_units; unit += n_warps, buf ^= 1) {
    const uint32_t rl = (uint32_t)(unit / n_seg), seg = (uint32_t)(unit - (uint64_t)rl * n_seg);
    const uint64_t row = (uint64_t)prm.s0 * C + rl;
    const uint32_t s = (uint32_t)(row / C);
    const LofStreamState& st = state[s];
    const uint32_t o_lo = seg * OUT, o_hi = min(T, o_lo + OUT);
    const uint32_t t_lo = o_lo >= H ? o_lo - H : 0;        // multiple of 32
    uint32_t* sg = stage[buf][warp];
    const uint64_t base = row * T;
    if (async) {
      if (unit + n_warps < n_units) { issue(unit + n_warps, buf ^ 1); lof_lr_wait<1>(); }
      else lof_lr_wait<0>();
    } else {
#pragma unroll 4
      for (int q = 0; q < LOF_LR_TILE / 32; ++q) {
        const int i = q * 32 + lane;
        const uint32_t t = t_lo + i;
        sg[lof_lr_swz(i)] = t < T ? In::raw_of(in.ld(base + t)) : 0u;
      }
    }
    __syncwarp();
    const uint32_t t_w = t_lo + 32 * lane;                  // first sample of this lane's word
    const uint32_t valid = t_w >= T ? 0u : (T - t_w >= 32 ? 0xFFFFFFFFu : ((1u << (T - t_w)) - 1u));
    // the lane's 32 samples from the staging strip (again on a restart: the strip keeps the raw samples);
    // beyond the row's end: -inf, which never exceeds a threshold and kills every window it is part of
    auto load = [&](float2 (&x2)[16], bool) {
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        const uint4 v = reinterpret_cast<const uint4*>(sg)[(8 * lane + q) ^ (lane & 7)];
        x2[2 * q] = make_float2(In::from_raw(v.x, async), In::from_raw(v.y, async));
        x2[2 * q + 1] = make_float2(In::from_raw(v.z, async), In::from_raw(v.w, async));
      }
      if (valid != 0xFFFFFFFFu) {
#pragma unroll
        for (int m = 0; m < 16; ++m) {
          if (!((valid >> (2 * m)) & 1u)) x2[m].x = -INFINITY;
          if (!((valid >> (2 * m + 1)) & 1u)) x2[m].y = -INFINITY;
        }
      }
    };
    // start from the frequency run's mask (F10): its flagged samples enter the row core as LOF_MARK
    uint32_t fb = 0;
    if (prm.n_lev_f > 0 && valid) fb = fmask[row * W + (t_w >> 5)];
    float lane_sum = 0.f;
    bool have_sum = false;
    if (st.nonfinite) fb = valid;                           // DESIGN.md S6: the whole stream is flagged
    else if (prm.n_lev_t > 0) {
      lof_row_flag<32, 7>(load, fb, st.thr_f, st.dead_t, (int)prm.n_lev_t, lane, lane_sum);
      have_sum = true;
    }
    fb &= valid;
    const bool mine = t_w >= o_lo && t_w < o_hi;            // this lane's word belongs to the segment's output
    if (mine) flags[row * W + (t_w >> 5)] = fb;
    if (!have_sum || valid != 0xFFFFFFFFu) {
      float2 x2[16];
      load(x2, true);
      lane_sum = lof_sum_unflagged(x2, fb | ~valid);
    }
    double rs = mine ? (double)lane_sum : 0.0;
    rs = lof_warp_sum(rs);
    const uint32_t nf = __reduce_add_sync(0xffffffffu, mine ? (uint32_t)__popc(fb) : 0u);
    const uint32_t nu = __reduce_add_sync(0xffffffffu, mine ? (uint32_t)__popc(valid & ~fb) : 0u);
    if (lane == 0) {
      part_sum[(uint64_t)rl * n_seg + seg] = rs;
      part_cnt[(uint64_t)rl * n_seg + seg] = nu;
      if (nf) atomicAdd(reinterpret_cast<unsigned long long*>(&stats[s].n_flagged), (unsigned long long)nf);
    }
    __syncwarp();                                           // the strip is free for the prefetch after next
  }
}

// ---- CTA-cooperative time run for wide cones (max_window >= 256): 8 warps share a tile of 8192 samples
// (halo H on each side), each warp holding 1024 of them as in lof_k_time_seg.  Per iteration the warps
// exchange only what crosses their borders, through shared memory: the first D window sums / counts of the
// next warp (partners of the last lanes), and the last fired window start of the previous warps (dilation).
#define LOF_CO_WARPS 8
#define LOF_CO_TILE (LOF_CO_WARPS * LOF_LR_TILE)

struct LofCoopSmem {
  uint32_t stage[2][LOF_CO_WARPS][LOF_LR_TILE];         // load staging (raw 4-byte samples), one 1024-sample strip per
                                                        // warp, double-buffered over the CTA's tiles
  float bu[LOF_CO_WARPS][512];                          // published window sums: the first D of step D at [D, 2D), so
  float be[LOF_CO_WARPS][512];                          // every step keeps its own (a strip that sits out a restart
                                                        // does not publish again); be: the counts
  int wmax[LOF_CO_WARPS];                               // last fired window start per warp
  int chg[LOF_CO_WARPS];                                // strip got new flags in the last test
  uint32_t fm[2][LOF_CO_WARPS][32];                     // the strips' frequency-run mask words, copied with them
};

// One doubling step of distance D on a strip of 1024 samples (lane l: 32 samples as 16 pairs); partners beyond
// the strip come from the next warp's published sums nb_u / nb_e (its first D positions), or do not exist.
template <int D>
__device__ __forceinline__ void lof_row_step_coop(float2 (&u2)[16], float2 (&e2)[16], int lane, const float* nb_u,
                                                  const float* nb_e, bool has_nb) {
  if constexpr (D == 1) {
    float pu = __shfl_down_sync(0xffffffffu, u2[0].x, 1);
    float pe = __shfl_down_sync(0xffffffffu, e2[0].x, 1);
    if (lane == 31) { pu = has_nb ? nb_u[0] : -INFINITY; pe = has_nb ? nb_e[0] : 0.f; }
#pragma unroll
    for (int m = 0; m < 16; ++m) {
      u2[m].x += u2[m].y; e2[m].x += e2[m].y;
      u2[m].y += (m + 1 < 16) ? u2[m + 1].x : pu; e2[m].y += (m + 1 < 16) ? e2[m + 1].x : pe;
    }
  } else {
    constexpr int H = D / 2;                              // distance in pairs
    constexpr int NQ = H < 16 ? H : 16;
    // one tree at a time (the partners fetched from other lanes are live for one of them only)
    auto one = [&](float2 (&a2)[16], const float* nb, float none) {
      float2 pa[NQ];
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        const int m = 16 - NQ + q, src = (m + H) % 16, off = (m + H) / 16;
        pa[q].x = __shfl_down_sync(0xffffffffu, a2[src].x, off); pa[q].y = __shfl_down_sync(0xffffffffu, a2[src].y, off);
        if (lane + off > 31) {                            // the partner lives in the next warp's strip
          const int p = (lane + off - 32) * 32 + 2 * src; // its position there, < D (even)
          pa[q] = has_nb ? *reinterpret_cast<const float2*>(nb + p) : make_float2(none, none);
        }
      }
#pragma unroll
      for (int m = 0; m < 16; ++m) a2[m] = __fadd2_rn(a2[m], (m + H < 16) ? a2[m + H] : pa[m - (16 - NQ)]);
    };
    one(u2, nb_u, -INFINITY);
    one(e2, nb_e, 0.f);
  }
}

// Test of iteration I = 2^K on a strip; like lof_row_eval, but windows fired in previous warps' strips dilate
// into this one (carry through wmax[]), and "any" is taken over the CTA.  Contains __syncthreads: CTA-uniform.
template <int K>
__device__ __forceinline__ bool lof_row_eval_coop(const float2 (&u2)[16], const float2 (&e2)[16], int lane, int warp,
                                                  float thr, float tdead, uint32_t& fb, int* wmax, int* chg,
                                                  bool& dead) {
  constexpr int I = 1 << K;
  const float2 negT = make_float2(-thr, -thr), negD = make_float2(-tdead, -tdead);
  float tm[2] = {-INFINITY, -INFINITY}, td[2] = {-INFINITY, -INFINITY};
#pragma unroll
  for (int m = 0; m < 16; ++m) {
    const float2 v = __ffma2_rn(e2[m], negT, u2[m]), w = __ffma2_rn(e2[m], negD, u2[m]);
    tm[m & 1] = lof_max3(tm[m & 1], v.x, v.y);
    td[m & 1] = lof_max3(td[m & 1], w.x, w.y);
  }
  // one barrier decides the usual case (nothing fired, and no window of I samples has an unflagged mean above
  // tdead: the tile is done, lof_dead_level); a second one tells the two apart otherwise
  const bool fired = fmaxf(tm[0], tm[1]) > 0.f, alive = fmaxf(td[0], td[1]) > 0.f;
  dead = false;
  if (!__syncthreads_or(fired || alive)) { dead = true; return false; }
  if (!__syncthreads_or(fired)) return false;
  uint32_t tg[4] = {0u, 0u, 0u, 0u};                       // partial masks: no serial chain
#pragma unroll
  for (int m = 0; m < 16; ++m) {
    tg[m & 1] |= (fmaf(e2[m].x, -thr, u2[m].x) > 0.f) ? (1u << (2 * m)) : 0u;
    tg[2 + (m & 1)] |= (fmaf(e2[m].y, -thr, u2[m].y) > 0.f) ? (2u << (2 * m)) : 0u;
  }
  const uint32_t trig = (tg[0] | tg[1]) | (tg[2] | tg[3]);
  uint32_t own = trig;
#pragma unroll
  for (int s = 1; s < I && s < 32; s <<= 1) own |= own << s;
  const int pos0 = warp * LOF_LR_TILE + lane * 32;        // tile coordinate of this lane's first sample
  int pm = trig ? (pos0 + 31 - __clz(trig)) : -(1 << 20);
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, pm, o); if (lane >= o) pm = max(pm, v); }
  if (lane == 31) wmax[warp] = pm;
  __syncthreads();
  int prev = __shfl_up_sync(0xffffffffu, pm, 1);
  if (lane == 0) prev = -(1 << 20);
  for (int w = 0; w < warp; ++w) prev = max(prev, wmax[w]);
  int cnt = prev + I - pos0;
  cnt = cnt < 0 ? 0 : (cnt > 32 ? 32 : cnt);
  const uint32_t pre = cnt >= 32 ? 0xFFFFFFFFu : ((1u << cnt) - 1u);
  const uint32_t nf = fb | own | pre;
  const bool changed = nf != fb;
  fb = nf;
  const bool wch = __any_sync(0xffffffffu, changed);
  if (lane == 0) chg[warp] = wch;
  return __syncthreads_or(changed) != 0;
}

// grid.x = n_rows * n_tile; a CTA of 8 warps covers [t_lo, t_lo + 8192) of one row and writes the words of
// its OUT = 8192 - 2H central samples.  All control flow around barriers is CTA-uniform.
template <class In>
__global__ void __launch_bounds__(LOF_CO_WARPS * 32, 2)
lof_k_time_coop(In in, LofKParams prm, const LofStreamState* __restrict__ state, const uint32_t* __restrict__ fmask,
                uint32_t* __restrict__ flags, double* __restrict__ part_sum, uint32_t* __restrict__ part_cnt,
                lof_stream_stats* __restrict__ stats, uint32_t OUT, uint32_t H, uint32_t n_tile, uint32_t n_units) {
  extern __shared__ __align__(16) unsigned char co_raw[];
  LofCoopSmem& sm = *reinterpret_cast<LofCoopSmem*>(co_raw);
  __shared__ double red_sum[LOF_CO_WARPS];
  __shared__ uint32_t red_cnt[2][LOF_CO_WARPS];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t W = prm.W, C = prm.C, T = prm.T;
  const bool async = (T & 3) == 0;
  const unsigned char* raw = reinterpret_cast<const unsigned char*>(in.p);
  // persistent over tiles: the strips of the NEXT tile are on their way (LDGSTS) while this one is processed — the
  // kernel had 5 warps per issued instruction waiting on its own global loads
  auto issue = [&](uint32_t u, int buf) {
    const uint32_t rl = u / n_tile, tile = u - rl * n_tile;
    const uint64_t row = (uint64_t)prm.s0 * C + rl;
    const uint32_t o_lo = tile * OUT;
    const uint32_t t_lo = (o_lo >= H ? o_lo - H : 0) + warp * LOF_LR_TILE;
    uint4* sg4 = reinterpret_cast<uint4*>(sm.stage[buf][warp]);
#pragma unroll
    for (int q = 0; q < LOF_LR_TILE / 128; ++q) {
      const int g = q * 32 + lane;
      const uint32_t t = t_lo + 4 * g;
      if (t < T) lof_lr_cp16(sg4 + (g ^ ((g >> 3) & 7)), raw + (row * T + t) * 4);
    }
    if (prm.n_lev_f > 0 && t_lo + 32 * lane < T) lof_lr_cp4(&sm.fm[buf][warp][lane], fmask + row * W + (t_lo >> 5) + lane);
    lof_lr_commit();
  };
  int buf = 0;
  if (async && blockIdx.x < n_units) issue(blockIdx.x, 0);
#pragma unroll 1
  for (uint32_t unit = blockIdx.x; unit < n_units; unit += gridDim.x, buf ^= 1) {
  const uint32_t rl = unit / n_tile, tile = unit - rl * n_tile;
  const uint64_t row = (uint64_t)prm.s0 * C + rl;
  const uint32_t s = (uint32_t)(row / C);
  const LofStreamState& st = state[s];
  const uint32_t o_lo = tile * OUT, o_hi = min(T, o_lo + OUT);
  const uint32_t t_lo = (o_lo >= H ? o_lo - H : 0) + warp * LOF_LR_TILE;   // this warp's strip
  uint32_t* sg = sm.stage[buf][warp];
  const uint64_t base = row * T;
  if (async) {
    if (unit + gridDim.x < n_units) { issue(unit + gridDim.x, buf ^ 1); lof_lr_wait<1>(); }
    else lof_lr_wait<0>();
  } else {
#pragma unroll 4
    for (int q = 0; q < LOF_LR_TILE / 32; ++q) {
      const int i = q * 32 + lane;
      const uint32_t t = t_lo + i;
      sg[lof_lr_swz(i)] = t < T ? In::raw_of(in.ld(base + t)) : 0u;
    }
  }
  __syncwarp();
  const uint32_t t_w = t_lo + 32 * lane;
  const uint32_t valid = t_w >= T ? 0u : (T - t_w >= 32 ? 0xFFFFFFFFu : ((1u << (T - t_w)) - 1u));
  auto load = [&](float2 (&x2)[16]) {
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const uint4 v = reinterpret_cast<const uint4*>(sg)[(8 * lane + q) ^ (lane & 7)];
      x2[2 * q] = make_float2(In::from_raw(v.x, async), In::from_raw(v.y, async));
      x2[2 * q + 1] = make_float2(In::from_raw(v.z, async), In::from_raw(v.w, async));
    }
    if (valid != 0xFFFFFFFFu) {                           // beyond the row's end: -inf
#pragma unroll
      for (int m = 0; m < 16; ++m) {
        if (!((valid >> (2 * m)) & 1u)) x2[m].x = -INFINITY;
        if (!((valid >> (2 * m + 1)) & 1u)) x2[m].y = -INFINITY;
      }
    }
  };
  uint32_t fb = 0;
  if (prm.n_lev_f > 0 && valid) fb = async ? sm.fm[buf][warp][lane] : fmask[row * W + (t_w >> 5)];   // the frequency run's flags (F10)
  const int nlt = (int)prm.n_lev_t;
  float lane_sum = 0.f;
  bool have_sum = false;
  if (st.nonfinite) fb = valid;
  else if (nlt > 0) {
    const float* thr = st.thr_f;
    const float* dead = st.dead_t;
    const float T0 = thr[0], D0 = dead[0];
    float2 u2[16], e2[16];
    int k_next = 1;
    bool again = true;
    const bool has_nb = warp + 1 < LOF_CO_WARPS;
    have_sum = true;
    // A restart rebuilds the trees only in the strips that can have changed: those with new flags and the one
    // before each (its windows reach up to 511 samples into the next strip).  The other warps keep the trees of
    // the iteration that fired, whose published sums are still in place, and join again at iteration k_next;
    // they pass the same barriers.  (Restarting all 8 warps for every new flag in 8192 samples had been most of
    // this kernel's instructions.)
    bool sit = false;
    float mu = 0.f;
#pragma unroll 1
    while (again) {
      if (!sit) {
        float2 x2[16];
        load(x2);
        if (fb) lof_mark<16>(x2, fb);                     // flags of the frequency run and of earlier restarts
        fb = ~lof_level0<16>(x2, T0, u2, e2, mu);
        lane_sum = lof_lane_sum<16>(u2);
      }
      // no iteration left, or no unflagged sample of the tile above every later threshold (lof_dead_level)
      if (k_next >= nlt || __syncthreads_and(mu <= D0)) break;
      again = false;
      bool dead_ = false;
#define LOF_CO_LEVEL(K)                                                                          \
      if (K < nlt && !again && !dead_) {                                                         \
        constexpr int D = 1 << (K - 1);                                                          \
        const bool act = !sit || K >= k_next;                                                    \
        float* pbu = sm.bu[warp] + D; float* pbe = sm.be[warp] + D;                              \
        /* publish the first D sums / counts of this strip for the previous warp */             \
        if (act && lane * 32 < D) {                                                              \
          _Pragma("unroll") for (int m = 0; m < 16; ++m) if (lane * 32 + 2 * m < D) {            \
            if (D == 1) { pbu[0] = u2[0].x; pbe[0] = e2[0].x; }                                  \
            else { *reinterpret_cast<float2*>(pbu + lane * 32 + 2 * m) = u2[m];                  \
                   *reinterpret_cast<float2*>(pbe + lane * 32 + 2 * m) = e2[m]; }                \
          }                                                                                      \
        }                                                                                        \
        __syncthreads();                                                                         \
        if (act) lof_row_step_coop<D>(u2, e2, lane, sm.bu[has_nb ? warp + 1 : warp] + D,         \
                                      sm.be[has_nb ? warp + 1 : warp] + D, has_nb);              \
        if (K >= k_next && lof_row_eval_coop<K>(u2, e2, lane, warp, thr[K], dead[K], fb, sm.wmax, sm.chg, dead_)) { \
          again = true; k_next = K + 1 < nlt ? K + 1 : 99;                                       \
          sit = !(sm.chg[warp] || (has_nb && sm.chg[warp + 1]));                                 \
        }                                                                                        \
      }
      LOF_CO_LEVEL(1) LOF_CO_LEVEL(2) LOF_CO_LEVEL(3) LOF_CO_LEVEL(4) LOF_CO_LEVEL(5)
      LOF_CO_LEVEL(6) LOF_CO_LEVEL(7) LOF_CO_LEVEL(8) LOF_CO_LEVEL(9)
#undef LOF_CO_LEVEL
      __syncthreads();                                    // a restart republishes into the same buffers
    }
  }
  fb &= valid;
  const bool mine = t_w >= o_lo && t_w < o_hi;
  if (mine) flags[row * W + (t_w >> 5)] = fb;
  if (!have_sum || valid != 0xFFFFFFFFu) {
    float2 x2[16];
    load(x2);
    lane_sum = lof_sum_unflagged(x2, fb | ~valid);
  }
  double rs = mine ? (double)lane_sum : 0.0;
  rs = lof_warp_sum(rs);
  uint32_t nf = mine ? __popc(fb) : 0u, nu = mine ? __popc(valid & ~fb) : 0u;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    nf += __shfl_down_sync(0xffffffffu, nf, o);
    nu += __shfl_down_sync(0xffffffffu, nu, o);
  }
  if (lane == 0) { red_sum[warp] = rs; red_cnt[0][warp] = nu; red_cnt[1][warp] = nf; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0; uint32_t cu = 0, cf = 0;
    for (int w = 0; w < LOF_CO_WARPS; ++w) { a += red_sum[w]; cu += red_cnt[0][w]; cf += red_cnt[1][w]; }
    part_sum[(uint64_t)rl * n_tile + tile] = a;
    part_cnt[(uint64_t)rl * n_tile + tile] = cu;
    if (cf) atomicAdd(reinterpret_cast<unsigned long long*>(&stats[s].n_flagged), (unsigned long long)cf);
  }
  __syncthreads();                                        // the reductions' scratch and the staging strips are free
  }
}
