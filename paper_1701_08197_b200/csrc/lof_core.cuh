// lof_core.cuh — the register-resident SumThreshold cores shared by the fused kernel
// (lof_fused.cuh) and the long-row kernels (lof_longrow.cuh):
//   lof_col_flag<C>   one lane per line of C samples (the frequency run: a time column of 16/32/64 channels)
//   lof_pcol_flag     two lanes per line of 64 samples (the 64-channel column of the fused kernel)
//   lof_row_flag<L>   one warp per line of 32 L samples, lane l holding samples [l L, l L + L) (the time run)
//
// Formulation.  The paper's test "window sum with flagged samples replaced by threshold_I > I * threshold_I"
// (reading F7) is  u > e * threshold_I  with u = sum of the window's unflagged samples and e = their number.
// Both come from doubling trees, X_2I[t] = X_I[t] + X_I[t + I], kept as fp32 PAIRS of neighbouring positions so
// that one packed sm_100 instruction serves two window positions: FADD2 doubles u and e, FFMA2 forms
// u - e*T, FMNMX3 folds both results into a running maximum; only a warp in which some maximum is positive
// builds the bit mask of the fired windows.  e is a small integer, exact in fp32.
//
// Level 0 (I = 1, the simple thresholder of PAPER.md:45) produces, per sample, e = (x <= threshold_1) as 1.0/0.0
// with one FSET, u = x*e, and the lane's mask of unflagged samples as an exact fp32 number (one FFMA2 per pair:
// a Horner chain in base 4), so that the select / bit-insert chains of a mask-first formulation disappear.
// A sample flagged earlier (by the other direction's run, or by a window of this run before a restart) is
// represented IN THE DATA as LOF_MARK = FLT_MAX: it exceeds every threshold, so level 0 flags it again and
// gives it u = e = 0, which is exactly the substitution rule.  Flags are frozen during an iteration (F8): an
// iteration that sets a new flag marks it in the registers and restarts the trees from level 0.
//
// Early exit: lof_dead_level (lof_common.cuh) — after iteration j, no window of 2^j samples with an unflagged
// mean above every later threshold => no later iteration can fire; tested with the same packed instructions.
#pragma once
#include "lof_common.cuh"

#define LOF_MARK 3.4028234663852886e38f     // FLT_MAX
#define LOF_BELOW_MARK 3.4028232635611926e38f   // the float below it: a threshold only marks exceed

__host__ __device__ constexpr int lof_ilog2c(int v) { return v <= 1 ? 0 : 1 + lof_ilog2c(v / 2); }

// 1.0f if x <= t, else 0.0f (also for NaN): FSET
__device__ __forceinline__ float lof_le1(float x, float t) {
  float d;
  asm("set.le.f32.f32 %0, %1, %2;" : "=f"(d) : "f"(x), "f"(t));
  return d;
}
__device__ __forceinline__ float2 lof_le2(float2 x, float t) { return make_float2(lof_le1(x.x, t), lof_le1(x.y, t)); }

// Level 0 of NP pairs: e = (x <= T0), u = x*e.  Returns the mask of UNFLAGGED samples (bit j = sample j of the
// pairs, 2*NP <= 32 bits) and raises `mu` to the largest unflagged sample (flagged ones count as 0).
// The mask is accumulated as fp32 numbers: per group of at most 8 (12 when NP == 12) pairs a Horner chain in base
// 4, acc = 4*acc + (e_even, e_odd), exact below 2^24; mask = acc.x + 2*acc.y.
template <int NP>
__device__ __forceinline__ uint32_t lof_level0(const float2 (&x2)[NP], float T0, float2 (&u2)[NP], float2 (&e2)[NP],
                                               float& mu) {
  constexpr int G = (NP <= 12) ? NP : 8;                  // pairs per chain: 4^G <= 2^24
  static_assert(NP % G == 0, "pairs per lane: <= 12, or a multiple of 8");
  const float2 c44 = make_float2(4.f, 4.f);
  uint32_t unf = 0;
  float a0 = mu, a1 = 0.f;
#pragma unroll
  for (int g = 0; g < NP / G; ++g) {
    float2 acc = make_float2(0.f, 0.f);
#pragma unroll
    for (int i = G - 1; i >= 0; --i) {
      const int m = g * G + i;
      e2[m] = lof_le2(x2[m], T0);
      u2[m] = __fmul2_rn(x2[m], e2[m]);
      acc = __ffma2_rn(acc, c44, e2[m]);
      if (m & 1) a1 = lof_max3(a1, u2[m].x, u2[m].y); else a0 = lof_max3(a0, u2[m].x, u2[m].y);
    }
    unf |= __float2uint_rz(fmaf(acc.y, 2.f, acc.x)) << (2 * G * g);
  }
  mu = fmaxf(a0, a1);
  return unf;
}

// bit j of `fb` set -> x[j] = LOF_MARK (a restart: samples flagged by a window enter level 0 as flagged)
template <int NP>
__device__ __forceinline__ void lof_mark(float2 (&x2)[NP], uint32_t fb) {
#pragma unroll
  for (int m = 0; m < NP; ++m) {
    x2[m].x = ((fb >> (2 * m)) & 1u) ? LOF_MARK : x2[m].x;
    x2[m].y = ((fb >> (2 * m + 1)) & 1u) ? LOF_MARK : x2[m].y;
  }
}

// ------------------------------------------------------------------------------------------------------------
// Column core, one lane per line of C samples (C = 16, 32, 64), pairs (2m, 2m+1).

// doubling step to windows of I = 2^K: position c gets X[c] + X[c + I/2] for every c + I <= C (ascending c, so
// X[c + I/2] is still the previous level)
template <int C, int K>
__device__ __forceinline__ void lof_col_step(float2 (&u2)[C / 2], float2 (&e2)[C / 2]) {
  constexpr int d = 1 << (K - 1), I = 1 << K;
  if constexpr (K == 1) {
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
      u2[m].x += u2[m].y; e2[m].x += e2[m].y;
      if (2 * m + 1 + I <= C) { u2[m].y += u2[m + 1].x; e2[m].y += e2[m + 1].x; }
    }
  } else {
#pragma unroll
    for (int m = 0; 2 * m + I <= C; ++m) {                 // C - I is even: position 2m+1 is beyond it only in
      if (2 * m + 1 + I <= C) {                            // the last pair, whose .y is never read again
        u2[m] = __fadd2_rn(u2[m], u2[m + d / 2]); e2[m] = __fadd2_rn(e2[m], e2[m + d / 2]);
      } else {
        u2[m].x += u2[m + d / 2].x; e2[m].x += e2[m + d / 2].x;
      }
    }
  }
}

// Test of iteration I = 2^K after its doubling step.  Returns (warp-uniform) whether any flag is new; `dead`
// (warp-uniform, meaningful when nothing is new) says that no window of I samples of the warp's lines has an
// unflagged mean above `tdead`: no later iteration can flag anything (lof_dead_level).
template <int C, int K>
__device__ __forceinline__ bool lof_col_eval(const float2 (&u2)[C / 2], const float2 (&e2)[C / 2], float thr,
                                             float tdead, uint64_t& fb, bool& dead) {
  constexpr int I = 1 << K;
  const float2 negT = make_float2(-thr, -thr), negD = make_float2(-tdead, -tdead);
  float tm[2] = {-INFINITY, -INFINITY}, td[2] = {-INFINITY, -INFINITY};
#pragma unroll
  for (int m = 0; 2 * m + I <= C; ++m) {
    if (2 * m + 1 + I <= C) {
      const float2 v = __ffma2_rn(e2[m], negT, u2[m]), w = __ffma2_rn(e2[m], negD, u2[m]);
      tm[m & 1] = lof_max3(tm[m & 1], v.x, v.y);           // u - e*T > 0 <=> window flagged
      td[m & 1] = lof_max3(td[m & 1], w.x, w.y);
    } else {
      tm[m & 1] = fmaxf(tm[m & 1], fmaf(e2[m].x, -thr, u2[m].x));
      td[m & 1] = fmaxf(td[m & 1], fmaf(e2[m].x, -tdead, u2[m].x));
    }
  }
  dead = __all_sync(0xffffffffu, fmaxf(td[0], td[1]) <= 0.f);
  const bool fired = fmaxf(tm[0], tm[1]) > 0.f;
  if (!__any_sync(0xffffffffu, fired)) return false;
  bool changed = false;
  if (fired) {
    uint32_t tg[4] = {0u, 0u, 0u, 0u};                     // partial masks: no serial chain
#pragma unroll
    for (int m = 0; 2 * m + I <= C; ++m) {
      tg[(2 * m) >> 5] |= (fmaf(e2[m].x, -thr, u2[m].x) > 0.f) ? (1u << ((2 * m) & 31)) : 0u;
      if (2 * m + 1 + I <= C) tg[2 + ((2 * m) >> 5)] |= (fmaf(e2[m].y, -thr, u2[m].y) > 0.f) ? (2u << ((2 * m) & 31)) : 0u;
    }
    const uint64_t trig = (uint64_t)(tg[0] | tg[2]) | ((uint64_t)(tg[1] | tg[3]) << 32);
    uint64_t dil = trig;
#pragma unroll
    for (int s = 1; s < I; s <<= 1) dil |= dil << s;
    const uint64_t nf = fb | dil;
    changed = nf != fb;
    fb = nf;
  }
  return __any_sync(0xffffffffu, changed);
}

// The run along one line of C samples: ld(c) returns sample c (called again on a restart; a sample flagged by
// an earlier run must read as LOF_MARK).  thr[k]: threshold of iteration k; dead[k]: its early-exit level.
// Returns the line's flag mask (bit c).  Every lane of the warp must call it (warp-uniform restarts and exits).
template <int C, class Ld>
__device__ __forceinline__ uint64_t lof_col_flag(Ld ld, const float* thr, const float* dead, int nlf) {
  static_assert(C == 16 || C == 32 || C == 64, "column core: 16, 32 or 64 samples per line");
  constexpr int KMAX = lof_ilog2c(C), NP = C / 2, NH = NP <= 16 ? NP : 16;
  float2 u2[NP], e2[NP];
  uint64_t fb = 0;
  const float T0 = thr[0], D0 = dead[0];
  int k_next = 1;
#pragma unroll 1
  for (;;) {
    // level 0 under the current mask, 32 samples at a time
    float mu = 0.f;
    uint64_t unf = 0;
#pragma unroll
    for (int h = 0; h < NP / NH; ++h) {
      float2 x2[NH], uh[NH], eh[NH];
#pragma unroll
      for (int m = 0; m < NH; ++m) x2[m] = make_float2(ld(2 * (h * NH + m)), ld(2 * (h * NH + m) + 1));
      if (k_next > 1) lof_mark<NH>(x2, (uint32_t)(fb >> (2 * NH * h)));
      unf |= (uint64_t)lof_level0<NH>(x2, T0, uh, eh, mu) << (2 * NH * h);
#pragma unroll
      for (int m = 0; m < NH; ++m) { u2[h * NH + m] = uh[m]; e2[h * NH + m] = eh[m]; }
    }
    fb = ~unf & (C == 64 ? ~0ull : ((1ull << C) - 1ull));
    // no unflagged sample above every later threshold: no later iteration can flag anything (lof_dead_level)
    if (__all_sync(0xffffffffu, mu <= D0)) break;
    // one test per level on the way down: past the last level -> done; new flags with levels to go ->
    // back to level 0 under the new mask
#define LOF_COL_LEVEL(K)                                                             \
    if (K > KMAX || K >= nlf) break;                                                 \
    lof_col_step<C, (K <= KMAX ? K : 1)>(u2, e2);                                    \
    if (K >= k_next) {                                                               \
      bool dead_;                                                                    \
      if (lof_col_eval<C, (K <= KMAX ? K : 1)>(u2, e2, thr[K], dead[K], fb, dead_) && \
          K + 1 <= KMAX && K + 1 < nlf) { k_next = K + 1; LOF_PROF_CNT(6); continue; } \
      if (dead_) break;                                                              \
    }
    LOF_COL_LEVEL(1) LOF_COL_LEVEL(2) LOF_COL_LEVEL(3) LOF_COL_LEVEL(4)
    LOF_COL_LEVEL(5) LOF_COL_LEVEL(6)
#undef LOF_COL_LEVEL
    break;
  }
  return fb;
}

// A warp's 32 column masks -> one word per channel (lane c & 31 ends up holding channel c's word).
template <int C>
__device__ __forceinline__ void lof_col_words(uint64_t fb, int lane, uint32_t& mine0, uint32_t& mine1) {
  mine0 = 0; mine1 = 0;
  if (__any_sync(0xffffffffu, fb != 0)) {
#pragma unroll
    for (int c = 0; c < C; ++c) {
      const uint32_t word = __ballot_sync(0xffffffffu, (fb >> c) & 1ull);
      if ((c & 31) == lane) { if (c < 32) mine0 = word; else mine1 = word; }
    }
  }
}

// ------------------------------------------------------------------------------------------------------------
// Column core, two lanes per line of 64 samples.  Lane l of the warp holds line p = l & 15 of the warp's 16
// lines, samples [32h, 32h+32) with h = l >> 4; the lane holding the other half is l ^ 16.  Half the registers
// per thread and half the lines per task of lof_col_flag<64>.  Windows that start in the lower half reach into
// the upper half through shuffles of the upper half's first D sums; a window that would leave the line gets
// -inf and never fires.
template <int D>
__device__ __forceinline__ void lof_pcol_step(float2 (&u2)[16], float2 (&e2)[16], int h) {
  if constexpr (D == 1) {
    float pu = __shfl_xor_sync(0xffffffffu, u2[0].x, 16);
    const float pe = __shfl_xor_sync(0xffffffffu, e2[0].x, 16);
    if (h) pu = -INFINITY;
#pragma unroll
    for (int m = 0; m < 16; ++m) {
      u2[m].x += u2[m].y; e2[m].x += e2[m].y;
      u2[m].y += (m + 1 < 16) ? u2[m + 1].x : pu; e2[m].y += (m + 1 < 16) ? e2[m + 1].x : pe;
    }
  } else {
    float2 pu[D / 2], pe[D / 2];
#pragma unroll
    for (int jj = 0; jj < D / 2; ++jj) {
      pu[jj].x = __shfl_xor_sync(0xffffffffu, u2[jj].x, 16); pu[jj].y = __shfl_xor_sync(0xffffffffu, u2[jj].y, 16);
      pe[jj].x = __shfl_xor_sync(0xffffffffu, e2[jj].x, 16); pe[jj].y = __shfl_xor_sync(0xffffffffu, e2[jj].y, 16);
      if (h) pu[jj] = make_float2(-INFINITY, -INFINITY);
    }
#pragma unroll
    for (int m = 0; m < 16; ++m) {
      u2[m] = __fadd2_rn(u2[m], (m + D / 2 < 16) ? u2[m + D / 2] : pu[m + D / 2 - 16]);
      e2[m] = __fadd2_rn(e2[m], (m + D / 2 < 16) ? e2[m + D / 2] : pe[m + D / 2 - 16]);
    }
  }
}

// Test of iteration I = 2^K <= 32 after its doubling step.  Returns (warp-uniform) whether any flag is new;
// `dead` as in lof_col_eval.
template <int K>
__device__ __forceinline__ bool lof_pcol_eval(const float2 (&u2)[16], const float2 (&e2)[16], int h, float thr,
                                              float tdead, uint32_t& fb, bool& dead) {
  constexpr int I = 1 << K;
  const float2 negT = make_float2(-thr, -thr), negD = make_float2(-tdead, -tdead);
  float tm[2] = {-INFINITY, -INFINITY}, td[2] = {-INFINITY, -INFINITY};
#pragma unroll
  for (int m = 0; m < 16; ++m) {
    const float2 v = __ffma2_rn(e2[m], negT, u2[m]), w = __ffma2_rn(e2[m], negD, u2[m]);
    tm[m & 1] = lof_max3(tm[m & 1], v.x, v.y);
    td[m & 1] = lof_max3(td[m & 1], w.x, w.y);
  }
  dead = __all_sync(0xffffffffu, fmaxf(td[0], td[1]) <= 0.f);
  const bool fired = fmaxf(tm[0], tm[1]) > 0.f;
  if (!__any_sync(0xffffffffu, fired)) return false;
  uint32_t tg[4] = {0u, 0u, 0u, 0u};                       // partial masks: no serial chain
  if (fired) {
#pragma unroll
    for (int m = 0; m < 16; ++m) {
      tg[m & 1] |= (fmaf(e2[m].x, -thr, u2[m].x) > 0.f) ? (1u << (2 * m)) : 0u;
      tg[2 + (m & 1)] |= (fmaf(e2[m].y, -thr, u2[m].y) > 0.f) ? (2u << (2 * m)) : 0u;
    }
  }
  const uint32_t trig = (tg[0] | tg[1]) | (tg[2] | tg[3]);
  uint64_t dil = trig;
#pragma unroll
  for (int s = 1; s < I; s <<= 1) dil |= dil << s;
  // windows started in the lower half reach into the upper half
  const uint32_t spill = __shfl_xor_sync(0xffffffffu, (uint32_t)(dil >> 32), 16);
  const uint32_t nf = fb | (uint32_t)dil | (h ? spill : 0u);
  const bool changed = nf != fb;
  fb = nf;
  return __any_sync(0xffffffffu, changed);
}

// The run along 16 lines x 64 samples by one warp: ld(j) returns this lane's sample 32h + j (called again on a
// restart).  Returns the lane's flag mask (bit j = sample 32h + j).
template <class Ld>
__device__ __forceinline__ uint32_t lof_pcol_flag(Ld ld, const float* thr, const float* dead, int nlf, int h) {
  float2 u2[16], e2[16];
  uint32_t fb = 0;
  const float T0 = thr[0], D0 = dead[0];
  int k_next = 1;
#pragma unroll 1
  for (;;) {
    float mu = 0.f;
    {
      float2 x2[16];
#pragma unroll
      for (int m = 0; m < 16; ++m) x2[m] = make_float2(ld(2 * m), ld(2 * m + 1));
      if (k_next > 1) lof_mark<16>(x2, fb);
      fb = ~lof_level0<16>(x2, T0, u2, e2, mu);
    }
    if (__all_sync(0xffffffffu, mu <= D0)) break;         // lof_dead_level: no later iteration can flag anything
#define LOF_PCOL_LEVEL(K)                                                          \
    if (K >= nlf) break;                                                           \
    lof_pcol_step<(1 << (K - 1))>(u2, e2, h);                                      \
    if (K >= k_next) {                                                             \
      bool dead_;                                                                  \
      if (lof_pcol_eval<K>(u2, e2, h, thr[K], dead[K], fb, dead_) && K + 1 < nlf) { \
        k_next = K + 1; LOF_PROF_CNT(6);                                            \
        continue;                                                                  \
      }                                                                            \
      if (dead_) break;                                                            \
    }
    LOF_PCOL_LEVEL(1) LOF_PCOL_LEVEL(2) LOF_PCOL_LEVEL(3) LOF_PCOL_LEVEL(4) LOF_PCOL_LEVEL(5)
#undef LOF_PCOL_LEVEL
    if (6 < nlf) {
      // I = 64: the one window that is the whole line
      const float ub = __shfl_xor_sync(0xffffffffu, u2[0].x, 16);
      const float eb = __shfl_xor_sync(0xffffffffu, e2[0].x, 16);
      const float v = fmaf(e2[0].x + eb, -thr[6], u2[0].x + ub);
      if (v > 0.f) fb = 0xFFFFFFFFu;             // both lanes of the pair see the same v
    }
    break;
  }
  return fb;
}

// ------------------------------------------------------------------------------------------------------------
// Row core: one warp per line of 32 L samples; lane l holds samples [l*L, l*L+L) as L/2 pairs.
// One doubling step of distance D (window 2D): partners beyond the lane's own L samples come from the
// following lanes by shuffle.  A window that leaves the line picks up some lane's own sums instead (the shuffle
// returns the caller's value): a harmless finite value, because it is a sum of valid windows, and lof_row_eval
// drops the window starts beyond the line's end before they can flag anything.
template <int L, int D>
__device__ __forceinline__ void lof_row_step(float2 (&u2)[L / 2], float2 (&e2)[L / 2], int lane) {
  constexpr int NP2 = L / 2;
  if constexpr (D == 1) {
    const float pu = __shfl_down_sync(0xffffffffu, u2[0].x, 1);
    const float pe = __shfl_down_sync(0xffffffffu, e2[0].x, 1);
#pragma unroll
    for (int m = 0; m < NP2; ++m) {
      u2[m].x += u2[m].y; e2[m].x += e2[m].y;
      u2[m].y += (m + 1 < NP2) ? u2[m + 1].x : pu; e2[m].y += (m + 1 < NP2) ? e2[m + 1].x : pe;
    }
  } else {
    constexpr int H = D / 2;                              // distance in pairs
    constexpr int NQ = H < NP2 ? H : NP2;                 // pairs whose partner lives in a following lane
    // first the sums, then the counts: the partners fetched by shuffle are live for one of them at a time
    {
      float2 pu[NQ];
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        const int m = NP2 - NQ + q, src = (m + H) % NP2, off = (m + H) / NP2;
        pu[q].x = __shfl_down_sync(0xffffffffu, u2[src].x, off); pu[q].y = __shfl_down_sync(0xffffffffu, u2[src].y, off);
      }
#pragma unroll
      for (int m = 0; m < NP2; ++m) u2[m] = __fadd2_rn(u2[m], (m + H < NP2) ? u2[m + H] : pu[m - (NP2 - NQ)]);
    }
    {
      float2 pe[NQ];
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        const int m = NP2 - NQ + q, src = (m + H) % NP2, off = (m + H) / NP2;
        pe[q].x = __shfl_down_sync(0xffffffffu, e2[src].x, off); pe[q].y = __shfl_down_sync(0xffffffffu, e2[src].y, off);
      }
#pragma unroll
      for (int m = 0; m < NP2; ++m) e2[m] = __fadd2_rn(e2[m], (m + H < NP2) ? e2[m + H] : pe[m - (NP2 - NQ)]);
    }
  }
}

// Test of iteration I = 2^K on a line after its doubling step: fire windows with u > e*T, dilate the fired
// starts over I samples across lanes, OR into fb.  Returns (warp-uniform) whether any flag is new; `dead`
// (warp-uniform) says that no window of I samples has an unflagged mean above `tdead` (lof_dead_level).
template <int L, int K>
__device__ __forceinline__ bool lof_row_eval(const float2 (&u2)[L / 2], const float2 (&e2)[L / 2], int lane, float thr,
                                             float tdead, uint32_t& fb, bool& dead) {
  constexpr int I = 1 << K;
  const float2 negT = make_float2(-thr, -thr), negD = make_float2(-tdead, -tdead);
  float tm[2] = {-INFINITY, -INFINITY}, td[2] = {-INFINITY, -INFINITY};
#pragma unroll
  for (int m = 0; m < L / 2; ++m) {
    const float2 v = __ffma2_rn(e2[m], negT, u2[m]), w = __ffma2_rn(e2[m], negD, u2[m]);
    tm[m & 1] = lof_max3(tm[m & 1], v.x, v.y);
    td[m & 1] = lof_max3(td[m & 1], w.x, w.y);
  }
  dead = __all_sync(0xffffffffu, fmaxf(td[0], td[1]) <= 0.f);
  if (!__any_sync(0xffffffffu, fmaxf(tm[0], tm[1]) > 0.f)) return false;
  uint32_t tg[4] = {0u, 0u, 0u, 0u};                       // partial masks: no serial chain
#pragma unroll
  for (int m = 0; m < L / 2; ++m) {
    tg[m & 1] |= (fmaf(e2[m].x, -thr, u2[m].x) > 0.f) ? (1u << (2 * m)) : 0u;
    tg[2 + (m & 1)] |= (fmaf(e2[m].y, -thr, u2[m].y) > 0.f) ? (2u << (2 * m)) : 0u;
  }
  uint32_t trig = (tg[0] | tg[1]) | (tg[2] | tg[3]);
  {
    // only windows that lie inside the line: starts t = lane*L + j <= 32*L - I
    int nv = 32 * L - I + 1 - lane * L;
    nv = nv < 0 ? 0 : (nv > L ? L : nv);
    trig &= nv >= 32 ? 0xFFFFFFFFu : ((1u << nv) - 1u);
  }
  // own windows, inside the lane's L bits
  uint32_t own = trig;
#pragma unroll
  for (int s = 1; s < I && s < 32; s <<= 1) own |= own << s;
  // windows started in earlier lanes: sample p is covered iff p < (last start before this lane) + I
  const int hi = trig ? (lane * L + 31 - __clz(trig)) : -(1 << 20);
  int pm = hi;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, pm, o); if (lane >= o) pm = max(pm, v); }
  int prev = __shfl_up_sync(0xffffffffu, pm, 1);
  if (lane == 0) prev = -(1 << 20);
  int cnt = prev + I - lane * L;
  cnt = cnt < 0 ? 0 : (cnt > L ? L : cnt);
  const uint32_t maskL = (L == 32) ? 0xFFFFFFFFu : ((1u << L) - 1u);
  const uint32_t pre = cnt >= 32 ? 0xFFFFFFFFu : ((1u << cnt) - 1u);
  const uint32_t nf = (fb | own | pre) & maskL;
  const bool changed = nf != fb;
  fb = nf;
  return __any_sync(0xffffffffu, changed);
}

// Sum of the lane's unflagged samples from the level-0 array u2 (flagged samples are 0 there): two packed
// partial sums, then (a.x + a.y) + (b.x + b.y)
template <int NP>
__device__ __forceinline__ float lof_lane_sum(const float2 (&u2)[NP]) {
  float2 a = make_float2(0.f, 0.f), b = make_float2(0.f, 0.f);
#pragma unroll
  for (int m = 0; m < NP; m += 2) { a = __fadd2_rn(a, u2[m]); if (m + 1 < NP) b = __fadd2_rn(b, u2[m + 1]); }
  return (a.x + a.y) + (b.x + b.y);
}

// The run along one line held by a warp (lane l: samples [l*L, l*L+L)): level 0, then the doubling levels with
// restarts and the early exit of lof_dead_level.  `load(x2, again)` fills the lane's samples as pairs; it is
// called once with again = false (samples flagged by an earlier run either hold LOF_MARK already or are named by
// the bits of `fb` on entry) and once more per restart with again = true (it may then read the raw data from
// anywhere: every flag so far is in fb and is re-applied).  The samples are not kept in registers across the
// levels.  fb leaves as the line's final mask (bit j = sample l*L + j); lane_sum as the sum of the lane's
// unflagged samples under that mask.  Warp-uniform control flow.
// KMAX: the largest iteration compiled in (windows up to 2^KMAX <= 512); the caller guarantees nlt <= KMAX + 1.
template <int L, int KMAX, class Load>
__device__ __forceinline__ void lof_row_flag(Load load, uint32_t& fb, const float* thr, const float* dead, int nlt,
                                             int lane, float& lane_sum) {
  static_assert(KMAX >= 1 && KMAX <= 9, "row core: windows of 2 .. 512 samples");
  constexpr int NP = L / 2;
  const uint32_t maskL = (L == 32) ? 0xFFFFFFFFu : ((1u << L) - 1u);
  float2 u2[NP], e2[NP];
  const float T0 = thr[0], D0 = dead[0];
  int k_next = 1;
#pragma unroll 1
  for (;;) {
    // level 0 (I = 1) under the current mask: x > threshold_1 on samples not yet flagged
    float mu = 0.f;
    {
      float2 x2[NP];
      load(x2, k_next > 1);
      if (__any_sync(0xffffffffu, fb != 0)) lof_mark<NP>(x2, fb);
      fb = ~lof_level0<NP>(x2, T0, u2, e2, mu) & maskL;
    }
    lane_sum = lof_lane_sum<NP>(u2);
    // no iteration left; nothing left that any later iteration could flag (lof_dead_level); nothing left to test
    if (k_next >= nlt) return;
    if (__all_sync(0xffffffffu, mu <= D0 || fb == maskL)) return;
    // one test per level on the way down: past the last level -> done; new flags with levels to go ->
    // back to level 0 under the new mask (continue), re-doubling up to k_next without testing
#define LOF_ROW_LEVEL(K)                                                                 \
    if (K > KMAX || K >= nlt) break;                                                     \
    lof_row_step<L, (1 << ((K <= KMAX ? K : 1) - 1))>(u2, e2, lane);                     \
    if (K >= k_next) {                                                                   \
      bool dead_;                                                                        \
      if (lof_row_eval<L, (K <= KMAX ? K : 1)>(u2, e2, lane, thr[K], dead[K], fb, dead_)) { \
        k_next = K + 1 < nlt ? K + 1 : 99;                /* 99: level 0 once more, for the row sum */ \
        LOF_PROF_CNT(7);                                                                  \
        continue;                                                                        \
      }                                                                                  \
      if (dead_) break;                                                                  \
    }
    LOF_ROW_LEVEL(1) LOF_ROW_LEVEL(2) LOF_ROW_LEVEL(3) LOF_ROW_LEVEL(4) LOF_ROW_LEVEL(5)
    LOF_ROW_LEVEL(6) LOF_ROW_LEVEL(7) LOF_ROW_LEVEL(8) LOF_ROW_LEVEL(9)
#undef LOF_ROW_LEVEL
    break;
  }
}
