// lof_history.cuh — the history flagger of PAPER.md:87-116 (pseudocode :97-113): one ring of
// float32 block means per (stream, channel) ("32bits"), fp64 arithmetic.
#pragma once
#include "lof_common.cuh"

// One thread per row (stream, channel).  Steps H1-H6 of DESIGN.md §2:
//   cur = rowsum/rowcnt; thr = mean(ring) + sens*stddev(ring) (population, storage order);
//   cur < thr -> push cur, else push thr and mark the row.
__global__ void lof_k_history_decide(float* __restrict__ ring, uint32_t* __restrict__ head,
                                     uint32_t* __restrict__ count, const double* __restrict__ rowsum,
                                     const uint32_t* __restrict__ rowcnt, uint8_t* __restrict__ row_flagged,
                                     uint64_t n_rows, uint32_t H, uint32_t min_fill, double sens) {
  const uint64_t r = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n_rows) return;
  float* h = ring + r * H;
  uint32_t hd = head[r], cnt = count[r];
  uint8_t flagged = 0;
  bool do_push = false; float v = 0.f;
  if (rowcnt[r] == 0) {
    flagged = 1;                                        // H1: nothing left to average; row stays flagged
  } else {
    const double cur = rowsum[r] / (double)rowcnt[r];   // meanOfUnflaggedSamples()
    if (cnt < min_fill) { do_push = true; v = (float)cur; }            // H3 (H3')
    else {
      double m = 0.0;
      for (uint32_t i = 0; i < cnt; ++i) m += (double)h[i];             // meanOfMeans(), :103
      m /= (double)cnt;
      double ss = 0.0;
      for (uint32_t i = 0; i < cnt; ++i) { const double d = (double)h[i] - m; ss += d * d; }
      const double sd = sqrt(ss / (double)cnt);                         // stddevOfMeans(), :104
      const double thr = m + sens * sd;                                 // :105-106
      do_push = true;
      if (cur < thr) v = (float)cur;                                    // :108-109
      else { v = (float)thr; flagged = 1; }                             // :110-113
    }
  }
  if (do_push) {
    h[hd] = v;
    hd = (hd + 1) % H;
    cnt = min(cnt + 1, H);
    head[r] = hd; count[r] = cnt;
  }
  row_flagged[r] = flagged;
}

// flagThisIntegrationTime(): every sample of a marked row, padding bits stay 0.
// One warp per row; rows not marked are left untouched.
__global__ void lof_k_history_fill(const uint8_t* __restrict__ row_flagged, uint32_t* __restrict__ flags,
                                   uint64_t n_rows, uint32_t W, uint32_t T) {
  const uint64_t r = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const uint32_t lane = threadIdx.x & 31;
  if (r >= n_rows || !row_flagged[r]) return;
  uint32_t* f = flags + r * W;
  const uint32_t last = (T & 31) ? ((1u << (T & 31)) - 1u) : 0xFFFFFFFFu;
  for (uint32_t w = lane; w < W; w += 32) f[w] = (w == W - 1) ? last : 0xFFFFFFFFu;
}

__global__ void lof_k_zero_u32(uint32_t* p, uint64_t n) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = 0;
}
