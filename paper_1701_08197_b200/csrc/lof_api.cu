// lof_api.cu — host side of the C-ABI in include/lof.h: context, scratch, launch sequencing.
// Every compute step is a kernel launch on the caller's stream; nothing here computes on the CPU
// except the factor table and launch geometry.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include "lof_common.cuh"
#include "lof_stats.cuh"
#include "lof_stats_lr.cuh"
#include "lof_flag_generic.cuh"
#include "lof_history.cuh"
#include "lof_fused.cuh"
#include "lof_longrow.cuh"
#include "lof_sir.cuh"
#include "lof_integrated.cuh"

static thread_local char g_cuda_err[256] = "";

#define LOF_CUDA(call)                                                              \
  do {                                                                              \
    cudaError_t e_ = (call);                                                        \
    if (e_ != cudaSuccess) {                                                        \
      snprintf(g_cuda_err, sizeof g_cuda_err, "%s: %s", #call, cudaGetErrorString(e_)); \
      return LOF_E_CUDA;                                                            \
    }                                                                               \
  } while (0)

struct lof_ctx {
  lof_params prm;
  LofKParams kp;
  int path;                       // 0 auto, 1 force generic
  int path_used;                  // what the last lof_flag_block ran: LOF_PATH_* (lof.h)
  int sm_count;
  uint32_t fused_grid;            // persistent grid of the fused kernel for this shape (0: no fused instantiation)
  uint32_t group_alloc;           // streams per group the scratch was allocated for (lof_set_group lowers `group`)
  uint64_t launches;
  bool block_pending;             // a lof_flag_block result is waiting for lof_history_update
  // geometry of the generic path
  uint32_t group;                 // streams per group (bounded so a group's input stays in L2)
  uint32_t n_chunks;              // statistics chunks per stream
  bool lr_dirty;                  // path 1 ran since path 0 last left its histogram slots zeroed
  uint32_t TT, halo, n_tiles;     // time tiling
  bool lr_freq, lr_time;          // register-resident long-row kernels usable (lof_longrow.cuh)
  uint32_t seg_out, seg_halo, n_seg;
  uint32_t co_out, n_co;          // cooperative 8192-sample tiles for wide cones
  size_t smem_freq, smem_time;
  // device memory owned by the context
  LofStreamState* d_state;
  LofStreamState* d_state2;       // MAD mode: state of the selection over |x - median|
  lof_stream_stats* d_stats2;
  uint32_t* d_hist;               // [group][4096] (the radix passes use 2048 of them)
  float* d_cand;                  // [group][LOF_LR_CAND] samples of the median's bin (lof_stats_lr.cuh)
  uint32_t* d_ctr;                // [group][2] non-finite samples, candidates gathered (lof_stats_lr.cuh)
  double* d_partial;              // [group][n_chunks][2]
  uint32_t* d_fmask;              // [S][C][W] mask after the frequency run
  double* d_part_sum;             // [group*C][n_tiles]
  uint32_t* d_part_cnt;
  double* d_rowsum;               // [S][C]
  uint32_t* d_rowcnt;
  lof_stream_stats* d_stats;      // [S] internal copy
  float* d_ring;                  // [S][C][H]
  uint32_t* d_head; uint32_t* d_count;
  uint8_t* d_row_flagged;
  // fully integrated mode (lof_integrated.cuh), allocated on first use: two inner contexts run the 1-D
  // SumThreshold over the spectrum (S x 1 x C) and over the series (S x 1 x T)
  lof_ctx* ig_freq; lof_ctx* ig_time;
  double* d_ig_rowpart; double* d_ig_colsum; float* d_ig_spec; float* d_ig_series;
  uint32_t* d_ig_cmask; uint32_t* d_ig_tmask; uint32_t ig_tiles;
  unsigned long long* d_diag;     // per-context diagnostics of the fused kernel: [0..4) counters, [8..16) cycles
  // staging for lof_flag_block_host
  void* d_in_stage; size_t in_stage_bytes;
  uint32_t* d_flags_stage;
  cudaStream_t host_stream;
};

static bool is_pow2(uint32_t v) { return v && !(v & (v - 1)); }

static int validate(const lof_params* p) {
  if (!p) return LOF_E_NULL;
  if (p->struct_size != sizeof(lof_params)) return LOF_E_PARAM;
  if (!p->n_streams || !p->n_channels || !p->n_time) return LOF_E_PARAM;
  if (p->n_channels > 256) return LOF_E_PARAM;
  if (!is_pow2(p->max_window) || p->max_window > 1024) return LOF_E_PARAM;
  if (!p->directions || (p->directions & ~3u)) return LOF_E_PARAM;
  if (!(p->p > 0.f) || !std::isfinite(p->p)) return LOF_E_PARAM;
  if (!(p->sensitivity > 0.f) || !std::isfinite(p->sensitivity)) return LOF_E_PARAM;
  if (!(p->start_threshold > 0.f) || !std::isfinite(p->start_threshold)) return LOF_E_PARAM;
  if ((uint64_t)p->n_channels * p->n_time > 0xFFFFFFFFull) return LOF_E_PARAM;
  // an empty ring has no mean: with min_fill = 0 the first threshold would be 0/0 and every later one NaN
  if (p->history_length > 0 && p->history_min_fill == 0) return LOF_E_PARAM;
  if (!std::isfinite(p->history_sensitivity)) return LOF_E_PARAM;
  if (!(p->sir_eta >= 0.f && p->sir_eta <= 1.f)) return LOF_E_PARAM;
  if (p->stats_mode > LOF_STATS_MAD) return LOF_E_PARAM;
  return LOF_OK;
}

extern "C" int lof_factor_table(const lof_params* p, double* out, uint32_t n_out) {
  if (!p || !out) return LOF_E_NULL;
  // factor_I = startThreshold * p^(log2 I) / I = startThreshold * (p/2)^k, I = 2^k
  double f = (double)p->start_threshold;
  const double r = (double)p->p / 2.0;
  for (uint32_t k = 0; k < n_out; ++k) { out[k] = f; f *= r; }
  return LOF_OK;
}

extern "C" const char* lof_strerror(int code) {
  switch (code) {
    case LOF_OK: return "success";
    case LOF_E_NULL: return "required pointer is NULL";
    case LOF_E_PARAM: return "invalid parameter";
    case LOF_E_ALIGN: return "device pointer not 16-byte aligned";
    case LOF_E_STATE: return "call order violated";
    case LOF_E_CUDA: return "CUDA runtime failure (see lof_last_cuda_error)";
    case LOF_E_SIZE: return "problem larger than the static scratch of a no-allocation entry point";
    default: return "unknown error";
  }
}
extern "C" const char* lof_last_cuda_error(void) { return g_cuda_err; }

template <class T>
static cudaError_t dev_alloc(T** p, size_t n) {
  *p = nullptr;
  if (n == 0) n = 1;
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T));
  if (e == cudaSuccess) e = cudaMemset(*p, 0, n * sizeof(T));
  return e;
}

extern "C" int lof_destroy(lof_ctx* c) {
  if (!c) return LOF_OK;
  cudaSetDevice(c->prm.device);
  cudaDeviceSynchronize();
  cudaFree(c->d_state); cudaFree(c->d_state2); cudaFree(c->d_stats2); cudaFree(c->d_hist); cudaFree(c->d_cand); cudaFree(c->d_ctr); cudaFree(c->d_partial); cudaFree(c->d_fmask);
  cudaFree(c->d_part_sum); cudaFree(c->d_part_cnt); cudaFree(c->d_rowsum); cudaFree(c->d_rowcnt);
  cudaFree(c->d_stats); cudaFree(c->d_ring); cudaFree(c->d_head); cudaFree(c->d_count);
  cudaFree(c->d_row_flagged); cudaFree(c->d_diag); cudaFree(c->d_in_stage); cudaFree(c->d_flags_stage);
  if (c->host_stream) cudaStreamDestroy(c->host_stream);
  lof_destroy(c->ig_freq); lof_destroy(c->ig_time);
  cudaFree(c->d_ig_rowpart); cudaFree(c->d_ig_colsum); cudaFree(c->d_ig_spec); cudaFree(c->d_ig_series);
  cudaFree(c->d_ig_cmask); cudaFree(c->d_ig_tmask);
  delete c;
  return LOF_OK;
}

static cudaError_t lof_generic_set_attributes(size_t smem_freq, size_t smem_time) {
  cudaError_t e = cudaSuccess;
  auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  const int f = (int)smem_freq, t = (int)smem_time;
  A(cudaFuncSetAttribute(lof_k_freq_generic<InF32>, cudaFuncAttributeMaxDynamicSharedMemorySize, f));
  A(cudaFuncSetAttribute(lof_k_freq_generic<InCI16>, cudaFuncAttributeMaxDynamicSharedMemorySize, f));
  A(cudaFuncSetAttribute(lof_k_time_generic<InF32>, cudaFuncAttributeMaxDynamicSharedMemorySize, t));
  A(cudaFuncSetAttribute(lof_k_time_generic<InCI16>, cudaFuncAttributeMaxDynamicSharedMemorySize, t));
  A(cudaFuncSetAttribute(lof_k_freq_stg<32, InF32>, cudaFuncAttributeMaxDynamicSharedMemorySize, LOF_FREQ_SMEM(32)));
  A(cudaFuncSetAttribute(lof_k_freq_stg<32, InCI16>, cudaFuncAttributeMaxDynamicSharedMemorySize, LOF_FREQ_SMEM(32)));
  A(cudaFuncSetAttribute(lof_k_freq_stg<64, InF32>, cudaFuncAttributeMaxDynamicSharedMemorySize, LOF_FREQ_SMEM(64)));
  A(cudaFuncSetAttribute(lof_k_freq_stg<64, InCI16>, cudaFuncAttributeMaxDynamicSharedMemorySize, LOF_FREQ_SMEM(64)));
  A(cudaFuncSetAttribute(lof_k_time_seg<InF32>, cudaFuncAttributeMaxDynamicSharedMemorySize, LOF_SEG_SMEM));
  A(cudaFuncSetAttribute(lof_k_time_seg<InCI16>, cudaFuncAttributeMaxDynamicSharedMemorySize, LOF_SEG_SMEM));
  A(cudaFuncSetAttribute(lof_k_time_coop<InF32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(LofCoopSmem)));
  A(cudaFuncSetAttribute(lof_k_time_coop<InCI16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(LofCoopSmem)));
  return e;
}

static cudaError_t fused_prepare_any(lof_ctx* c);       // below, with the fused launch

static uint32_t ilog2(uint32_t v) { uint32_t k = 0; while ((1u << (k + 1)) <= v) ++k; return k; }

extern "C" int lof_create(const lof_params* p, lof_ctx** out) {
  if (!out) return LOF_E_NULL;
  *out = nullptr;
  int rc = validate(p);
  if (rc) return rc;
  int ndev = 0;
  LOF_CUDA(cudaGetDeviceCount(&ndev));
  if (p->device < 0 || p->device >= ndev) {
    snprintf(g_cuda_err, sizeof g_cuda_err, "device %d not present (%d devices)", p->device, ndev);
    return LOF_E_CUDA;
  }
  LOF_CUDA(cudaSetDevice(p->device));
  lof_ctx* c = new (std::nothrow) lof_ctx();
  if (!c) return LOF_E_CUDA;
  memset(c, 0, sizeof *c);
  c->prm = *p;
  {
    cudaError_t ea = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, p->device);
    if (ea != cudaSuccess) {
      snprintf(g_cuda_err, sizeof g_cuda_err, "cudaDeviceGetAttribute: %s", cudaGetErrorString(ea));
      delete c;
      return LOF_E_CUDA;
    }
  }
  const uint32_t S = p->n_streams, C = p->n_channels, T = p->n_time, W = (T + 31) / 32;
  LofKParams& kp = c->kp;
  kp.S = S; kp.C = C; kp.T = T; kp.W = W;
  kp.n_levels = ilog2(p->max_window) + 1;
  kp.n_lev_f = (p->directions & LOF_DIR_FREQ) ? ilog2(p->max_window < C ? p->max_window : C) + 1 : 0;
  kp.n_lev_t = (p->directions & LOF_DIR_TIME) ? ilog2(p->max_window < T ? p->max_window : T) + 1 : 0;
  kp.s0 = 0;
  lof_factor_table(p, kp.factor, LOF_MAX_LEVELS);
  kp.sensitivity = (double)p->sensitivity;

  const uint64_t N = (uint64_t)C * T;
  c->n_chunks = (uint32_t)((N + LOF_STATS_CHUNK - 1) / LOF_STATS_CHUNK);
  // groups of streams per launch sequence.  Measured on B200: groups small enough to stay in L2 (80 MB, so
  // that the five kernels of a group re-read the input from L2) were 23 % SLOWER than groups of 640 MB — the
  // kernels are bound by instruction issue, not by bandwidth, and every launch of a small group pays its ramp
  // and its tail.  The bound below only limits the per-group scratch (histograms, candidate lists, partials).
  const uint64_t group_bytes = 640ull << 20;
  uint64_t g = group_bytes / (N * 4);
  if (g < 1) g = 1;
  if (g > 1024) g = 1024;
  if (g > S) g = S;
  c->group = (uint32_t)g;
  c->group_alloc = c->group;
  // time tiling: halo = dependency cone sum_k (2^k - 1) of the time run, rounded up to 32
  uint32_t cone = 0;
  for (uint32_t k = 0; k < kp.n_lev_t; ++k) cone += (1u << k) - 1;
  const uint32_t TT0 = 4096;
  if (T <= TT0 + 2 * ((cone + 31) & ~31u)) { c->TT = (T + 31) & ~31u; c->halo = 0; c->n_tiles = 1; }
  else { c->TT = TT0; c->halo = (cone + 31) & ~31u; c->n_tiles = (T + TT0 - 1) / TT0; }
  // register-resident long-row kernels: columns of 16/32/64 channels; row segments of 1024 samples whose
  // halo (the cone, rounded up to 32) leaves at least half of the segment as output
  c->lr_freq = (C == 16 || C == 32 || C == 64);
  c->seg_halo = (cone + 31) & ~31u;
  c->lr_time = c->seg_halo <= 256;
  c->seg_out = c->lr_time ? LOF_LR_TILE - 2 * c->seg_halo : LOF_LR_TILE;
  c->n_seg = (T + c->seg_out - 1) / c->seg_out;
  c->co_out = LOF_CO_TILE - 2 * c->seg_halo;             // seg_halo <= 2048 for max_window <= 1024
  c->n_co = (T + c->co_out - 1) / c->co_out;
  c->smem_freq = (size_t)C * 32 * LOF_GEN_BYTES_PER_ELEM;
  c->smem_time = (size_t)((c->TT + 2 * c->halo + 31) & ~31u) * LOF_GEN_BYTES_PER_ELEM;

  cudaError_t e = cudaSuccess;
  auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  A(dev_alloc(&c->d_state, S));
  if (p->stats_mode == LOF_STATS_MAD) { A(dev_alloc(&c->d_state2, S)); A(dev_alloc(&c->d_stats2, S)); }
  A(dev_alloc(&c->d_hist, (size_t)c->group * LOF_LR_NBINS));
  A(dev_alloc(&c->d_cand, (size_t)c->group * LOF_LR_CAND));
  A(dev_alloc(&c->d_ctr, (size_t)c->group * 2));
  A(dev_alloc(&c->d_partial, (size_t)c->group * c->n_chunks * 2));
  A(dev_alloc(&c->d_fmask, (size_t)S * C * W));
  size_t n_part = c->n_tiles > c->n_seg ? c->n_tiles : c->n_seg;
  if (c->n_co > n_part) n_part = c->n_co;
  A(dev_alloc(&c->d_part_sum, (size_t)c->group * C * n_part));
  A(dev_alloc(&c->d_part_cnt, (size_t)c->group * C * n_part));
  A(dev_alloc(&c->d_rowsum, (size_t)S * C));
  A(dev_alloc(&c->d_rowcnt, (size_t)S * C));
  A(dev_alloc(&c->d_stats, S));
  A(dev_alloc(&c->d_ring, (size_t)S * C * p->history_length));
  A(dev_alloc(&c->d_head, (size_t)S * C));
  A(dev_alloc(&c->d_count, (size_t)S * C));
  A(dev_alloc(&c->d_row_flagged, (size_t)S * C));
  A(dev_alloc(&c->d_diag, (size_t)LOF_DIAG_WORDS));
  if (e == cudaSuccess) e = lof_generic_set_attributes(c->smem_freq, c->smem_time);
  if (e == cudaSuccess) e = fused_prepare_any(c);
  if (e != cudaSuccess) {
    snprintf(g_cuda_err, sizeof g_cuda_err, "lof_create: %s", cudaGetErrorString(e));
    lof_destroy(c);
    return LOF_E_CUDA;
  }
  *out = c;
  return LOF_OK;
}

// ---- the hot path: statistics -> thresholds -> SumThreshold(freq) -> SumThreshold(time) -> pack
template <class In>
static int flag_block_generic(lof_ctx* c, In in, uint32_t* d_flags, cudaStream_t st) {
  const uint32_t S = c->prm.n_streams, C = c->prm.n_channels;
  for (uint32_t s0 = 0; s0 < S; s0 += c->group) {
    const uint32_t G = (S - s0 < c->group) ? S - s0 : c->group;
    LofKParams kp = c->kp;
    kp.s0 = s0;
    const uint32_t nb = G * c->n_chunks;
    if (c->path == 0) {
      // two passes over the group's input, three launches (lof_stats_lr.cuh): about twelve CTAs per SM over the launch, each
      // over consecutive chunks of one stream
      uint32_t cpb = (nb + (uint32_t)c->sm_count * 12 - 1) / ((uint32_t)c->sm_count * 12);
      if (cpb < 1) cpb = 1;
      const uint32_t n_blk = (c->n_chunks + cpb - 1) / cpb;
      if (c->lr_dirty) {        // the radix passes of path 1 used the slots' histograms since the last group here
        lof_k_zero_u32<<<(unsigned)(((size_t)c->group * LOF_LR_NBINS + 255) / 256), 256, 0, st>>>(c->d_hist, (size_t)c->group * LOF_LR_NBINS);
        lof_k_zero_u32<<<1, 256, 0, st>>>(c->d_ctr, (size_t)c->group * 2);
        c->lr_dirty = false;
        c->launches += 2;
      }
      lof_k_lr_hist<In><<<G * n_blk, LOF_STATS_THREADS, 0, st>>>(in, kp, c->d_state, c->d_hist, c->d_ctr, c->d_partial,
                                                               c->n_chunks, cpb, n_blk);
      lof_k_lr_gather<In><<<G * n_blk, LOF_STATS_THREADS, 0, st>>>(in, kp, c->d_state, c->d_hist, c->d_ctr, c->d_cand,
                                                                 c->n_chunks, cpb, n_blk);
      lof_k_lr_select2<In><<<G, 256, 0, st>>>(in, kp, c->d_state, c->d_hist, c->d_ctr, c->d_partial, c->n_chunks,
                                              c->d_cand, c->d_stats);
      c->launches += 3;
    } else {
      // three radix passes (lof_stats.cuh): the second implementation, kept for tests and as a reference
      c->lr_dirty = true;
      lof_k_clear_state<<<(G + 255) / 256, 256, 0, st>>>(c->d_state, s0, G);
      lof_k_zero_u32<<<(unsigned)(((size_t)G * LOF_HIST_BINS + 255) / 256), 256, 0, st>>>(c->d_hist, (size_t)G * LOF_HIST_BINS);
      lof_k_hist<In, 0><<<nb, LOF_STATS_THREADS, 0, st>>>(in, kp, c->d_state, c->d_hist, c->d_partial, c->n_chunks);
      lof_k_scan<In, 0><<<G, 256, 0, st>>>(in, kp, c->d_state, c->d_hist, c->d_partial, c->n_chunks, c->d_stats);
      lof_k_hist<In, 1><<<nb, LOF_STATS_THREADS, 0, st>>>(in, kp, c->d_state, c->d_hist, c->d_partial, c->n_chunks);
      lof_k_scan<In, 1><<<G, 256, 0, st>>>(in, kp, c->d_state, c->d_hist, c->d_partial, c->n_chunks, c->d_stats);
      lof_k_hist<In, 2><<<nb, LOF_STATS_THREADS, 0, st>>>(in, kp, c->d_state, c->d_hist, c->d_partial, c->n_chunks);
      lof_k_scan<In, 2><<<G, 256, 0, st>>>(in, kp, c->d_state, c->d_hist, c->d_partial, c->n_chunks, c->d_stats);
      c->launches += 8;
    }
    if (c->prm.stats_mode == LOF_STATS_MAD) {
      // robust scale: the rank floor(N/2) element of |x - median| by the three radix passes, then 1.4826 * MAD
      // replaces the stddev in the thresholds (R1)
      InAbsDev<In> dev{in, c->d_state, (uint64_t)C * c->prm.n_time, in.p};
      lof_k_clear_state<<<(G + 255) / 256, 256, 0, st>>>(c->d_state2, s0, G);
      lof_k_zero_u32<<<(unsigned)(((size_t)G * LOF_HIST_BINS + 255) / 256), 256, 0, st>>>(c->d_hist, (size_t)G * LOF_HIST_BINS);
      lof_k_hist<InAbsDev<In>, 0><<<nb, LOF_STATS_THREADS, 0, st>>>(dev, kp, c->d_state2, c->d_hist, c->d_partial, c->n_chunks);
      lof_k_scan<InAbsDev<In>, 0><<<G, 256, 0, st>>>(dev, kp, c->d_state2, c->d_hist, c->d_partial, c->n_chunks, c->d_stats2);
      lof_k_hist<InAbsDev<In>, 1><<<nb, LOF_STATS_THREADS, 0, st>>>(dev, kp, c->d_state2, c->d_hist, c->d_partial, c->n_chunks);
      lof_k_scan<InAbsDev<In>, 1><<<G, 256, 0, st>>>(dev, kp, c->d_state2, c->d_hist, c->d_partial, c->n_chunks, c->d_stats2);
      lof_k_hist<InAbsDev<In>, 2><<<nb, LOF_STATS_THREADS, 0, st>>>(dev, kp, c->d_state2, c->d_hist, c->d_partial, c->n_chunks);
      lof_k_scan<InAbsDev<In>, 2><<<G, 256, 0, st>>>(dev, kp, c->d_state2, c->d_hist, c->d_partial, c->n_chunks, c->d_stats2);
      lof_k_mad_apply<<<(G + 255) / 256, 256, 0, st>>>(c->d_state, c->d_state2, kp, c->d_stats, s0, G);
      c->lr_dirty = true;
      c->launches += 9;
    }
    const bool fast = c->path == 0;                     // path 1 forces the shared-memory generic kernels
    int used = LOF_PATH_GENERIC;
    if (kp.n_lev_f) {
      // persistent: as many CTAs as the SMs hold (2 / 1 per SM for 32 / 64 channels)
      const uint32_t nb_all = (uint32_t)(((uint64_t)G * kp.W + LOF_LR_WARPS - 1) / LOF_LR_WARPS);
      const uint32_t nb_res = (uint32_t)c->sm_count * (C == 32 ? 2u : 1u);
      const uint32_t nb_f = nb_all < nb_res ? nb_all : nb_res;
      if (fast && c->lr_freq && C == 16)                  // not staged: a CTA per 8 units
        lof_k_freq_reg<16, In><<<nb_all, LOF_LR_THREADS, 0, st>>>(in, kp, c->d_state, c->d_fmask, G);
      else if (fast && c->lr_freq && C == 32)
        lof_k_freq_stg<32, In><<<nb_f, LOF_LR_THREADS, LOF_FREQ_SMEM(32), st>>>(in, kp, c->d_state, c->d_fmask, G);
      else if (fast && c->lr_freq && C == 64)
        lof_k_freq_stg<64, In><<<nb_f, LOF_LR_THREADS, LOF_FREQ_SMEM(64), st>>>(in, kp, c->d_state, c->d_fmask, G);
      else
        lof_k_freq_generic<In><<<G * kp.W, LOF_GEN_THREADS, c->smem_freq, st>>>(in, kp, c->d_state, c->d_fmask);
      c->launches += 1;
    }
    const uint32_t rows = G * C;
    uint32_t n_part;
    const bool freq_reg = !kp.n_lev_f || (fast && c->lr_freq);
    if (fast && c->lr_time) {
      if (freq_reg) used = LOF_PATH_LONGROW_SEG;
      n_part = c->n_seg;
      uint32_t nb_t = (uint32_t)(((uint64_t)rows * n_part + LOF_LR_WARPS - 1) / LOF_LR_WARPS);
      if (nb_t > (uint32_t)c->sm_count * 2) nb_t = (uint32_t)c->sm_count * 2;     // persistent: two CTAs per SM
      lof_k_time_seg<In><<<nb_t, LOF_LR_THREADS, LOF_SEG_SMEM, st>>>(in, kp, c->d_state, c->d_fmask, d_flags, c->d_part_sum,
                                                        c->d_part_cnt, c->d_stats, c->seg_out, c->seg_halo, n_part, rows);
    } else if (fast && kp.n_lev_t <= 10) {                // the cooperative kernel exchanges windows of up to 512
      if (freq_reg) used = LOF_PATH_LONGROW_COOP;
      n_part = c->n_co;
      {
        const uint32_t n_units = rows * n_part;               // persistent: two CTAs per SM walk over the tiles
        const uint32_t grid = n_units < (uint32_t)c->sm_count * 2 ? n_units : (uint32_t)c->sm_count * 2;
        lof_k_time_coop<In><<<grid, LOF_CO_WARPS * 32, sizeof(LofCoopSmem), st>>>(
            in, kp, c->d_state, c->d_fmask, d_flags, c->d_part_sum, c->d_part_cnt, c->d_stats, c->co_out, c->seg_halo, n_part,
            n_units);
      }
    } else {
      n_part = c->n_tiles;
      lof_k_time_generic<In><<<rows * c->n_tiles, LOF_GEN_THREADS, c->smem_time, st>>>(
          in, kp, c->d_state, c->d_fmask, d_flags, c->d_part_sum, c->d_part_cnt, c->d_stats, c->TT, c->halo, c->n_tiles);
    }
    lof_k_rowsum_final<<<(rows + 255) / 256, 256, 0, st>>>(c->d_part_sum, c->d_part_cnt, c->d_rowsum, c->d_rowcnt,
                                                           (uint64_t)s0 * C, rows, n_part);
    c->launches += 2;
    c->path_used = used;
  }
  LOF_CUDA(cudaGetLastError());
  return LOF_OK;
}

// ---- fused path: streams that fit one SM's shared memory (lof_fused.cuh)
// Shapes with a fused instantiation, as (C, L) with T = 32 L.
#define LOF_FUSED_SHAPES(X) X(64, 24) X(16, 24) X(32, 24) X(16, 8) X(32, 32) X(64, 16) X(16, 32)

// lof_create: opt the kernel of this shape in to its shared memory and size the persistent grid (SMs x CTAs per
// SM) once; both are per device, so every context does it for its own device (idempotent, no shared state).
template <int C, int L>
static cudaError_t fused_prepare(lof_ctx* c) {
  using Cfg = LofFusedCfg<C, L>;
  cudaError_t e = cudaFuncSetAttribute(lof_k_fused<C, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::smem_bytes);
  if (e != cudaSuccess) return e;
  int per_sm = 1;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lof_k_fused<C, L>, Cfg::NT, Cfg::smem_bytes);
  if (e != cudaSuccess) return e;
  if (per_sm < 1) per_sm = 1;
  uint32_t grid = (uint32_t)(c->sm_count * per_sm);
  if (grid > c->prm.n_streams) grid = c->prm.n_streams;
  c->fused_grid = grid;
  return cudaSuccess;
}

static cudaError_t fused_prepare_any(lof_ctx* c) {
  const uint32_t C = c->prm.n_channels, T = c->prm.n_time;
  c->fused_grid = 0;
  if (c->kp.n_lev_t > LOF_FUSED_KMAX + 1) return cudaSuccess;   // the fused kernel compiles windows of up to 64 samples in
#define X(CC, LL) if (C == CC && T == 32 * LL) return fused_prepare<CC, LL>(c);
  LOF_FUSED_SHAPES(X)
#undef X
  return cudaSuccess;
}

// returns 1 if the shape has a fused instantiation and it was launched, 0 if not, <0 on error
static int flag_block_fused(lof_ctx* c, const float* d_power, uint32_t* d_flags, cudaStream_t st) {
  const uint32_t C = c->prm.n_channels, T = c->prm.n_time;
  if (!c->fused_grid) return 0;
  // the ticket counter of the kernel's dynamic hand-out of streams starts every launch at zero (reset here rather than
  // by the last CTA to leave: a launch that died would otherwise leave the next one skipping streams)
  LOF_CUDA(cudaMemsetAsync(c->d_diag + LOF_DIAG_TICKET, 0, sizeof(unsigned long long), st));
  bool done = false;
#define X(CC, LL)                                                                                              \
  if (!done && C == CC && T == 32 * LL) {                                                                      \
    lof_k_fused<CC, LL><<<c->fused_grid, LofFusedCfg<CC, LL>::NT, LofFusedCfg<CC, LL>::smem_bytes, st>>>(      \
        d_power, d_flags, c->d_stats, c->d_rowsum, c->d_rowcnt, c->kp, c->d_diag);                             \
    done = true;                                                                                               \
  }
  LOF_FUSED_SHAPES(X)
#undef X
  if (!done) return 0;
  c->launches += 1;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(g_cuda_err, sizeof g_cuda_err, "fused launch: %s", cudaGetErrorString(e));
    return LOF_E_CUDA;
  }
  return 1;
}
static int flag_block_fused(lof_ctx*, const int16_t*, uint32_t*, cudaStream_t) { return 0; }

// ---- SIR operator on the packed mask (lof_sir.cuh): frequency, then time; ping-pong between the caller's
// flags and the context's mask buffer
// the shortest run that the operator grows: the smallest m <= limit with floor(eta * m) >= 1 (limit + 1 if none)
static uint32_t sir_min_run(float eta, uint32_t limit) {
  uint32_t m = 1;
  while (m <= limit && (uint32_t)std::floor((double)eta * (double)m) == 0) ++m;
  return m;
}

template <int G>
static void sir_time_launch(const uint32_t* in, uint32_t* out, lof_ctx* c, cudaStream_t st) {
  const uint64_t rows = (uint64_t)c->prm.n_streams * c->prm.n_channels;
  const uint64_t threads = rows * G;
  const unsigned grid = (unsigned)((threads + 255) / 256);
  const size_t stage = (size_t)2 * (256 / G) * c->kp.W * 4;   // in and out copies of the CTA's rows
  if (stage <= 40 * 1024)
    lof_k_sir_time<G, true><<<grid, 256, stage, st>>>(in, out, c->d_stats, rows, c->prm.n_channels, c->kp.W,
                                                      c->prm.n_time, c->prm.sir_eta, sir_min_run(c->prm.sir_eta, c->prm.n_time));
  else
    lof_k_sir_time<G, false><<<grid, 256, 0, st>>>(in, out, c->d_stats, rows, c->prm.n_channels, c->kp.W,
                                                   c->prm.n_time, c->prm.sir_eta, sir_min_run(c->prm.sir_eta, c->prm.n_time));
}

static int sir_apply(lof_ctx* c, uint32_t* d_flags, cudaStream_t st) {
  const float eta = c->prm.sir_eta;
  if (!(eta > 0.f)) return LOF_OK;
  const uint32_t C = c->prm.n_channels, W = c->kp.W;
  const size_t words = (size_t)c->prm.n_streams * C * W;
  uint32_t* cur = d_flags;
  uint32_t* other = c->d_fmask;
  if (c->prm.directions & LOF_DIR_FREQ) {
    const uint32_t m_min = sir_min_run(eta, C);          // shortest run that grows at all
    const uint64_t n_cols = (uint64_t)c->prm.n_streams * W;
    const dim3 g8(c->prm.n_streams, (W + 7) / 8);                // a warp per word column, 8 per CTA
    if (C == 64) lof_k_sir_freq_reg<64><<<g8, 256, 0, st>>>(cur, other, c->d_stats, W, eta, m_min);
    else if (C == 32) lof_k_sir_freq_reg<32><<<g8, 256, 0, st>>>(cur, other, c->d_stats, W, eta, m_min);
    else if (C == 16) lof_k_sir_freq_reg<16><<<g8, 256, 0, st>>>(cur, other, c->d_stats, W, eta, m_min);
    else lof_k_sir_freq<<<(unsigned)((n_cols + 255) / 256), 256, 0, st>>>(cur, other, c->d_stats, n_cols, C, W, eta, m_min);
    c->launches += 1;
    uint32_t* t = cur; cur = other; other = t;
  }
  if (c->prm.directions & LOF_DIR_TIME) {
    uint32_t G = 1;
    while (G < 32 && G * 8 < W) G <<= 1;                  // about eight words per lane
    switch (G) {
      case 1: sir_time_launch<1>(cur, other, c, st); break;
      case 2: sir_time_launch<2>(cur, other, c, st); break;
      case 4: sir_time_launch<4>(cur, other, c, st); break;
      case 8: sir_time_launch<8>(cur, other, c, st); break;
      case 16: sir_time_launch<16>(cur, other, c, st); break;
      default: sir_time_launch<32>(cur, other, c, st); break;
    }
    c->launches += 1;
    uint32_t* t = cur; cur = other; other = t;
  }
  LOF_CUDA(cudaGetLastError());
  if (cur != d_flags) LOF_CUDA(cudaMemcpyAsync(d_flags, cur, words * 4, cudaMemcpyDeviceToDevice, st));
  return LOF_OK;
}

template <class In>
static int flag_block_any(lof_ctx* c, In in, uint32_t* d_flags, lof_stream_stats* d_stats, void* cuda_stream) {
  if (!c || !in.p || !d_flags) return LOF_E_NULL;
  if (((uintptr_t)in.p & 15) || ((uintptr_t)d_flags & 15) || ((uintptr_t)d_stats & 7)) return LOF_E_ALIGN;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LOF_CUDA(cudaSetDevice(c->prm.device));
  // (the MAD scale needs a second selection pass: it runs on the multi-kernel paths)
  int rc = (c->path == 0 && c->prm.stats_mode == LOF_STATS_PLAIN) ? flag_block_fused(c, in.p, d_flags, st) : 0;
  if (rc < 0) return rc;
  if (rc == 1) c->path_used = LOF_PATH_FUSED;
  if (rc == 0) { rc = flag_block_generic(c, in, d_flags, st); if (rc) return rc; }
  rc = sir_apply(c, d_flags, st);
  if (rc) return rc;
  if (d_stats)
    LOF_CUDA(cudaMemcpyAsync(d_stats, c->d_stats, (size_t)c->prm.n_streams * sizeof(lof_stream_stats),
                             cudaMemcpyDeviceToDevice, st));
  c->block_pending = true;
  return LOF_OK;
}

extern "C" int lof_flag_block(lof_ctx* c, const float* d_power, uint32_t* d_flags, lof_stream_stats* d_stats,
                              void* cuda_stream) {
  return flag_block_any(c, InF32{d_power}, d_flags, d_stats, cuda_stream);
}
extern "C" int lof_flag_block_ci16(lof_ctx* c, const int16_t* d_volt, uint32_t* d_flags, lof_stream_stats* d_stats,
                                   void* cuda_stream) {
  return flag_block_any(c, InCI16{d_volt}, d_flags, d_stats, cuda_stream);
}

// ---- fully integrated mode
static int integrated_prepare(lof_ctx* c) {
  if (c->d_ig_colsum) return LOF_OK;
  const uint32_t S = c->prm.n_streams, C = c->prm.n_channels, T = c->prm.n_time;
  lof_params q = c->prm;
  q.n_channels = 1; q.directions = LOF_DIR_TIME; q.history_length = 0; q.sir_eta = 0.f;
  q.n_time = C;
  int rc = lof_create(&q, &c->ig_freq);
  if (rc) return rc;
  q.n_time = T;
  rc = lof_create(&q, &c->ig_time);
  if (rc) return rc;
  c->ig_tiles = (T + LOF_IG_TILE - 1) / LOF_IG_TILE;
  cudaError_t e = cudaSuccess;
  auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  A(dev_alloc(&c->d_ig_rowpart, (size_t)S * C * c->ig_tiles));
  A(dev_alloc(&c->d_ig_spec, (size_t)S * ((C + 3) & ~3u)));
  A(dev_alloc(&c->d_ig_series, (size_t)S * T + 4));
  A(dev_alloc(&c->d_ig_cmask, (size_t)S * ((C + 31) / 32) + 4));
  A(dev_alloc(&c->d_ig_tmask, (size_t)S * c->kp.W + 4));
  A(dev_alloc(&c->d_ig_colsum, (size_t)S * T));
  if (e != cudaSuccess) {
    snprintf(g_cuda_err, sizeof g_cuda_err, "integrated mode scratch: %s", cudaGetErrorString(e));
    return LOF_E_CUDA;
  }
  return LOF_OK;
}

// One SumThreshold run over S vectors of n samples: the single-CTA kernel for short vectors, an inner context
// (statistics kernels + row kernels of the long-row path) for long ones.
// vectors of n samples take the warp-per-vector kernel (the row core runs windows of up to 512 samples)
static bool integrated_warp_path(const lof_ctx* c, uint32_t n) {
  return n <= 1024 && (c->prm.max_window < 1024 || n < 1024);
}
static int integrated_run(lof_ctx* c, lof_ctx* inner, const float* d_vec, uint32_t n, uint32_t* d_mask,
                          lof_stream_stats* d_stats_out, cudaStream_t st, LofVecFuse fz = LofVecFuse{}) {
  const uint32_t S = c->prm.n_streams;
  if (integrated_warp_path(c, n)) {
    // a warp per vector (lof_k_vec_warp), L = samples per lane
    LofKParams kp = c->kp;
    const uint32_t mw = c->prm.max_window < n ? c->prm.max_window : n;
    uint32_t n_lev = 0;
    while ((1u << n_lev) <= mw) ++n_lev;
    const unsigned grid = (S + 7) / 8;
    lof_stream_stats* so = d_stats_out ? d_stats_out : inner->d_stats;     // straight into the caller's array
    if (n <= 64) lof_k_vec_warp<2><<<grid, 256, 0, st>>>(d_vec, n, S, kp, n_lev, d_mask, so, fz);
    else if (n <= 256) lof_k_vec_warp<8><<<grid, 256, 0, st>>>(d_vec, n, S, kp, n_lev, d_mask, so, fz);
    else if (n <= 768) lof_k_vec_warp<24><<<grid, 256, 0, st>>>(d_vec, n, S, kp, n_lev, d_mask, so, fz);
    else lof_k_vec_warp<32><<<grid, 256, 0, st>>>(d_vec, n, S, kp, n_lev, d_mask, so, fz);
    c->launches += 1;
    LOF_CUDA(cudaGetLastError());
    return LOF_OK;
  }
  if (n <= LOF_VEC_MAX) {
    const uint32_t Mpad = (n + 31) & ~31u;
    uint32_t npad = 32;
    while (npad < n) npad <<= 1;
    const size_t smem = (size_t)Mpad * LOF_GEN_BYTES_PER_ELEM + 32 + (size_t)npad * 4;
    LOF_CUDA(cudaFuncSetAttribute(lof_k_vec_flag, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    LofKParams kp = c->kp;
    const uint32_t mw = c->prm.max_window < n ? c->prm.max_window : n;
    uint32_t n_lev = 0;
    while ((1u << n_lev) <= mw) ++n_lev;
    lof_k_vec_flag<<<S, LOF_GEN_THREADS, smem, st>>>(d_vec, n, kp, n_lev, d_mask, inner->d_stats);
    c->launches += 1;
    LOF_CUDA(cudaGetLastError());
    if (d_stats_out)
      LOF_CUDA(cudaMemcpyAsync(d_stats_out, inner->d_stats, (size_t)S * sizeof(lof_stream_stats), cudaMemcpyDeviceToDevice, st));
    return LOF_OK;
  }
  const uint64_t l0 = inner->launches;
  const int rc = lof_flag_block(inner, d_vec, d_mask, d_stats_out, st);
  c->launches += inner->launches - l0;
  return rc;
}

extern "C" int lof_flag_block_integrated(lof_ctx* c, const float* d_power, uint32_t* d_flags,
                                         lof_stream_stats* d_stats_freq, lof_stream_stats* d_stats_time,
                                         void* cuda_stream) {
  if (!c || !d_power || !d_flags) return LOF_E_NULL;
  if (((uintptr_t)d_power & 15) || ((uintptr_t)d_flags & 15) || ((uintptr_t)d_stats_freq & 7) ||
      ((uintptr_t)d_stats_time & 7)) return LOF_E_ALIGN;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LOF_CUDA(cudaSetDevice(c->prm.device));
  int rc = integrated_prepare(c);
  if (rc) return rc;
  const uint32_t S = c->prm.n_streams, C = c->prm.n_channels, T = c->prm.n_time, W = c->kp.W;
  const uint32_t CW = (C + 31) / 32;
  // one read of the block: sums over time per channel, sums over all channels per time sample
  lof_k_integ_sums<<<dim3(c->ig_tiles, S), LOF_IG_THREADS, 0, st>>>(d_power, c->d_ig_rowpart, c->d_ig_colsum, C, T,
                                                                    c->ig_tiles);
  const uint64_t rows = (uint64_t)S * C;
  c->launches += 1;
  // the spectrum a[s][c]: formed inside the spectrum run's kernel when that is the warp-per-vector one
  const bool fuse_f = (c->prm.directions & LOF_DIR_FREQ) && integrated_warp_path(c, C);
  const bool fuse_t = (c->prm.directions & LOF_DIR_TIME) && integrated_warp_path(c, T);
  if (!fuse_f) {
    lof_k_integ_spectrum<<<(unsigned)((rows + 255) / 256), 256, 0, st>>>(c->d_ig_rowpart, c->d_ig_spec, rows, c->ig_tiles, T);
    c->launches += 1;
  }
  // frequency first: one SumThreshold run over the time-integrated spectrum of every stream
  if (c->prm.directions & LOF_DIR_FREQ) {
    LofVecFuse fz{};
    if (fuse_f) { fz.rowpart = c->d_ig_rowpart; fz.n_tiles = c->ig_tiles; fz.T = T; fz.spec_out = c->d_ig_spec; }
    rc = integrated_run(c, c->ig_freq, c->d_ig_spec, C, c->d_ig_cmask, d_stats_freq, st, fz);
    if (rc) return rc;
  } else {
    LOF_CUDA(cudaMemsetAsync(c->d_ig_cmask, 0, (size_t)S * CW * 4, st));
    if (d_stats_freq) LOF_CUDA(cudaMemsetAsync(d_stats_freq, 0, (size_t)S * sizeof(lof_stream_stats), st));
  }
  // then time: the series integrated over the channels that are left
  if (!fuse_t) {
    lof_k_integ_series<<<dim3((T + 256 * LOF_IG_SER - 1) / (256 * LOF_IG_SER), S), 256, 0, st>>>(d_power, c->d_ig_colsum, c->d_ig_cmask,
                                                                  c->d_ig_series, C, T);
    c->launches += 1;
  }
  if (c->prm.directions & LOF_DIR_TIME) {
    LofVecFuse fz{};
    if (fuse_t) {                                          // the series run forms the series and writes the block's flags
      fz.cmask = c->d_ig_cmask; fz.flags = d_flags; fz.C = C;
      fz.block = d_power; fz.colsum = c->d_ig_colsum; fz.series_out = c->d_ig_series;
    }
    rc = integrated_run(c, c->ig_time, c->d_ig_series, T, c->d_ig_tmask, d_stats_time, st, fz);
    if (rc) return rc;
  } else {
    LOF_CUDA(cudaMemsetAsync(c->d_ig_tmask, 0, (size_t)S * W * 4, st));
    if (d_stats_time) LOF_CUDA(cudaMemsetAsync(d_stats_time, 0, (size_t)S * sizeof(lof_stream_stats), st));
  }
  if (!fuse_t) {
    lof_k_integ_combine<<<S, 256, 0, st>>>(c->d_ig_cmask, c->d_ig_tmask, d_flags, C, W, T);
    c->launches += 1;
  }
  LOF_CUDA(cudaGetLastError());
  c->block_pending = false;                               // no row sums of this block: the history flagger needs lof_flag_block
  return LOF_OK;
}

extern "C" int lof_integrated_vectors(lof_ctx* c, float* d_spectrum, float* d_series, void* cuda_stream) {
  if (!c) return LOF_E_NULL;
  if (!c->d_ig_colsum) return LOF_E_STATE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LOF_CUDA(cudaSetDevice(c->prm.device));
  const size_t S = c->prm.n_streams;
  if (d_spectrum) LOF_CUDA(cudaMemcpyAsync(d_spectrum, c->d_ig_spec, S * c->prm.n_channels * 4, cudaMemcpyDeviceToDevice, st));
  if (d_series) LOF_CUDA(cudaMemcpyAsync(d_series, c->d_ig_series, S * c->prm.n_time * 4, cudaMemcpyDeviceToDevice, st));
  return LOF_OK;
}

extern "C" int lof_history_update(lof_ctx* c, uint32_t* d_flags, uint8_t* d_row_flagged, void* cuda_stream) {
  if (!c || !d_flags) return LOF_E_NULL;
  if ((uintptr_t)d_flags & 15) return LOF_E_ALIGN;
  if (!c->block_pending || c->prm.history_length == 0) return LOF_E_STATE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LOF_CUDA(cudaSetDevice(c->prm.device));
  const uint64_t rows = (uint64_t)c->prm.n_streams * c->prm.n_channels;
  const double sens = c->prm.history_sensitivity > 0.f ? (double)c->prm.history_sensitivity
                                                       : (double)c->prm.sensitivity;
  lof_k_history_decide<<<(unsigned)((rows + 127) / 128), 128, 0, st>>>(
      c->d_ring, c->d_head, c->d_count, c->d_rowsum, c->d_rowcnt, c->d_row_flagged, rows,
      c->prm.history_length, c->prm.history_min_fill, sens);
  lof_k_history_fill<<<(unsigned)((rows * 32 + 255) / 256), 256, 0, st>>>(c->d_row_flagged, d_flags, rows,
                                                                         c->kp.W, c->prm.n_time);
  c->launches += 2;
  LOF_CUDA(cudaGetLastError());
  if (d_row_flagged)
    LOF_CUDA(cudaMemcpyAsync(d_row_flagged, c->d_row_flagged, rows, cudaMemcpyDeviceToDevice, st));
  c->block_pending = false;
  return LOF_OK;
}

extern "C" int lof_reset(lof_ctx* c, void* cuda_stream) {
  if (!c) return LOF_E_NULL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LOF_CUDA(cudaSetDevice(c->prm.device));
  const size_t rows = (size_t)c->prm.n_streams * c->prm.n_channels;
  LOF_CUDA(cudaMemsetAsync(c->d_ring, 0, rows * c->prm.history_length * sizeof(float) + (c->prm.history_length ? 0 : 4), st));
  LOF_CUDA(cudaMemsetAsync(c->d_head, 0, rows * 4, st));
  LOF_CUDA(cudaMemsetAsync(c->d_count, 0, rows * 4, st));
  c->block_pending = false;
  return LOF_OK;
}

extern "C" int lof_row_sums(lof_ctx* c, double* d_rowsum, uint32_t* d_rowcnt, void* cuda_stream) {
  if (!c) return LOF_E_NULL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LOF_CUDA(cudaSetDevice(c->prm.device));
  const size_t rows = (size_t)c->prm.n_streams * c->prm.n_channels;
  if (d_rowsum) LOF_CUDA(cudaMemcpyAsync(d_rowsum, c->d_rowsum, rows * 8, cudaMemcpyDeviceToDevice, st));
  if (d_rowcnt) LOF_CUDA(cudaMemcpyAsync(d_rowcnt, c->d_rowcnt, rows * 4, cudaMemcpyDeviceToDevice, st));
  return LOF_OK;
}

extern "C" int lof_history_export(lof_ctx* c, float* d_ring, uint32_t* d_head, uint32_t* d_count, void* cuda_stream) {
  if (!c) return LOF_E_NULL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LOF_CUDA(cudaSetDevice(c->prm.device));
  const size_t rows = (size_t)c->prm.n_streams * c->prm.n_channels;
  if (d_ring && c->prm.history_length)
    LOF_CUDA(cudaMemcpyAsync(d_ring, c->d_ring, rows * c->prm.history_length * 4, cudaMemcpyDeviceToDevice, st));
  if (d_head) LOF_CUDA(cudaMemcpyAsync(d_head, c->d_head, rows * 4, cudaMemcpyDeviceToDevice, st));
  if (d_count) LOF_CUDA(cudaMemcpyAsync(d_count, c->d_count, rows * 4, cudaMemcpyDeviceToDevice, st));
  return LOF_OK;
}

extern "C" int lof_flag_block_host(lof_ctx* c, const void* h_input, int is_ci16, uint32_t* h_flags,
                                   lof_stream_stats* h_stats) {
  if (!c || !h_input || !h_flags) return LOF_E_NULL;
  LOF_CUDA(cudaSetDevice(c->prm.device));
  const size_t n = (size_t)c->prm.n_streams * c->prm.n_channels * c->prm.n_time;
  const size_t in_bytes = n * 4;                        // float32, or 2 x int16
  const size_t fl_bytes = (size_t)c->prm.n_streams * c->prm.n_channels * c->kp.W * 4;
  if (!c->host_stream) LOF_CUDA(cudaStreamCreateWithFlags(&c->host_stream, cudaStreamNonBlocking));
  if (!c->d_in_stage) {
    LOF_CUDA(cudaMalloc(&c->d_in_stage, in_bytes));
    LOF_CUDA(cudaMalloc(reinterpret_cast<void**>(&c->d_flags_stage), fl_bytes));
    c->in_stage_bytes = in_bytes;
  }
  cudaStream_t st = c->host_stream;
  LOF_CUDA(cudaMemcpyAsync(c->d_in_stage, h_input, in_bytes, cudaMemcpyHostToDevice, st));
  int rc = is_ci16 ? lof_flag_block_ci16(c, (const int16_t*)c->d_in_stage, c->d_flags_stage, nullptr, st)
                   : lof_flag_block(c, (const float*)c->d_in_stage, c->d_flags_stage, nullptr, st);
  if (rc) return rc;
  LOF_CUDA(cudaMemcpyAsync(h_flags, c->d_flags_stage, fl_bytes, cudaMemcpyDeviceToHost, st));
  if (h_stats)
    LOF_CUDA(cudaMemcpyAsync(h_stats, c->d_stats, (size_t)c->prm.n_streams * sizeof(lof_stream_stats),
                             cudaMemcpyDeviceToHost, st));
  LOF_CUDA(cudaStreamSynchronize(st));
  return LOF_OK;
}

extern "C" uint64_t lof_launch_count(const lof_ctx* c) { return c ? c->launches : 0; }

extern "C" int lof_fused_counters(lof_ctx* c, uint64_t* h_out, int reset) {
  if (!c || !h_out) return LOF_E_NULL;
  LOF_CUDA(cudaSetDevice(c->prm.device));
  LOF_CUDA(cudaDeviceSynchronize());
  unsigned long long v[LOF_DIAG_WORDS];
  LOF_CUDA(cudaMemcpy(v, c->d_diag, sizeof v, cudaMemcpyDeviceToHost));
  for (int i = 0; i < 4; ++i) h_out[i] = v[i];
  if (reset) {
    LOF_CUDA(cudaMemset(c->d_diag, 0, sizeof v));
#ifdef LOF_FUSED_PROF
    const unsigned long long z[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    LOF_CUDA(cudaMemcpyToSymbol(lof_fused_cycles_dev, z, sizeof z));
#endif
  }
  return LOF_OK;
}

extern "C" int lof_fused_cycles(lof_ctx* c, uint64_t* h_out) {
  if (!c || !h_out) return LOF_E_NULL;
  LOF_CUDA(cudaSetDevice(c->prm.device));
  LOF_CUDA(cudaDeviceSynchronize());
  for (int i = 0; i < 8; ++i) h_out[i] = 0;
#ifdef LOF_FUSED_PROF
  unsigned long long v[8];
  LOF_CUDA(cudaMemcpyFromSymbol(v, lof_fused_cycles_dev, sizeof v));
  for (int i = 0; i < 8; ++i) h_out[i] = v[i];
#endif
  return LOF_OK;
}

extern "C" int lof_set_path(lof_ctx* c, int path) {
  if (!c) return LOF_E_NULL;
  if (path < 0 || path > 1) return LOF_E_PARAM;
  c->path = path;
  return LOF_OK;
}

extern "C" int lof_path_used(const lof_ctx* c) { return c ? c->path_used : LOF_E_NULL; }

extern "C" int lof_set_group(lof_ctx* c, uint32_t max_streams) {
  if (!c) return LOF_E_NULL;
  if (max_streams == 0) return LOF_E_PARAM;
  c->group = max_streams < c->group_alloc ? max_streams : c->group_alloc;
  return LOF_OK;
}

// ---- lof_sir_noalloc: the SIR operator on a packed mask with no context and no allocation (include/lof.h).
// The intermediate mask (the frequency pass's output, input of the time pass) lives in a file-scope device array
// instead of a context's cudaMalloc'ed buffer: every GPU that loads this library holds LOF_NOALLOC_MAX_WORDS * 4
// bytes (8 MiB) for it until the process exits.  Every call on a device shares the array; both kernels write every
// word they later read, so nothing has to start at zero and the previous call's contents do not matter — but two
// calls whose kernels overlap on one GPU (different streams, or threads) race on it.
// `lof_noalloc_scratch` below is, in host code, a host-side stand-in for the symbol and NOT a device address: the
// device address is looked up once per device with cudaGetSymbolAddress, that device current, and kept.
static __device__ __align__(256) uint32_t lof_noalloc_scratch[LOF_NOALLOC_MAX_WORDS];

#define LOF_NOALLOC_MAX_DEVICES 64
static std::mutex g_noalloc_mu;
static uint32_t* g_noalloc_ptr[LOF_NOALLOC_MAX_DEVICES];   // device address of the array, per device (0: not looked up)

// device must be current
static int noalloc_scratch(int device, uint32_t** out) {
  std::lock_guard<std::mutex> lk(g_noalloc_mu);
  if (!g_noalloc_ptr[device]) {
    uint32_t* p = nullptr;
    LOF_CUDA(cudaGetSymbolAddress((void**)&p, lof_noalloc_scratch));
    if (!p) { snprintf(g_cuda_err, sizeof g_cuda_err, "cudaGetSymbolAddress gave a null address"); return LOF_E_CUDA; }
    g_noalloc_ptr[device] = p;
  }
  *out = g_noalloc_ptr[device];
  return LOF_OK;
}

template <int G>
static void noalloc_sir_time(const uint32_t* in, uint32_t* out, lof_stream_stats* d_stats, uint64_t rows, uint32_t C,
                             uint32_t W, uint32_t T, float eta, cudaStream_t st) {
  const unsigned grid = (unsigned)((rows * G + 255) / 256);
  const size_t stage = (size_t)2 * (256 / G) * W * 4;
  const uint32_t m_min = sir_min_run(eta, T);
  if (stage <= 40 * 1024) lof_k_sir_time<G, true><<<grid, 256, stage, st>>>(in, out, d_stats, rows, C, W, T, eta, m_min);
  else lof_k_sir_time<G, false><<<grid, 256, 0, st>>>(in, out, d_stats, rows, C, W, T, eta, m_min);
}

extern "C" int lof_sir_noalloc(uint32_t* d_flags, lof_stream_stats* d_stats, uint32_t n_streams, uint32_t n_channels,
                               uint32_t n_time, float eta, uint32_t directions, int device, void* cuda_stream) {
  if (!d_flags || !d_stats) return LOF_E_NULL;
  if (((uintptr_t)d_flags & 15) || ((uintptr_t)d_stats & 7)) return LOF_E_ALIGN;
  if (n_streams == 0 || n_channels == 0 || n_time == 0 || n_channels > 256) return LOF_E_PARAM;
  if (!(eta >= 0.f && eta <= 1.f)) return LOF_E_PARAM;                  // also rejects NaN
  if (directions == 0 || (directions & ~(uint32_t)(LOF_DIR_FREQ | LOF_DIR_TIME))) return LOF_E_PARAM;
  if (device < 0 || device >= LOF_NOALLOC_MAX_DEVICES) return LOF_E_PARAM;
  const uint32_t S = n_streams, C = n_channels, T = n_time, W = (T + 31) / 32;
  const uint64_t words = (uint64_t)S * C * W;
  if (words > (uint64_t)LOF_NOALLOC_MAX_WORDS) return LOF_E_SIZE;
  if (!(eta > 0.f)) return LOF_OK;                                      // the operator is the identity
  cudaStream_t st = (cudaStream_t)cuda_stream;
  LOF_CUDA(cudaSetDevice(device));
  uint32_t* scratch = nullptr;
  const int rc = noalloc_scratch(device, &scratch);
  if (rc) return rc;
  uint32_t* cur = d_flags;
  uint32_t* other = scratch;
  if (directions & LOF_DIR_FREQ) {
    const uint32_t m_min = sir_min_run(eta, C);          // shortest run that grows at all
    const uint64_t n_cols = (uint64_t)S * W;
    const dim3 g8(S, (W + 7) / 8);                             // a warp per word column, 8 per CTA
    if (C == 64) lof_k_sir_freq_reg<64><<<g8, 256, 0, st>>>(cur, other, d_stats, W, eta, m_min);
    else if (C == 32) lof_k_sir_freq_reg<32><<<g8, 256, 0, st>>>(cur, other, d_stats, W, eta, m_min);
    else if (C == 16) lof_k_sir_freq_reg<16><<<g8, 256, 0, st>>>(cur, other, d_stats, W, eta, m_min);
    else lof_k_sir_freq<<<(unsigned)((n_cols + 255) / 256), 256, 0, st>>>(cur, other, d_stats, n_cols, C, W, eta, m_min);
    uint32_t* t = cur; cur = other; other = t;
  }
  if (directions & LOF_DIR_TIME) {
    const uint64_t rows = (uint64_t)S * C;
    uint32_t G = 1;
    while (G < 32 && G * 8 < W) G <<= 1;                  // about eight words per lane
    switch (G) {
      case 1: noalloc_sir_time<1>(cur, other, d_stats, rows, C, W, T, eta, st); break;
      case 2: noalloc_sir_time<2>(cur, other, d_stats, rows, C, W, T, eta, st); break;
      case 4: noalloc_sir_time<4>(cur, other, d_stats, rows, C, W, T, eta, st); break;
      case 8: noalloc_sir_time<8>(cur, other, d_stats, rows, C, W, T, eta, st); break;
      case 16: noalloc_sir_time<16>(cur, other, d_stats, rows, C, W, T, eta, st); break;
      default: noalloc_sir_time<32>(cur, other, d_stats, rows, C, W, T, eta, st); break;
    }
    uint32_t* t = cur; cur = other; other = t;
  }
  LOF_CUDA(cudaGetLastError());
  if (cur != d_flags) LOF_CUDA(cudaMemcpyAsync(d_flags, cur, words * 4, cudaMemcpyDeviceToDevice, st));
  return LOF_OK;
}
