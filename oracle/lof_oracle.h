/* lof_oracle.h — ORACLE (test infrastructure, not the product).
 *
 * A plain, slow, single-threaded C++ restatement of the LOFAR Online Flagger hot path of
 * arXiv 1701.08197: per-stream statistics, SumThreshold along frequency then
 * time, bit-packing + row sums, and the history flagger.  Written from the paper; shares no
 * code with the CUDA path (paper_1701_08197_b200/csrc).  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * All pointers are HOST pointers.  All arithmetic is fp64 unless stated.
 * Readings of the paper (F1..F10, S1..S6, H1'..H7') are listed in DESIGN.md §3.
 *
 * Parity pins (tests/test_oracle_pins.py): factor table, hand vectors
 * V1-V6, brute force vs fast window sums, std::sort median, closed-form noise statistics,
 * invariants.  UNPINNED against the authors' code (not available): readings F7, F8, F10,
 * S1-S4, H3'-H6' — "parity unpinned" beyond the reasoning in DESIGN.md.
 */
#ifndef LOF_ORACLE_H
#define LOF_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  uint32_t n_streams, n_channels, n_time;
  double   p;                   /* PAPER.md:43, default 1.5 */
  double   sensitivity;         /* PAPER.md:43, default 1.0 */
  double   start_threshold;     /* 6.0 ("6 sigma") */
  uint32_t max_window;          /* power of two */
  uint32_t directions;          /* 1 = frequency, 2 = time, 3 = both (frequency first) */
  uint32_t history_length;      /* H */
  uint32_t history_min_fill;
  double   history_sensitivity; /* <= 0: use sensitivity */
  double   sir_eta;             /* SIR operator: every run of flagged samples is extended by
                                   floor(sir_eta * length) samples before and after; 0 = off; typical 0.2 */
  uint32_t stats_mode;          /* 0: stddev as PAPER.md:41 is written; 1: 1.4826 * MAD in its place (PAPER.md:120
                                   lists the MAD among the statistics used; reading R1) */
} lofo_params;

typedef struct {
  float    median;
  uint32_t n_nonfinite;
  double   mean, stddev;
  uint64_t n_flagged;
} lofo_stream_stats;

/* factor_I = start * p^(log2 I) / I = start * (p/2)^k for I = 2^k, k = 0..n_out-1. */
void lofo_factor_table(double start_threshold, double p, uint32_t n_out, double* out);

/* threshold_I = median + stddev * factor_I * sensitivity. */
void lofo_threshold_table(double median, double stddev, double start_threshold, double p,
                          double sensitivity, uint32_t n_out, double* out);

/* O1-O3: mean (index order), population stddev (two-pass), median = rank floor(N/2) element. */
void lofo_statistics(const float* x, uint64_t n, lofo_stream_stats* out);

/* Median absolute deviation: the rank floor(N/2) element of d_i = (float)|x_i - median|, the
 * difference taken exactly and rounded once to float32 (which is what a float32 subtraction does). */
float lofo_mad(const float* x, uint64_t n, float median);

/* One SumThreshold run along one line of n samples x[i*stride]; mask[i*mask_stride] is
 * uint8 0/1, updated in place.  thresholds[k] is T_I for I = 2^k; levels k = 0..n_levels-1
 * with I <= n are run in order, flags frozen at the start of each iteration.
 * margin (may be NULL): margin[i*mask_stride] set to 1 for samples covered by a window with
 * |S - I*T_I| <= margin_rel * |I*T_I|.
 * _literal: the double loop of PAPER.md:37-47 exactly as written (O(n*I) per iteration).
 * _fast:    same sums from an fp64 prefix array (O(n) per iteration).                    */
void lofo_sumthreshold_1d_literal(const float* x, uint64_t n, int64_t stride, uint8_t* mask,
                                  int64_t mask_stride, const double* thresholds,
                                  uint32_t n_levels, uint8_t* margin, double margin_rel);
void lofo_sumthreshold_1d_fast(const float* x, uint64_t n, int64_t stride, uint8_t* mask,
                               int64_t mask_stride, const double* thresholds,
                               uint32_t n_levels, uint8_t* margin, double margin_rel);

/* Whole block: power[S][C][T] -> flags uint32[S][C][ceil(T/32)] (LSB first, padding 0),
 * stats[S], rowsum[S][C] (fp64 sum of unflagged samples), rowcnt[S][C], and optionally
 * mask_freq uint8[S][C][T] (mask after the frequency run) and margin uint8[S][C][T].
 * use_literal != 0 selects the literal window sums.  Any of the optional outputs may be NULL. */
int lofo_flag_block(const lofo_params* prm, const float* power, uint32_t* flags,
                    lofo_stream_stats* stats, double* rowsum, uint32_t* rowcnt,
                    uint8_t* mask_freq, uint8_t* margin, double margin_rel, int use_literal);

/* Scale-invariant rank operator as PAPER.md:55 states it: "all ranges of consecutive flagged samples are
 * extended by flagging 20% more samples, before and after the original range".  One line of n mask bytes
 * (mask[i*stride], 0/1), in place: every maximal run of flagged samples of the INPUT mask, of length len, gets
 * floor(eta*len) more samples flagged on each side, clipped at the ends of the line; run lengths are those of
 * the input (extensions do not lengthen one another).  Readings SIR-1..4 of DESIGN.md §3. */
void lofo_sir_1d(uint8_t* mask, uint64_t n, int64_t stride, double eta);

/* The operator on a packed block mask flags[S][C][ceil(T/32)] in place: along frequency (channels of one time
 * sample), then along time on the result, for the directions set in `directions` (reading SIR-5). */
void lofo_sir_block(uint32_t* flags, uint64_t S, uint64_t C, uint64_t T, double eta, uint32_t directions);

/* Fully integrated mode (Fig. 4): "integrate the time direction fully for frequency flagging,
 * and ... the frequency direction fully for time domain flagging. We first flag in the frequency direction."
 * Per stream X[C][T] (readings I1-I5):
 *   a[c] = (float)(sum_t X[c][t] / T)                       fp64 sum in index order, rounded once
 *   channel mask = one SumThreshold run over a[0..C), thresholds from the median / stddev of a itself
 *   b[t] = (float)(sum over unflagged channels c of X[c][t] / their number)   (no unflagged channel: b = 0)
 *   time mask    = one SumThreshold run over b[0..T), thresholds from the median / stddev of b itself
 *   sample (c, t) is flagged iff its channel or its time sample is.
 * A vector with a non-finite entry is flagged completely (S6).  Outputs: flags uint32[S][C][ceil(T/32)],
 * spectrum float[S][C] = a, series float[S][T] = b, chan_mask uint8[S][C], time_mask uint8[S][T],
 * stats_freq / stats_time [S] = statistics of a / of b (n_flagged: flagged channels / time samples).  Any output
 * may be NULL.  prm->directions selects the runs (1 = channel run only, 2 = time run only, 3 = both). */
int lofo_flag_block_integrated(const lofo_params* prm, const float* power, uint32_t* flags, float* spectrum,
                               float* series, uint8_t* chan_mask, uint8_t* time_mask,
                               lofo_stream_stats* stats_freq, lofo_stream_stats* stats_time);

/* x = (float)(uint32)(re*re + im*im) for complex int16 volt[n][2] (reading S5). */
void lofo_power_from_ci16(const int16_t* volt, uint64_t n, float* power);

/* History flagger state: rings float32[S][C][H], head/count per ring. */
typedef struct lofo_history lofo_history;
lofo_history* lofo_history_create(const lofo_params* prm);
void lofo_history_destroy(lofo_history*);
void lofo_history_reset(lofo_history*);
/* H1-H6 for every (stream, channel).  flags is updated in place (row -> all ones, padding 0).
 * row_flagged uint8[S][C]; near uint8[S][C] (may be NULL) = 1 where |cur-thr| <= near_rel*|thr|. */
void lofo_history_update(lofo_history*, const double* rowsum, const uint32_t* rowcnt,
                         uint32_t* flags, uint8_t* row_flagged, uint8_t* near, double near_rel);
/* copy out ring state: ring float[S][C][H], head uint32[S][C], count uint32[S][C] */
void lofo_history_export(const lofo_history*, float* ring, uint32_t* head, uint32_t* count);

#ifdef __cplusplus
}
#endif
#endif
