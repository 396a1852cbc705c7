/* lof.h — C-ABI boundary of the B200-native LOFAR Online Flagger (LOF) hot path.
 *
 * Method: arXiv 1701.08197.  Per-stream statistics, SumThreshold
 * with windows I = 1, 2, 4, ... and threshold_I = median + stddev * factor_I * sensitivity,
 * factor_I = startThreshold * p^(log2 I) / I, run along frequency then time
 * (PAPER.md:83, :180), then the history flagger over consecutive blocks.
 * The readings taken where the paper is silent or garbled are listed in DESIGN.md §3.
 *
 * Every step runs in hand-written sm_100a CUDA kernels (paper_1701_08197_b200/csrc).  There is
 * no CPU fallback: a call on a machine without a usable CUDA device returns LOF_E_CUDA.
 *
 * Conventions
 *  - A block is power[n_streams][n_channels][n_time], float32, time fastest.  A stream is one
 *    [n_channels][n_time] slice; statistics, thresholds and flags of a stream depend on that
 *    stream only.
 *  - Pointers named d_* are DEVICE pointers owned by the caller, 16-byte aligned, valid until the
 *    work queued on `cuda_stream` has completed; pointers named h_* are HOST pointers.  The
 *    library never frees or retains caller pointers.
 *  - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device
 *    calls only enqueue work on it and never synchronise the host.
 *  - A context is not thread-safe, and its calls must be ordered on ONE stream at a time: it owns the scratch
 *    (statistics, masks, row sums, history rings) that consecutive calls reuse.  lof_flag_block_host uses a
 *    private stream and returns after synchronising it; do not call it while device calls on the same context
 *    are still in flight on another stream.
 *  - Flag bit of sample t of row (s, c): word (s*n_channels + c)*ceil(n_time/32) + t/32,
 *    bit t%32 (LSB first), 1 = flagged.  Padding bits of a row's last word are 0.
 *  - Return value: 0 on success, a negative LOF_E_* code otherwise; nothing throws or aborts
 *    across this boundary.  lof_strerror() gives a static description; after LOF_E_CUDA,
 *    lof_last_cuda_error() gives the CUDA runtime's text for the calling thread's last failure.
 */
#ifndef LOF_H
#define LOF_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define LOF_OK        0
#define LOF_E_NULL   -1   /* a required pointer is NULL                                         */
#define LOF_E_PARAM  -2   /* bad lof_params (see lof_create)                                    */
#define LOF_E_ALIGN  -3   /* a device pointer is not 16-byte aligned                            */
#define LOF_E_STATE  -4   /* call order violated (see lof_history_update)                       */
#define LOF_E_CUDA   -5   /* a CUDA runtime call failed, or no usable device                    */
#define LOF_E_SIZE   -6   /* problem larger than the static scratch of lof_sir_noalloc          */

#define LOF_DIR_FREQ 1u   /* SumThreshold along channels (run first)               */
#define LOF_DIR_TIME 2u   /* SumThreshold along time                                            */

#define LOF_MAX_LEVELS 11 /* windows 1 .. 1024                                                  */

typedef struct lof_ctx lof_ctx;   /* opaque; owns all scratch memory and the history rings */

typedef struct {
  uint32_t struct_size;         /* = sizeof(lof_params); anything else -> LOF_E_PARAM            */
  int32_t  device;              /* CUDA device ordinal                                           */
  uint32_t n_streams;           /* S > 0, fixed for the context                                  */
  uint32_t n_channels;          /* C > 0 (<= 256)                                                */
  uint32_t n_time;              /* T > 0                                                         */
  float    p;                   /* > 0; paper default 1.5                          */
  float    sensitivity;         /* > 0; paper default 1.0                          */
  float    start_threshold;     /* > 0; 6.0 = "6 sigma" at I = 1                   */
  uint32_t max_window;          /* power of two in 1..1024; "7-10 iterations"      */
  uint32_t directions;          /* LOF_DIR_FREQ | LOF_DIR_TIME, non-zero; freq always runs first */
  uint32_t history_length;      /* H entries per (stream, channel) ring; 0 disables the history
                                   flagger; the paper's example is 300            */
  uint32_t history_min_fill;    /* below this many entries a ring only records (H3')   */
  float    history_sensitivity; /* <= 0: use `sensitivity`, the literal text of PAPER.md:106     */
  float    sir_eta;             /* scale-invariant rank operator: every run of flagged
                                   samples grows by floor(sir_eta * length) samples on each side, along
                                   frequency and then along time (the directions set in `directions`);
                                   0 = off, the paper's typical value is 0.2; in [0, 1]               */
  uint32_t stats_mode;          /* LOF_STATS_PLAIN (0): stddev of all samples, as PAPER.md:41 is written;
                                   LOF_STATS_MAD (1): 1.4826 * median absolute deviation in its place,
                                   one of the robust statistics PAPER.md:120 lists (R1)     */
} lof_params;

#define LOF_STATS_PLAIN 0u
#define LOF_STATS_MAD   1u

/* Per-stream results of lof_flag_block (32 bytes, no padding surprises: 4+4+8+8+8). */
typedef struct {
  float    median;       /* element of rank floor(N/2) of the stream's N = C*T samples (bit-exact) */
  uint32_t n_nonfinite;  /* NaN/Inf samples; if > 0 the whole stream is flagged and the other
                            fields except n_flagged are unspecified (S6)                 */
  double   mean;         /* of all N samples, before any flagging (S1)      */
  double   stddev;       /* population standard deviation about the mean                           */
  uint64_t n_flagged;    /* flagged samples of the stream after the SumThreshold runs              */
} lof_stream_stats;

/* Validate params (LOF_E_PARAM when: struct_size mismatch; S, C or T zero; C > 256; max_window
 * zero, not a power of two or > 1024; directions zero or with unknown bits; p, sensitivity or
 * start_threshold not > 0 and finite; history_length > 0 with history_min_fill == 0 — an empty ring has no
 * mean; history_sensitivity not finite; sir_eta not in [0, 1]; stats_mode unknown), select the device, allocate scratch and history rings
 * (zero-filled, all rings empty).  *out receives the handle; on failure *out = NULL. */
int lof_create(const lof_params* params, lof_ctx** out);

/* Frees everything the context owns.  Synchronises the device first.  NULL is accepted. */
int lof_destroy(lof_ctx* ctx);

/* One pass of the hot path over one block:
 *   statistics -> thresholds -> SumThreshold(frequency) -> SumThreshold(time) -> bit-pack,
 *   per-row sums of unflagged samples (kept inside the context for lof_history_update),
 *   then, if sir_eta > 0, the SIR operator on the packed mask (it works on the mask only,
 *   the row sums are those of the SumThreshold mask; n_flagged counts the final mask).
 * d_power [S][C][T] float32 (in), d_flags [S][C][ceil(T/32)] uint32 (out, fully overwritten),
 * d_stats [S] (out, may be NULL).  Asynchronous on cuda_stream. */
int lof_flag_block(lof_ctx* ctx, const float* d_power, uint32_t* d_flags,
                   lof_stream_stats* d_stats, void* cuda_stream);

/* Same, for raw complex voltages ("we may have to compute amplitudes first"):
 * d_volt [S][C][T][2] int16 (re, im); the power x = (float)(uint32)(re*re + im*im) is formed in
 * registers on load and never written to memory (S5). */
int lof_flag_block_ci16(lof_ctx* ctx, const int16_t* d_volt, uint32_t* d_flags,
                        lof_stream_stats* d_stats, void* cuda_stream);

/* Fully integrated mode (Fig. 4: "integrate the time direction fully for frequency flagging, and
 * ... the frequency direction fully for time domain flagging. We first flag in the frequency direction."), per stream:
 *   a[c] = mean over time of power[c][t]; one SumThreshold run over a (windows <= min(max_window, C)), thresholds
 *          from the median and stddev of a itself -> flagged channels;
 *   b[t] = mean over the UNFLAGGED channels of power[c][t] (0 if none is left); one run over b -> flagged times;
 *   sample (c, t) is flagged iff its channel or its time sample is (readings I1-I5).
 * `directions` selects the runs.  d_power [S][C][T] float32 (read once, plus the rows of flagged channels a
 * second time), d_flags [S][C][ceil(T/32)] (out, fully overwritten), d_stats_freq / d_stats_time [S] (out, may be
 * NULL): statistics of a / of b, n_flagged = number of flagged channels / time samples.  It leaves no row sums:
 * lof_history_update after it returns LOF_E_STATE.  The first call allocates this mode's scratch (S*T*12 bytes
 * and two inner contexts).  Asynchronous on cuda_stream. */
int lof_flag_block_integrated(lof_ctx* ctx, const float* d_power, uint32_t* d_flags,
                              lof_stream_stats* d_stats_freq, lof_stream_stats* d_stats_time, void* cuda_stream);

/* Copies the vectors of the last lof_flag_block_integrated to caller DEVICE buffers (either may be NULL):
 * spectrum [S][C] float32 = a, series [S][T] float32 = b.  LOF_E_STATE before the first integrated block. */
int lof_integrated_vectors(lof_ctx* ctx, float* d_spectrum, float* d_series, void* cuda_stream);

/* History flagger (PAPER.md:97-113 pseudocode), one ring per (stream, channel):
 *   cur = mean of the row's unflagged samples of the block just flagged;
 *   thr = mean(ring) + history_sensitivity * stddev(ring);
 *   cur < thr: push cur; else push thr and flag the whole row in d_flags.
 * d_flags (in/out) must be the flags lof_flag_block wrote for that block; d_row_flagged [S][C]
 * uint8 (out, may be NULL) is 1 for rows flagged here (or left without any unflagged sample).
 * LOF_E_STATE if no lof_flag_block call precedes it or it was already called for that block,
 * or if history_length == 0.  Asynchronous on cuda_stream. */
int lof_history_update(lof_ctx* ctx, uint32_t* d_flags, uint8_t* d_row_flagged, void* cuda_stream);

/* Empties every history ring and forgets a pending block.  Takes a stream (unlike the survey's sketch
 * lof_reset(ctx)) because, like every device call here, it only enqueues work (memsets) on cuda_stream. */
int lof_reset(lof_ctx* ctx, void* cuda_stream);

/* Copies to caller DEVICE buffers (either may be NULL) what the last lof_flag_block left in the
 * context for the history flagger: rowsum [S][C] double = sum of unflagged samples per row,
 * rowcnt [S][C] uint32 = their number (what PAPER.md:102 "meanOfUnflaggedSamples" is formed
 * from).  Asynchronous on cuda_stream. */
int lof_row_sums(lof_ctx* ctx, double* d_rowsum, uint32_t* d_rowcnt, void* cuda_stream);

/* Copies the history state to caller DEVICE buffers (any may be NULL): ring [S][C][H] float32,
 * head [S][C] uint32 (next write position), count [S][C] uint32.  Asynchronous. */
int lof_history_export(lof_ctx* ctx, float* d_ring, uint32_t* d_head, uint32_t* d_count,
                       void* cuda_stream);

/* End-to-end convenience with HOST buffers: copies h_power (or h_volt when is_ci16 != 0) to a
 * context-owned device buffer, runs lof_flag_block[_ci16], copies flags and stats back and
 * synchronises.  h_stats may be NULL.  Pinned host memory makes the copies asynchronous to
 * each other; pageable memory works too. */
int lof_flag_block_host(lof_ctx* ctx, const void* h_input, int is_ci16, uint32_t* h_flags,
                        lof_stream_stats* h_stats);

/* Host only: factor_I = start_threshold * (p/2)^k for I = 2^k, k = 0..n_out-1. */
int lof_factor_table(const lof_params* params, double* h_out, uint32_t n_out);

/* Number of kernel launches the library has enqueued for this context so far (bench.py's
 * gpu_launches is the difference over the timed region). */
uint64_t lof_launch_count(const lof_ctx* ctx);

/* Selects the kernel path: 0 = automatic (fused kernels where the shape allows), 1 = force the
 * generic multi-kernel path.  Both compute the same results; for tests and profiling. */
int lof_set_path(lof_ctx* ctx, int path);

/* Which kernels the last lof_flag_block[_ci16] of this context ran (the steps of PAPER.md:37-47, :83 are the
 * same on every path; only the decomposition differs):
 *   LOF_PATH_FUSED         one kernel per block: (n_channels, n_time) in {(64,768), (32,768), (16,768), (16,256),
 *                          (32,1024), (64,512), (16,1024)}, max_window <= 64, float32 input, stats_mode PLAIN — a stream fits one
 *                          SM's shared memory (n_time is a template parameter of that kernel: 32 x the samples a
 *                          lane holds; other shapes take the paths below, with the same results);
 *   LOF_PATH_LONGROW_SEG   statistics kernels + register-resident column kernel + independent row segments
 *                          (16/32/64 channels, dependency cone of the time run <= 256 samples);
 *   LOF_PATH_LONGROW_COOP  same with cooperative 8192-sample row tiles (wider cones, max_window <= 512);
 *   LOF_PATH_GENERIC       at least one step ran in the shared-memory generic kernels (any shape, several times
 *                          slower: other channel counts, max_window 1024 on long rows, or lof_set_path(ctx, 1)).
 * LOF_PATH_NONE before the first block; LOF_E_NULL for a NULL context. */
#define LOF_PATH_NONE          0
#define LOF_PATH_FUSED         1
#define LOF_PATH_LONGROW_SEG   2
#define LOF_PATH_LONGROW_COOP  3
#define LOF_PATH_GENERIC       4
int lof_path_used(const lof_ctx* ctx);

/* Tests only: lowers the number of streams the multi-kernel paths process per launch sequence (the default is
 * as many as fit 640 MB of input, at most 1024; values above that are clamped to it), so that a small block
 * exercises the loop over several groups.  LOF_E_PARAM for 0.  Results do not depend on it. */
int lof_set_group(lof_ctx* ctx, uint32_t max_streams_per_group);

/* Diagnostics of the fused kernels (streams that fit one SM's shared memory): how the exact median
 * of each stream of THIS context was found since the last reset: h_out[0] from samples gathered during the statistics pass (the fast case),
 * h_out[1] by one more gather pass, h_out[2] by a radix select over the whole stream, h_out[3]
 * streams with non-finite samples.  Synchronises the device.  reset != 0 zeroes the counters. */
int lof_fused_counters(lof_ctx* ctx, uint64_t* h_out /*[4]*/, int reset);

/* Profiling builds only (nvcc -DLOF_FUSED_PROF, see build.py LOF_NVCC_EXTRA): SM cycles thread 0 of
 * every CTA spent per phase of the fused kernel since the last lof_fused_counters(reset): h_out[0]
 * first load + statistics, [1] frequency pass, [2] plan of the next stream, [3] time pass with
 * the next stream's row statistics, [4] end of the next stream's statistics, [5..7] zero.
 * All zero in a normal build.  Synchronises the device. */
int lof_fused_cycles(lof_ctx* ctx, uint64_t* h_out /*[8]*/);

/* The SIR operator of PAPER.md:49-57 (readings SIR-1..6; the same kernels as lof_flag_block with
 * sir_eta > 0) applied IN PLACE to a packed mask, for callers that cannot allocate device memory (CUDA graph
 * capture, serving loops, harnesses that forbid cudaMalloc): no context, and no cudaMalloc / cudaFree / allocating
 * library call on any path.  Every run of set bits grows by floor(eta * length) on each side, along channels if
 * directions has LOF_DIR_FREQ, then along time if it has LOF_DIR_TIME.
 *   d_flags  device, in/out, uint32 [n_streams][n_channels][W], W = ceil(n_time / 32), bit t%32 of word t/32,
 *            16-byte aligned, owned by the caller; bits beyond n_time must be zero and stay zero.
 *   d_stats  device, in/out, lof_stream_stats [n_streams], 8-byte aligned: n_flagged of each stream grows by the
 *            number of bits the operator set in it; the other fields are not touched.
 *   device   CUDA device ordinal of both pointers (0..63); made current.   cuda_stream: the stream to enqueue on.
 * The intermediate mask lives in a static device array of LOF_NOALLOC_MAX_WORDS words (8 MiB per GPU that loads
 * the library, held until the process exits): n_streams * n_channels * W above that -> LOF_E_SIZE, nothing is
 * enqueued.  All calls on a device share the array: calls that overlap on the GPU (two streams, two threads) race
 * and give undefined masks; calls on one stream, or ordered by events, are safe.  Nothing needs clearing between
 * calls (each kernel writes every word the next one reads).  LOF_E_NULL / LOF_E_ALIGN as elsewhere; LOF_E_PARAM
 * for a zero dimension, n_channels > 256, eta outside [0, 1] or not finite, directions 0 or unknown bits, device
 * outside 0..63.  eta == 0 returns LOF_OK without touching the mask.  Only enqueues work, like lof_flag_block. */
#define LOF_NOALLOC_MAX_WORDS (2u * 1024u * 1024u)
int lof_sir_noalloc(uint32_t* d_flags, lof_stream_stats* d_stats, uint32_t n_streams, uint32_t n_channels,
                    uint32_t n_time, float eta, uint32_t directions, int device, void* cuda_stream);

const char* lof_strerror(int code);
const char* lof_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LOF_H */
