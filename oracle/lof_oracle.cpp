// lof_oracle.cpp — ORACLE (test infrastructure, not the product).  See lof_oracle.h.
// Plain single-threaded C++17, fp64 arithmetic, written from PAPER.md (arXiv 1701.08197).
// Shares no code with the CUDA path.  "parity unpinned" for readings F7, F8, F10, S1-S4,
// H3'-H6' against the authors' code (not available); see DESIGN.md §3.
#include "lof_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>

extern "C" {

// PAPER.md:41  factor_I = startThreshold * p^(log2 I) / I.  For I = 2^k this is
// startThreshold * (p/2)^k; computed by repeated multiplication (reading F1).
void lofo_factor_table(double start_threshold, double p, uint32_t n_out, double* out) {
  double f = start_threshold;
  for (uint32_t k = 0; k < n_out; ++k) {
    out[k] = f;
    f = f * (p / 2.0);
  }
}

// PAPER.md:41  threshold_I = median + stddev * factor_I * sensitivity.
void lofo_threshold_table(double median, double stddev, double start_threshold, double p,
                          double sensitivity, uint32_t n_out, double* out) {
  std::vector<double> factor(n_out);
  lofo_factor_table(start_threshold, p, n_out, factor.data());
  for (uint32_t k = 0; k < n_out; ++k) out[k] = median + stddev * factor[k] * sensitivity;
}

// O1-O3 (PAPER.md:41 uses median and stddev; :120 "means, medians, standard deviations").
void lofo_statistics(const float* x, uint64_t n, lofo_stream_stats* out) {
  out->median = 0.f; out->mean = 0.0; out->stddev = 0.0; out->n_flagged = 0; out->n_nonfinite = 0;
  if (n == 0) return;
  uint32_t bad = 0;
  for (uint64_t i = 0; i < n; ++i) if (!std::isfinite(x[i])) ++bad;
  out->n_nonfinite = bad;
  if (bad) return;                                   // reading S6: other fields unspecified
  double sum = 0.0;
  for (uint64_t i = 0; i < n; ++i) sum += (double)x[i];
  const double mean = sum / (double)n;
  double ss = 0.0;
  for (uint64_t i = 0; i < n; ++i) { const double d = (double)x[i] - mean; ss += d * d; }
  out->mean = mean;
  out->stddev = std::sqrt(ss / (double)n);           // population, about the mean (S2)
  std::vector<float> v(x, x + n);
  std::nth_element(v.begin(), v.begin() + n / 2, v.end());   // O(N) selection
  out->median = v[n / 2];                            // rank floor(N/2), 0-based (S3)
}

// PAPER.md:120 "the MAD (Median Absolute Deviation)": median of |x - median|, same rank convention as the median (S3).
float lofo_mad(const float* x, uint64_t n, float median) {
  if (n == 0) return 0.f;
  std::vector<float> d(n);
  for (uint64_t i = 0; i < n; ++i) d[i] = (float)std::fabs((double)x[i] - (double)median);
  std::nth_element(d.begin(), d.begin() + n / 2, d.end());
  return d[n / 2];
}

static inline void mark_margin(uint8_t* margin, int64_t ms, uint64_t t0, uint64_t I, double S,
                               double lim, double rel) {
  if (!margin) return;
  if (std::fabs(S - lim) <= rel * std::fabs(lim))
    for (uint64_t j = 0; j < I; ++j) margin[(int64_t)(t0 + j) * ms] = 1;
}

// PAPER.md:37-47, Fig. 1: window I = 1, 2, 4, ...; a window is flagged when its sum, with
// already-flagged samples replaced by threshold_I (F7), exceeds I*threshold_I (F4, strict F6).
// Flags are frozen at the start of each iteration (F8).  The literal double loop.
void lofo_sumthreshold_1d_literal(const float* x, uint64_t n, int64_t stride, uint8_t* mask,
                                  int64_t ms, const double* thresholds, uint32_t n_levels,
                                  uint8_t* margin, double margin_rel) {
  std::vector<uint8_t> P(n);
  for (uint32_t k = 0; k < n_levels; ++k) {
    const uint64_t I = (uint64_t)1 << k;
    if (I > n) break;                                // F9: window larger than the axis is skipped
    const double T = thresholds[k];
    const double lim = (double)I * T;
    for (uint64_t i = 0; i < n; ++i) P[i] = mask[(int64_t)i * ms];
    for (uint64_t t0 = 0; t0 + I <= n; ++t0) {
      double S = 0.0;
      for (uint64_t j = 0; j < I; ++j)
        S += P[t0 + j] ? T : (double)x[(int64_t)(t0 + j) * stride];
      mark_margin(margin, ms, t0, I, S, lim, margin_rel);
      if (S > lim)
        for (uint64_t j = 0; j < I; ++j) mask[(int64_t)(t0 + j) * ms] = 1;
    }
  }
}

// Same iteration in O(n): S - I*T = sum over the window of (v - T), v the substituted value,
// i.e. 0 for a flagged sample and x - T otherwise; taken as differences of an fp64 prefix
// array of those terms (a constant line gives exactly 0, keeping F6's "constant input yields
// no flags").  Checked against the literal loop in tests/test_oracle_pins.py (pin P2).
void lofo_sumthreshold_1d_fast(const float* x, uint64_t n, int64_t stride, uint8_t* mask,
                               int64_t ms, const double* thresholds, uint32_t n_levels,
                               uint8_t* margin, double margin_rel) {
  std::vector<double> pre(n + 1);
  std::vector<int32_t> diff(n + 1);
  for (uint32_t k = 0; k < n_levels; ++k) {
    const uint64_t I = (uint64_t)1 << k;
    if (I > n) break;
    const double T = thresholds[k];
    const double lim = (double)I * T;
    pre[0] = 0.0;
    for (uint64_t i = 0; i < n; ++i)
      pre[i + 1] = pre[i] + (mask[(int64_t)i * ms] ? 0.0 : (double)x[(int64_t)i * stride] - T);
    std::fill(diff.begin(), diff.end(), 0);
    for (uint64_t t0 = 0; t0 + I <= n; ++t0) {
      const double excess = pre[t0 + I] - pre[t0];          // S - I*T
      mark_margin(margin, ms, t0, I, excess + lim, lim, margin_rel);
      if (excess > 0.0) { diff[t0] += 1; diff[t0 + I] -= 1; }
    }
    int32_t cover = 0;
    for (uint64_t i = 0; i < n; ++i) {
      cover += diff[i];
      if (cover > 0) mask[(int64_t)i * ms] = 1;
    }
  }
}

// PAPER.md:75 "we may have to compute amplitudes first"; reading S5: x = re^2 + im^2 formed as an
// integer (at most 2 * 32768^2 = 2^31, so 64-bit arithmetic keeps (-32768, -32768) defined) and
// converted to float32 once, round-to-nearest.
void lofo_power_from_ci16(const int16_t* volt, uint64_t n, float* power) {
  for (uint64_t i = 0; i < n; ++i) {
    const int64_t re = volt[2 * i], im = volt[2 * i + 1];
    power[i] = (float)(re * re + im * im);
  }
}


// "all ranges of consecutive flagged samples are extended by flagging 20% more samples, before
// and after the original range".  Runs are those of the input mask (SIR-2); floor(eta * len) samples on each
// side (SIR-3), clipped at the ends of the line (SIR-4).
void lofo_sir_1d(uint8_t* mask, uint64_t n, int64_t stride, double eta) {
  if (!(eta > 0.0) || n == 0) return;
  std::vector<uint8_t> in(n);
  for (uint64_t i = 0; i < n; ++i) in[i] = mask[(int64_t)i * stride];
  uint64_t i = 0;
  while (i < n) {
    if (!in[i]) { ++i; continue; }
    uint64_t b = i;
    while (b < n && in[b]) ++b;                              // maximal run [i, b)
    const uint64_t len = b - i;
    const uint64_t ext = (uint64_t)std::floor(eta * (double)len);
    const uint64_t lo = ext > i ? 0 : i - ext;               // clipped at the start of the line
    const uint64_t hi = b + ext > n ? n : b + ext;           // ... and at its end
    for (uint64_t j = lo; j < i; ++j) mask[(int64_t)j * stride] = 1;
    for (uint64_t j = b; j < hi; ++j) mask[(int64_t)j * stride] = 1;
    i = b;
  }
}

// The operator on a packed block mask: frequency direction first, then time on the result (SIR-5, the order of
// the SumThreshold runs).
void lofo_sir_block(uint32_t* flags, uint64_t S, uint64_t C, uint64_t T, double eta, uint32_t directions) {
  if (!(eta > 0.0)) return;
  const uint64_t words = (T + 31) / 32;
  std::vector<uint8_t> M(C * T);
  for (uint64_t s = 0; s < S; ++s) {
    uint32_t* fs = flags + s * C * words;
    for (uint64_t c = 0; c < C; ++c)
      for (uint64_t t = 0; t < T; ++t) M[c * T + t] = (fs[c * words + (t >> 5)] >> (t & 31)) & 1u;
    if (directions & 1u)
      for (uint64_t t = 0; t < T; ++t) lofo_sir_1d(M.data() + t, C, (int64_t)T, eta);
    if (directions & 2u)
      for (uint64_t c = 0; c < C; ++c) lofo_sir_1d(M.data() + c * T, T, 1, eta);
    for (uint64_t c = 0; c < C; ++c) {
      for (uint64_t w = 0; w < words; ++w) fs[c * words + w] = 0;
      for (uint64_t t = 0; t < T; ++t)
        if (M[c * T + t]) fs[c * words + (t >> 5)] |= (uint32_t)1 << (t & 31);
    }
  }
}

// O1-O9 for a whole block (PAPER.md:37-47 per line; frequency first then time, PAPER.md:83,
// :180; the time run starts from and substitutes the frequency run's flags, reading F10;
// statistics over all samples of the stream before any flagging, reading S1).
int lofo_flag_block(const lofo_params* prm, const float* power, uint32_t* flags,
                    lofo_stream_stats* stats, double* rowsum, uint32_t* rowcnt,
                    uint8_t* mask_freq, uint8_t* margin, double margin_rel, int use_literal) {
  const uint64_t S = prm->n_streams, C = prm->n_channels, T = prm->n_time;
  if (!S || !C || !T || !prm->max_window || (prm->max_window & (prm->max_window - 1))) return -1;
  uint32_t n_levels = 0;
  while (((uint32_t)1 << n_levels) <= prm->max_window) ++n_levels;     // I = 1 .. max_window
  const uint64_t words = (T + 31) / 32;
  auto run = use_literal ? lofo_sumthreshold_1d_literal : lofo_sumthreshold_1d_fast;
  std::vector<uint8_t> M(C * T);
  std::vector<double> thr(n_levels);
  for (uint64_t s = 0; s < S; ++s) {
    const float* X = power + s * C * T;
    lofo_stream_stats st;
    lofo_statistics(X, C * T, &st);                                     // O1-O3
    uint8_t* mg = margin ? margin + s * C * T : nullptr;
    if (mg) std::memset(mg, 0, C * T);
    // robust scale (reading R1): 1.4826 * MAD takes the place of the standard deviation in threshold_I; the
    // factor makes it an estimate of sigma for Gaussian data.  The stats record reports the scale that was used.
    if (!st.n_nonfinite && prm->stats_mode == 1) st.stddev = 1.4826 * (double)lofo_mad(X, C * T, st.median);
    if (st.n_nonfinite) {                                               // reading S6
      std::fill(M.begin(), M.end(), (uint8_t)1);
    } else {
      lofo_threshold_table((double)st.median, st.stddev, prm->start_threshold, prm->p,
                           prm->sensitivity, n_levels, thr.data());     // O4
      std::fill(M.begin(), M.end(), (uint8_t)0);                        // O5
      if (prm->directions & 1u)                                         // O6: along channels
        for (uint64_t t = 0; t < T; ++t)
          run(X + t, C, (int64_t)T, M.data() + t, (int64_t)T, thr.data(), n_levels,
              mg ? mg + t : nullptr, margin_rel);
      if (mask_freq) std::memcpy(mask_freq + s * C * T, M.data(), C * T);
      if (prm->directions & 2u)                                         // O7: along time
        for (uint64_t c = 0; c < C; ++c)
          run(X + c * T, T, 1, M.data() + c * T, 1, thr.data(), n_levels,
              mg ? mg + c * T : nullptr, margin_rel);
    }
    if (st.n_nonfinite && mask_freq) std::memset(mask_freq + s * C * T, 1, C * T);
    uint64_t nf = 0;
    for (uint64_t c = 0; c < C; ++c) {                                  // O8, O9
      uint32_t* fw = flags + (s * C + c) * words;
      for (uint64_t w = 0; w < words; ++w) fw[w] = 0;
      double rs = 0.0; uint32_t rc = 0;
      for (uint64_t t = 0; t < T; ++t) {
        if (M[c * T + t]) { fw[t >> 5] |= (uint32_t)1 << (t & 31); ++nf; }
        else { rs += (double)X[c * T + t]; ++rc; }
      }
      if (rowsum) rowsum[s * C + c] = rs;
      if (rowcnt) rowcnt[s * C + c] = rc;
    }
    // SIR operator on the packed mask of this stream, after the row sums were taken: it "operates
    // on the flag masks only, and not on the actual data", reading SIR-6
    if (prm->sir_eta > 0.0) {
      lofo_sir_block(flags + s * C * words, 1, C, T, prm->sir_eta, prm->directions);
      nf = 0;
      for (uint64_t i = 0; i < C * words; ++i) nf += (uint64_t)__builtin_popcount(flags[s * C * words + i]);
    }
    st.n_flagged = nf;
    if (stats) stats[s] = st;
  }
  return 0;
}

// ---- fully integrated mode (Fig. 4).  One 1-D vector: statistics of the vector itself (O1-O3),
// thresholds (O4), one SumThreshold run (O7 on a single line).  Returns the number of flagged entries.
static uint64_t run_vector(const lofo_params* prm, const float* v, uint64_t n, uint8_t* mask, lofo_stream_stats* st_out) {
  uint32_t n_levels = 0;
  while (((uint32_t)1 << n_levels) <= prm->max_window) ++n_levels;
  lofo_stream_stats st;
  lofo_statistics(v, n, &st);
  if (st.n_nonfinite) std::fill(mask, mask + n, (uint8_t)1);          // S6
  else {
    std::vector<double> thr(n_levels);
    lofo_threshold_table((double)st.median, st.stddev, prm->start_threshold, prm->p, prm->sensitivity, n_levels,
                         thr.data());
    std::fill(mask, mask + n, (uint8_t)0);
    lofo_sumthreshold_1d_fast(v, n, 1, mask, 1, thr.data(), n_levels, nullptr, 0.0);
  }
  uint64_t nf = 0;
  for (uint64_t i = 0; i < n; ++i) nf += mask[i];
  st.n_flagged = nf;
  if (st_out) *st_out = st;
  return nf;
}

int lofo_flag_block_integrated(const lofo_params* prm, const float* power, uint32_t* flags, float* spectrum,
                               float* series, uint8_t* chan_mask, uint8_t* time_mask,
                               lofo_stream_stats* stats_freq, lofo_stream_stats* stats_time) {
  const uint64_t S = prm->n_streams, C = prm->n_channels, T = prm->n_time;
  if (!S || !C || !T || !prm->max_window || (prm->max_window & (prm->max_window - 1))) return -1;
  const uint64_t words = (T + 31) / 32;
  std::vector<float> a(C), b(T);
  std::vector<uint8_t> Mc(C), Mt(T);
  for (uint64_t s = 0; s < S; ++s) {
    const float* X = power + s * C * T;
    // "integrate the time direction fully for frequency flagging"; frequency first
    for (uint64_t c = 0; c < C; ++c) {
      double sum = 0.0;
      for (uint64_t t = 0; t < T; ++t) sum += (double)X[c * T + t];
      a[c] = (float)(sum / (double)T);
    }
    std::fill(Mc.begin(), Mc.end(), (uint8_t)0);
    lofo_stream_stats sf; std::memset(&sf, 0, sizeof sf);
    if (prm->directions & 1u) run_vector(prm, a.data(), C, Mc.data(), &sf);
    // "integrate the frequency direction fully for time domain flagging": over the channels left unflagged
    uint64_t n_unf = 0;
    for (uint64_t c = 0; c < C; ++c) n_unf += Mc[c] ? 0 : 1;
    for (uint64_t t = 0; t < T; ++t) {
      double sum = 0.0;
      for (uint64_t c = 0; c < C; ++c) if (!Mc[c]) sum += (double)X[c * T + t];
      b[t] = n_unf ? (float)(sum / (double)n_unf) : 0.f;
    }
    std::fill(Mt.begin(), Mt.end(), (uint8_t)0);
    lofo_stream_stats stt; std::memset(&stt, 0, sizeof stt);
    if ((prm->directions & 2u) && n_unf) run_vector(prm, b.data(), T, Mt.data(), &stt);
    if (flags)
      for (uint64_t c = 0; c < C; ++c) {
        uint32_t* fw = flags + (s * C + c) * words;
        for (uint64_t w = 0; w < words; ++w) fw[w] = 0;
        for (uint64_t t = 0; t < T; ++t) if (Mc[c] || Mt[t]) fw[t >> 5] |= (uint32_t)1 << (t & 31);
      }
    if (spectrum) std::memcpy(spectrum + s * C, a.data(), C * sizeof(float));
    if (series) std::memcpy(series + s * T, b.data(), T * sizeof(float));
    if (chan_mask) std::memcpy(chan_mask + s * C, Mc.data(), C);
    if (time_mask) std::memcpy(time_mask + s * T, Mt.data(), T);
    if (stats_freq) stats_freq[s] = sf;
    if (stats_time) stats_time[s] = stt;
  }
  return 0;
}

// ---- history flagger (PAPER.md:87-116 pseudocode; buffer of 32-bit means) ----
struct lofo_history {
  lofo_params prm;
  std::vector<float> ring;        // [S][C][H]
  std::vector<uint32_t> head, count;
};

lofo_history* lofo_history_create(const lofo_params* prm) {
  lofo_history* h = new lofo_history;
  h->prm = *prm;
  const uint64_t rows = (uint64_t)prm->n_streams * prm->n_channels;
  h->ring.assign(rows * prm->history_length, 0.f);
  h->head.assign(rows, 0);
  h->count.assign(rows, 0);
  return h;
}
void lofo_history_destroy(lofo_history* h) { delete h; }
void lofo_history_reset(lofo_history* h) {
  std::fill(h->ring.begin(), h->ring.end(), 0.f);
  std::fill(h->head.begin(), h->head.end(), 0u);
  std::fill(h->count.begin(), h->count.end(), 0u);
}

void lofo_history_update(lofo_history* h, const double* rowsum, const uint32_t* rowcnt,
                         uint32_t* flags, uint8_t* row_flagged, uint8_t* near, double near_rel) {
  const lofo_params& P = h->prm;
  const uint64_t rows = (uint64_t)P.n_streams * P.n_channels, T = P.n_time, H = P.history_length;
  const uint64_t words = (T + 31) / 32;
  const double sens = P.history_sensitivity > 0.0 ? P.history_sensitivity : P.sensitivity;
  for (uint64_t r = 0; r < rows; ++r) {
    if (near) near[r] = 0;
    if (H == 0) { row_flagged[r] = 0; continue; }
    float* ring = h->ring.data() + r * H;
    uint32_t& head = h->head[r];
    uint32_t& cnt = h->count[r];
    auto push = [&](float v) { ring[head] = v; head = (uint32_t)((head + 1) % H); cnt = std::min<uint32_t>(cnt + 1, (uint32_t)H); };
    if (rowcnt[r] == 0) { row_flagged[r] = 1; continue; }               // H1
    const double cur = rowsum[r] / (double)rowcnt[r];                   // H2: meanOfUnflaggedSamples()
    if (cnt < P.history_min_fill) { push((float)cur); row_flagged[r] = 0; continue; }   // H3
    double m = 0.0;
    for (uint32_t i = 0; i < cnt; ++i) m += (double)ring[i];            // H4: meanOfMeans()
    m /= (double)cnt;
    double ss = 0.0;
    for (uint32_t i = 0; i < cnt; ++i) { const double d = (double)ring[i] - m; ss += d * d; }
    const double sd = std::sqrt(ss / (double)cnt);                      // stddevOfMeans()
    const double thr = m + sens * sd;                                   // H5
    if (near && std::fabs(cur - thr) <= near_rel * std::fabs(thr)) near[r] = 1;
    if (cur < thr) { push((float)cur); row_flagged[r] = 0; }            // H6
    else {
      push((float)thr); row_flagged[r] = 1;
      uint32_t* fw = flags + r * words;
      for (uint64_t w = 0; w < words; ++w) fw[w] = 0xFFFFFFFFu;
      if (T & 31) fw[words - 1] = ((uint32_t)1 << (T & 31)) - 1;        // padding bits stay 0
    }
  }
}

void lofo_history_export(const lofo_history* h, float* ring, uint32_t* head, uint32_t* count) {
  if (ring) std::memcpy(ring, h->ring.data(), h->ring.size() * sizeof(float));
  if (head) std::memcpy(head, h->head.data(), h->head.size() * sizeof(uint32_t));
  if (count) std::memcpy(count, h->count.data(), h->count.size() * sizeof(uint32_t));
}

}  // extern "C"
