/*
 * oracle_sps.c -- CPU ORACLE for the boxcar single-pulse search on rows of the DM-time plane
 * (SURVEY.md 8(f) NEXT-2).
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing under oracle/ is part of the product; it shares no code, header or
 * table with paper_2605_03531_b200/csrc and includes nothing from include/.
 *
 * What the thesis fixes (section 2.1): "The SPS module searches for statistically
 * significant single pulses above a user-specified threshold using time-domain boxcar filtering."  Widths,
 * normalisation and the output are not given; the readings taken are listed in DESIGN.md (B1-B6) and written
 * out here step by step for one row x[0..n) of the DM-time plane (non-negative integers held in floats):
 *
 *   S1 = sum x, S2 = sum x^2                       exact unsigned 64-bit integers
 *   mean = S1/n, var = S2/n - mean*mean (>= 0), sigma = sqrt(var)          IEEE double, this operation order
 *   for k = 0..K-1, width w = 2^k (widths above n: snr 0, tmax -1, count 0):
 *     B[t]  = sum_{i<w} x[t+i],  t = 0..n-w         exact integers (running sum)
 *     best  = max_t B[t],  tmax = smallest t with B[t] = best
 *     den   = sigma*sqrt(w);  snr = sigma > 0 ? (best - w*mean)/den : 0     (rounded once to float)
 *     thr   = w*mean + threshold*den;  count = #{t : B[t] > thr}
 *
 * No FMA contraction (compile with -ffp-contract=off), so a device implementation that uses the same
 * round-to-nearest operations in the same order gets the same bits.
 *
 * "The list of candidates thus generated is filtered ..." -- the search hands a LIST on to the next
 * stage.  Reading B5: the list holds every (row, width index k, t) with B[t] > thr, each with
 * snr = (float)((B[t] - w*mean)/den) (0 when sigma = 0), ordered by row, then k, then t.  Its length per (row, k) is the
 * count above.  oracle_sps_candidates writes it (first `cap` entries) and returns the total through *total.
 *
 * Pins (tests/test_oracle_sps_pins.py): constant row, single impulse and boxcar pulse closed forms, a linear
 * ramp's mean and variance, count limits for extreme thresholds, a pure-Python brute force on random rows,
 * invariance of tmax under a constant offset.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define ORACLE_OK 0
#define ORACLE_ERR_INVALID (-1)
#define ORACLE_ERR_NOMEM (-3)

/* rows: [nrows][pitch] floats, the first n of each row are valid.  Outputs [nrows][K]. */
int oracle_sps(const float* rows, int64_t nrows, int64_t pitch, int64_t n, int K, double threshold, float* snr,
               int32_t* tmax, int32_t* count, double* mean_out, double* sigma_out) {
  if (!rows || !snr || !tmax || !count || nrows < 0 || n < 1 || pitch < n || K < 1 || K > 20) return ORACLE_ERR_INVALID;
  int rc = ORACLE_OK;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t r = 0; r < nrows; ++r) {
    const float* x = rows + r * pitch;
    uint64_t s1 = 0, s2 = 0;
    for (int64_t t = 0; t < n; ++t) {
      const uint64_t v = (uint64_t)x[t];
      s1 += v;
      s2 += v * v;
    }
    const double mean = (double)s1 / (double)n;
    double var = (double)s2 / (double)n - mean * mean;
    if (var < 0.0) var = 0.0;
    const double sigma = sqrt(var);
    if (mean_out) mean_out[r] = mean;
    if (sigma_out) sigma_out[r] = sigma;
    for (int k = 0; k < K; ++k) {
      const int64_t w = (int64_t)1 << k;
      float* o_snr = snr + r * K + k;
      int32_t* o_t = tmax + r * K + k;
      int32_t* o_c = count + r * K + k;
      if (w > n) {
        *o_snr = 0.0f, *o_t = -1, *o_c = 0;
        continue;
      }
      const double den = sigma * sqrt((double)w);
      const double thr = (double)w * mean + threshold * den;
      uint64_t b = 0;
      for (int64_t i = 0; i < w; ++i) b += (uint64_t)x[i];
      uint64_t best = b;
      int64_t tbest = 0;
      int32_t cnt = (double)b > thr ? 1 : 0;
      for (int64_t t = 1; t + w <= n; ++t) {
        b += (uint64_t)x[t + w - 1];
        b -= (uint64_t)x[t - 1];
        if (b > best) best = b, tbest = t;
        if ((double)b > thr) ++cnt;
      }
      *o_snr = sigma > 0.0 ? (float)(((double)best - (double)w * mean) / den) : 0.0f;
      *o_t = (int32_t)tbest;
      *o_c = cnt;
    }
  }
  return rc;
}

/* The candidate list (reading B5): entries (row, k, t, snr) in the order row, k, t.  cand_* hold `cap` entries; *total =
 * number of candidates found (may exceed cap: the rest is counted, not written). */
int oracle_sps_candidates(const float* rows, int64_t nrows, int64_t pitch, int64_t n, int K, double threshold,
                          int32_t* cand_row, int32_t* cand_k, int32_t* cand_t, float* cand_snr, int64_t cap, int64_t* total) {
  if (!rows || !total || nrows < 0 || n < 1 || pitch < n || K < 1 || K > 20 || cap < 0) return ORACLE_ERR_INVALID;
  if (cap > 0 && (!cand_row || !cand_k || !cand_t || !cand_snr)) return ORACLE_ERR_INVALID;
  int64_t nc = 0;
  for (int64_t r = 0; r < nrows; ++r) {
    const float* x = rows + r * pitch;
    uint64_t s1 = 0, s2 = 0;
    for (int64_t t = 0; t < n; ++t) {
      const uint64_t v = (uint64_t)x[t];
      s1 += v;
      s2 += v * v;
    }
    const double mean = (double)s1 / (double)n;
    double var = (double)s2 / (double)n - mean * mean;
    if (var < 0.0) var = 0.0;
    const double sigma = sqrt(var);
    for (int k = 0; k < K; ++k) {
      const int64_t w = (int64_t)1 << k;
      if (w > n) continue;
      const double den = sigma * sqrt((double)w);
      const double wmean = (double)w * mean;
      const double thr = wmean + threshold * den;
      for (int64_t t = 0; t + w <= n; ++t) {
        uint64_t b = 0;
        for (int64_t i = 0; i < w; ++i) b += (uint64_t)x[t + i]; /* the boxcar by its definition */
        if ((double)b > thr) {
          if (nc < cap) {
            cand_row[nc] = (int32_t)r;
            cand_k[nc] = k;
            cand_t[nc] = (int32_t)t;
            cand_snr[nc] = sigma > 0.0 ? (float)(((double)b - wmean) / den) : 0.0f;
          }
          ++nc;
        }
      }
    }
  }
  *total = nc;
  return ORACLE_OK;
}
