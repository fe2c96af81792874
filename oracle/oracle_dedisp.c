/*
 * oracle_dedisp.c -- CPU ORACLE for brute-force incoherent dedispersion.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing under oracle/ is part of the product.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
 * load or call it.  It shares no code, header, table or helper with the CUDA path
 * (paper_2605_03531_b200/csrc) and includes nothing from include/.
 *
 * The method is an exact sum, so the oracle is the plain definition written out
 * (SURVEY.md section 8(c), steps O1..O8), in the order and notation of the paper:
 *
 *   - cold-plasma delay law, PAPER.md:256-263 (Eq. 1.1):
 *         dt = 4.14881 ms * DM * (nu1^-2 - nu2^-2), nu in GHz
 *     used in the north_star's units: K = 4.148808e3 s MHz^2 cm^3/pc (reading A1).
 *   - "0 DM time series" = sum over channels without delay correction, PAPER.md:431 (Fig 3.3).
 *   - brute-force dedispersion is the O(m x N) direct sum per trial, PAPER.md:421 (section 3.2).
 *   - many trial DMs over a plan, PAPER.md:317 (section 2.1).
 *
 * Precision: delays in IEEE double, rounded half away from zero; samples summed as unsigned
 * 64-bit integers (exact); one conversion uint64 -> double -> float (round to nearest even)
 * at the end.  No blocking, fusion or reordering beyond the definition: loop order is
 * trial -> channel -> time.  OpenMP parallelises over trials only (independent sums).
 *
 * Pins (tests/test_oracle_pins.py, all run without a GPU): hand-worked Eq. 1.1 values
 * (tests/golden/delay_hand_values.txt), structural invariants of the delay table, DM=0 equals
 * the plain channel sum, injected impulse peaks at nchans*height, linearity, constant input,
 * time-shift covariance, single channel identity, decimation reduction, pure-Python brute
 * force on a tiny case with hand-derived delays, zeroed-channel subset.  Nothing here is
 * "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_INVALID (-1)
#define ORACLE_ERR_TOO_SHORT (-2)
#define ORACLE_ERR_NOMEM (-3)

/* Dispersion constant in s MHz^2 cm^3 / pc (north_star; PAPER.md:258 prints 4.14881 ms GHz^2). */
static const double ORACLE_K = 4.148808e3;

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* O2: f_c = f_top + c * width, c = 0..nchans-1 (channel 0 is the top of the band). */
int oracle_channel_freqs(double f_top_mhz, double chan_width_mhz, int32_t nchans, double *f_mhz) {
  if (!f_mhz || nchans < 1 || !(chan_width_mhz < 0.0) || !(f_top_mhz > 0.0)) return ORACLE_ERR_INVALID;
  if (!(f_top_mhz + (nchans - 1) * chan_width_mhz > 0.0)) return ORACLE_ERR_INVALID;
  for (int32_t c = 0; c < nchans; ++c) f_mhz[c] = f_top_mhz + (double)c * chan_width_mhz;
  return ORACLE_OK;
}

/*
 * O3 + O4: delay table of one DM range, PAPER.md:258 (Eq. 1.1).
 *   tsamp_r = tsamp * decim
 *   DM_j    = dm_lo + j * dm_step                        (a product, not a running sum)
 *   x       = K * DM_j * (1/f_c^2 - 1/f_top^2) / tsamp_r
 *   d(c,j)  = floor(x + 0.5)                             (x >= 0: round half away from zero)
 * delays: [ndm][nchans], row-major, int64.
 */
int oracle_delay_table(double f_top_mhz, double chan_width_mhz, int32_t nchans, double tsamp_s,
                       int32_t decim, double dm_lo, double dm_step, int32_t ndm, int64_t *delays) {
  if (!delays || nchans < 1 || ndm < 1 || !(tsamp_s > 0.0) || !(chan_width_mhz < 0.0)) return ORACLE_ERR_INVALID;
  if (!(decim == 1 || decim == 2 || decim == 4 || decim == 8)) return ORACLE_ERR_INVALID;
  if (!(dm_lo >= 0.0) || !(dm_step >= 0.0)) return ORACLE_ERR_INVALID;
  double *f = (double *)malloc(sizeof(double) * (size_t)nchans);
  if (!f) return ORACLE_ERR_NOMEM;
  int rc = oracle_channel_freqs(f_top_mhz, chan_width_mhz, nchans, f);
  if (rc != ORACLE_OK) { free(f); return rc; }
  const double tsamp_r = tsamp_s * (double)decim;
  for (int32_t j = 0; j < ndm; ++j) {
    const double dm = dm_lo + (double)j * dm_step;
    for (int32_t c = 0; c < nchans; ++c) {
      const double x = ORACLE_K * dm * (1.0 / (f[c] * f[c]) - 1.0 / (f_top_mhz * f_top_mhz)) / tsamp_r;
      delays[(size_t)j * (size_t)nchans + (size_t)c] = (int64_t)floor(x + 0.5);
    }
  }
  free(f);
  return ORACLE_OK;
}

/*
 * O6: time decimation by summing (not averaging) `decim` adjacent samples; blocks start at
 * sample 0 and the nsamps mod decim tail is dropped (reading A8).
 *   y[c][t'] = sum_{i<decim} x[c][decim*t' + i],  t' = 0 .. nsamps/decim - 1
 * x: [nchans][nsamps] unsigned, in_bits = 8 or 16.  y: [nchans][nsamps/decim] uint32.
 */
int oracle_decimate(const void *x, int32_t in_bits, int64_t nchans, int64_t nsamps, int32_t decim, uint32_t *y) {
  if (!x || !y || nchans < 1 || nsamps < 1) return ORACLE_ERR_INVALID;
  if (!(decim == 1 || decim == 2 || decim == 4 || decim == 8)) return ORACLE_ERR_INVALID;
  if (!(in_bits == 8 || in_bits == 16)) return ORACLE_ERR_INVALID;
  const int64_t ns_r = nsamps / decim;
  for (int64_t c = 0; c < nchans; ++c) {
    for (int64_t t = 0; t < ns_r; ++t) {
      uint32_t s = 0;
      for (int32_t i = 0; i < decim; ++i) {
        const int64_t idx = c * nsamps + decim * t + i;
        s += (in_bits == 8) ? (uint32_t)((const uint8_t *)x)[idx] : (uint32_t)((const uint16_t *)x)[idx];
      }
      y[c * ns_r + t] = s;
    }
  }
  return ORACLE_OK;
}

/*
 * O7: the direct sum, PAPER.md:421 (O(m x N) per trial) with the sign of PAPER.md:250/Eq. 1.1
 * (lower frequencies arrive later, so channel c is read d(c,j) samples LATER):
 *   S[j][t'] = sum_{c=0}^{nchans-1} y[c][t' + d(c,j)]
 * evaluated for the selected trials sel[0..nsel) (indices into the delay table; sel == NULL means
 * trials 0..nsel-1) and the output window t' = t0 .. t0+nt-1, which must lie inside the valid span
 * nout = ns_r - max_c d(c,j) of every selected trial (no padding, no wrap; reading A9).
 * out: [nsel][nt] float = (float)(double)S  (one rounding, to nearest even).
 */
int oracle_dedisperse(const uint32_t *y, int64_t nchans, int64_t ns_r, const int64_t *delays,
                      int32_t ndm, const int32_t *sel, int32_t nsel, int64_t t0, int64_t nt, float *out) {
  if (!y || !delays || !out || nchans < 1 || ns_r < 1 || ndm < 1 || nsel < 1 || t0 < 0 || nt < 1) return ORACLE_ERR_INVALID;
  for (int32_t s = 0; s < nsel; ++s) {
    const int32_t j = sel ? sel[s] : s;
    if (j < 0 || j >= ndm) return ORACLE_ERR_INVALID;
    for (int64_t c = 0; c < nchans; ++c) {
      const int64_t d = delays[(size_t)j * (size_t)nchans + (size_t)c];
      if (d < 0) return ORACLE_ERR_INVALID;
      if (t0 + nt + d > ns_r) return ORACLE_ERR_TOO_SHORT;
    }
  }
  int failed = 0;
#pragma omp parallel for schedule(dynamic, 1)
  for (int32_t s = 0; s < nsel; ++s) {
    const int32_t j = sel ? sel[s] : s;
    uint64_t *acc = (uint64_t *)calloc((size_t)nt, sizeof(uint64_t));
    if (!acc) { failed = 1; continue; }
    for (int64_t c = 0; c < nchans; ++c) {
      const int64_t d = delays[(size_t)j * (size_t)nchans + (size_t)c];
      const uint32_t *row = y + c * ns_r + t0 + d;
      for (int64_t t = 0; t < nt; ++t) acc[t] += (uint64_t)row[t];
    }
    for (int64_t t = 0; t < nt; ++t) out[(size_t)s * (size_t)nt + (size_t)t] = (float)(double)acc[t];
    free(acc);
  }
  return failed ? ORACLE_ERR_NOMEM : ORACLE_OK;
}
