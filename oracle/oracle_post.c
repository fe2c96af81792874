/*
 * oracle_post.c -- CPU ORACLE for the pulsar-side post-processing of a dedispersed time series
 * (SURVEY.md 8(f) NEXT-4): downsampling, running-median de-reddening, re-sampling.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing under oracle/ is part of the product; it shares no code, header or table
 * with paper_2605_03531_b200/csrc and includes nothing from include/.
 *
 * What the thesis fixes, and the readings taken where it is silent (C1-C7):
 *
 *   PAPER.md:421 (3.2)  "The dedispersed time series is then downsampled by a user-input factor"
 *       C1: y[k] = sum_{i<F} x[k*F + i], k < floor(n/F): a SUM of F adjacent samples (as the input decimation,
 *           reading A8; a mean differs by the exact scale 1/F), blocks start at sample 0, the n mod F tail is
 *           dropped.  Accumulated in IEEE double in index order, rounded once to float.
 *
 *   PAPER.md:425 (3.3)  "de-reddening of the time series using running-median subtraction", window size a user
 *       choice (:437: more than twice the widest pulse, less than half the fluctuation time scale)
 *       C2: window W odd, 1 <= W <= n, h = (W-1)/2.  med[t] = the (h+1)-th smallest of x[s .. s+W), with
 *           s = min(max(t-h, 0), n-W): centred on t, and held at the first / last full window where a centred
 *           one would leave the series (no padding, no invented samples).  The median is written out by its plain
 *           definition: copy the window, sort it, take element h.  out[t] = x[t] - med[t] (one float subtraction
 *           = the exact difference rounded once).
 *
 *   PAPER.md:441-484 (3.4, Eqs 3.1-3.6)  re-sampling to remove the frequency derivatives f1, f2:
 *       Eq 3.3: tau = tau0 * (1 + f' t / f0 + f'' t^2 / (2 f0)), "the power in a particular time bin of the
 *       resampled time series is calculated by summing fractional powers from the corresponding bins";
 *       f1 <= 0: f' = -f1, f'' = -f2 applied as is; f1 > 0: reverse the series, use (Eqs 3.5, 3.6)
 *       f0~ = f0 + f1 T + f2 T^2/2, f' = f1 + f2 T, f'' = -f2 with T = n*tau0, resample, reverse again.
 *       C3: t in Eq 3.3 is the time (original axis, seconds from the start of the series handed to the
 *           transformation) at which the output bin STARTS; bins are laid end to end.  Edges are kept in units
 *           of the input sampling interval, u_k = T_k / tau0 (so that no derivative gives u_k = k exactly):
 *               u_0 = 0,   t_k = u_k * tau0,   w_k = tau_k / tau0 = 1 + f' t_k / F0 + f'' t_k^2 / (2 F0),   u_{k+1} = u_k + w_k
 *           (F0 = f0, or f0~ for the reversed case), evaluated in IEEE double in exactly this order:
 *               w_k = (1 + (f' * t_k) / F0) + (f'' * (t_k * t_k)) / (2 * F0).
 *       C4: the output has M bins, M = the number of k with u_{k+1} <= n (only complete bins).  The thesis assumes
 *           that the series is only compressed (w_k >= 1: "we assume that the frequency derivative does not change
 *           sign ... to avoid the complications of compressing a part of the time series and stretching the
 *           remaining part"); mild stretching is still well defined by C5, so the bound enforced is w_k >= 1/2
 *           (a bin is never shorter than half an input sample; M <= 2n) and anything below it is an error.
 *       C5: out[k] = sum_i x[i] * |[u_k,u_{k+1}) n [i,i+1)|, i.e. with
 *           i0 = floor(u_k), i1 = floor(u_{k+1}):
 *               i0 == i1:  x[i0] * (u_{k+1} - u_k)
 *               else:      x[i0] * ((i0+1) - u_k)  +  x[i0+1] + ... + x[i1-1]  +  (i1 < n ? x[i1] * (u_{k+1} - i1) : 0)
 *           accumulated left to right in double without fused multiply-add, rounded once to float.
 *       C6: f1 = 0 takes the "as is" branch.  C7: the reversed case returns reverse(resample(reverse(x))).
 *
 * Pins (tests/test_oracle_post_pins.py): constant / ramp / impulse / step closed forms and a pure-Python
 * sort-the-window brute force for the median; block sums against numpy for the downsampler; identity, power
 * conservation, constant-series closed form, exact rational (fractions.Fraction) overlap sums on tiny inputs,
 * equal spacing of a chirped pulse train after re-sampling and the reversal identity of Eqs 3.5-3.6.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_ERR_INVALID (-1)
#define ORACLE_ERR_NOMEM (-3)

/* C1.  in: [nrows][in_pitch], first n of each row valid; out: [nrows][out_pitch], first n/F written. */
int oracle_downsample(const float* in, int64_t nrows, int64_t in_pitch, int64_t n, int32_t F, float* out,
                      int64_t out_pitch) {
  if (!in || !out || nrows < 0 || n < 1 || F < 1 || in_pitch < n || out_pitch < n / F) return ORACLE_ERR_INVALID;
  const int64_t m = n / F;
  for (int64_t r = 0; r < nrows; ++r)
    for (int64_t k = 0; k < m; ++k) {
      double s = 0.0;
      for (int32_t i = 0; i < F; ++i) s += (double)in[r * in_pitch + k * F + i];
      out[r * out_pitch + k] = (float)s;
    }
  return ORACLE_OK;
}

static int cmp_float(const void* a, const void* b) {
  const float x = *(const float*)a, y = *(const float*)b;
  return (x > y) - (x < y);
}

/* C2.  med and out may each be NULL (not wanted).  Rows are independent (OpenMP over rows only). */
int oracle_running_median(const float* in, int64_t nrows, int64_t in_pitch, int64_t n, int32_t W, float* med,
                          float* out, int64_t out_pitch) {
  if (!in || nrows < 0 || n < 1 || W < 1 || (W & 1) == 0 || W > n || in_pitch < n || out_pitch < n) return ORACLE_ERR_INVALID;
  const int64_t h = (W - 1) / 2;
  int failed = 0;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t r = 0; r < nrows; ++r) {
    float* win = (float*)malloc(sizeof(float) * (size_t)W);
    if (!win) { failed = 1; continue; }
    const float* x = in + r * in_pitch;
    for (int64_t t = 0; t < n; ++t) {
      int64_t s = t - h;
      if (s < 0) s = 0;
      if (s > n - W) s = n - W;
      memcpy(win, x + s, sizeof(float) * (size_t)W);
      qsort(win, (size_t)W, sizeof(float), cmp_float);
      const float m = win[h];
      if (med) med[r * out_pitch + t] = m;
      if (out) out[r * out_pitch + t] = x[t] - m;
    }
    free(win);
  }
  return failed ? ORACLE_ERR_NOMEM : ORACLE_OK;
}

/* C3 + C4, for the series as handed over (no reversal here): edges u[0..M] in input-sample units, u[0] = 0.
 * Returns M through *m_out; edges may be NULL to query M only; cap = capacity of edges in doubles. */
static int resample_edges_core(double F0, double fp, double fpp, double tau0, int64_t n, double* edges, int64_t cap,
                               int64_t* m_out) {
  double u = 0.0;
  int64_t k = 0;
  if (edges) {
    if (cap < 1) return ORACLE_ERR_INVALID;
    edges[0] = 0.0;
  }
  for (;;) {
    const double t = u * tau0;
    const double w = (1.0 + (fp * t) / F0) + (fpp * (t * t)) / (2.0 * F0);
    if (!(w >= 0.5)) return ORACLE_ERR_INVALID;
    const double un = u + w;
    if (!(un <= (double)n)) break;
    ++k;
    if (edges) {
      if (k >= cap) return ORACLE_ERR_INVALID;
      edges[k] = un;
    }
    u = un;
  }
  *m_out = k;
  return ORACLE_OK;
}

/* The parameters the transformation is applied with (Eqs 3.2, 3.5, 3.6): *reversed = 1 if f1 > 0. */
static void resample_params(double f0, double f1, double f2, double tau0, int64_t n, double* F0, double* fp, double* fpp,
                            int* reversed) {
  if (f1 > 0.0) {
    const double T = (double)n * tau0;
    *F0 = (f0 + f1 * T) + (f2 * (T * T)) / 2.0; /* Eq 3.5 */
    *fp = f1 + f2 * T;                          /* Eq 3.6 */
    *fpp = -f2;
    *reversed = 1;
  } else {
    *F0 = f0;
    *fp = -f1; /* Eq 3.2 / text under Eq 3.3 */
    *fpp = -f2;
    *reversed = 0;
  }
}

int oracle_resample_edges(double f0, double f1, double f2, double tau0, int64_t n, double* edges, int64_t cap,
                          int64_t* m_out, int32_t* reversed_out) {
  if (!m_out || n < 1 || !(tau0 > 0.0) || !(f0 > 0.0)) return ORACLE_ERR_INVALID;
  double F0, fp, fpp;
  int rev;
  resample_params(f0, f1, f2, tau0, n, &F0, &fp, &fpp, &rev);
  if (!(F0 > 0.0)) return ORACLE_ERR_INVALID;
  if (reversed_out) *reversed_out = rev;
  return resample_edges_core(F0, fp, fpp, tau0, n, edges, cap, m_out);
}

/* C5-C7.  in: [nrows][in_pitch] (n valid); out: [nrows][out_pitch] (M written, M from oracle_resample_edges). */
int oracle_resample(const float* in, int64_t nrows, int64_t in_pitch, int64_t n, double f0, double f1, double f2,
                    double tau0, float* out, int64_t out_pitch) {
  if (!in || !out || nrows < 0 || in_pitch < n) return ORACLE_ERR_INVALID;
  int64_t M = 0;
  int32_t rev = 0;
  int rc = oracle_resample_edges(f0, f1, f2, tau0, n, NULL, 0, &M, &rev);
  if (rc != ORACLE_OK) return rc;
  if (out_pitch < M) return ORACLE_ERR_INVALID;
  double* u = (double*)malloc(sizeof(double) * (size_t)(M + 1));
  float* xr = (float*)malloc(sizeof(float) * (size_t)n);
  if (!u || !xr) { free(u); free(xr); return ORACLE_ERR_NOMEM; }
  rc = oracle_resample_edges(f0, f1, f2, tau0, n, u, M + 1, &M, &rev);
  for (int64_t r = 0; r < nrows && rc == ORACLE_OK; ++r) {
    const float* x = in + r * in_pitch;
    if (rev) { /* C7: reverse, transform, reverse */
      for (int64_t i = 0; i < n; ++i) xr[i] = x[n - 1 - i];
      x = xr;
    }
    for (int64_t k = 0; k < M; ++k) {
      const double a = u[k], b = u[k + 1];
      const int64_t i0 = (int64_t)floor(a), i1 = (int64_t)floor(b);
      double s;
      if (i0 == i1) {
        s = (double)x[i0] * (b - a);
      } else {
        s = (double)x[i0] * ((double)(i0 + 1) - a);
        for (int64_t i = i0 + 1; i < i1; ++i) s = s + (double)x[i];
        if (i1 < n) s = s + (double)x[i1] * (b - (double)i1);
      }
      out[r * out_pitch + (rev ? M - 1 - k : k)] = (float)s;
    }
  }
  free(u);
  free(xr);
  return rc;
}
