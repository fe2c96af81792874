// dd_stream.cu -- streaming execution over blocks of spectra with a carried halo.
//
// The thesis's pipeline receives a beam as a sequence of shared-memory blocks (800 or 25600 spectra of 4096
// channels).  A dispersed pulse straddles block boundaries: the sum for output sample t needs
// input up to t + maxd.  A stream keeps the last `hist` input samples on the device, places every new block
// behind them and runs a tail plan (dd_plan_create_tail: each range reads only the end of the window it needs)
// on that window; per range the last block/decim output samples of each trial are new, and consecutive pushes
// join without a gap or an overlap:
//
//   window of push p   = input samples [p*B - hist, (p+1)*B)            (zeros before the first block)
//   rows of range r    = nout_r = B/decim_r + (< 16) samples, the last one being S_r[j][(p+1)*B/k - maxd_r - 1]
//   new samples        = the last B/decim_r of a row  <->  absolute index [p*B/k - maxd_r, (p+1)*B/k - maxd_r)
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <new>
#include <vector>

#include "dd_internal.h"

struct dd_stream {
  dd_plan_t* plan = nullptr;
  int64_t block = 0, hist = 0;  // input samples per push / carried over
  int nbeams = 0, nchans = 0, bytes = 1, layout = 0;
  void* win[2] = {nullptr, nullptr};  // [nbeams][nchans][hist+block] or [nbeams][hist+block][nchans], ping-pong
  int cur = 0;
  int64_t pushes = 0;
  int device = -1;
};

namespace {
constexpr double kDispersion = 4.148808e3;  // s MHz^2 cm^3 / pc, as in dd_plan.cu (BASELINE.json north_star)
inline int64_t round_up(int64_t a, int64_t b) { return (a + b - 1) / b * b; }
}  // namespace

extern "C" {

int dd_stream_create(const dd_config_t* cfg, dd_stream_t** stream_out) {
  if (!cfg || !stream_out) return DD_ERR_INVALID;
  *stream_out = nullptr;
  if (cfg->nchans < 1 || cfg->nsamps < 1 || cfg->nranges < 1 || !cfg->ranges || !(cfg->tsamp_s > 0.0) ||
      !(cfg->chan_width_mhz != 0.0) || !(cfg->f_top_mhz > 0.0))
    return DD_ERR_INVALID;
  // largest delay of any range in input samples: the last trial at the lowest channel (Eq. 1.1)
  const double f_other = cfg->f_top_mhz + (double)(cfg->nchans - 1) * cfg->chan_width_mhz;
  if (!(f_other > 0.0)) return DD_ERR_INVALID;
  const double f_hi = fmax(cfg->f_top_mhz, f_other), f_lo = fmin(cfg->f_top_mhz, f_other);
  int64_t hist = 0;
  int lcm = 1;
  for (int r = 0; r < cfg->nranges; ++r) {
    const dd_range_t& q = cfg->ranges[r];
    if (!(q.decim == 1 || q.decim == 2 || q.decim == 4 || q.decim == 8) || q.ndm < 1) return DD_ERR_INVALID;
    const double dm = q.dm_lo + (double)(q.ndm - 1) * q.dm_step;
    const double x = kDispersion * dm * (1.0 / (f_lo * f_lo) - 1.0 / (f_hi * f_hi)) / (cfg->tsamp_s * q.decim);
    hist = (int64_t)fmax((double)hist, (floor(x + 0.5) + 1.0) * q.decim);  // +1: slack against the plan's own rounding
    lcm = q.decim > lcm ? q.decim : lcm;
  }
  if (cfg->nsamps % lcm != 0) return DD_ERR_INVALID;  // a block must hold whole decimated samples of every range
  hist = round_up(hist, 64);                           // keeps rows 16-byte aligned and every decimation phase
  dd_stream* s = new (std::nothrow) dd_stream();
  if (!s) return DD_ERR_NOMEM;
  s->block = cfg->nsamps;
  s->hist = hist;
  s->nbeams = cfg->nbeams;
  s->nchans = cfg->nchans;
  s->bytes = cfg->in_bits / 8;
  s->layout = cfg->in_layout;
  dd_config_t inner = *cfg;
  inner.nsamps = hist + cfg->nsamps;
  // only the last block/decim (+ < 16) samples of every row are computed: no work is repeated between pushes
  int rc = dd_plan_create_tail(&inner, cfg->nsamps, &s->plan);
  if (rc != DD_OK) {
    delete s;
    return rc;
  }
  const size_t wbytes = (size_t)s->nbeams * s->nchans * (size_t)(hist + s->block) * s->bytes;
  for (int i = 0; i < 2; ++i) {
    if (cudaMalloc(&s->win[i], wbytes) != cudaSuccess || cudaMemset(s->win[i], 0, wbytes) != cudaSuccess) {
      cudaGetLastError();
      dd_stream_destroy(s);
      return DD_ERR_NOMEM;
    }
  }
  cudaError_t e = cudaDeviceSynchronize();
  if (e == cudaSuccess) e = cudaGetDevice(&s->device);
  if (e != cudaSuccess) {
    dd_stream_destroy(s);
    return dd::cuda_fail(e, "dd_stream_create");
  }
  *stream_out = s;
  return DD_OK;
}

int dd_stream_push(dd_stream_t* s, const void* block_dev, float* out_dev, void* cuda_stream) {
  if (!s || !block_dev || !out_dev) return DD_ERR_INVALID;
  {
    int cur = -1;
    cudaError_t ce = cudaGetDevice(&cur);
    if (ce != cudaSuccess) return dd::cuda_fail(ce, "cudaGetDevice");
    if (cur != s->device) return DD_ERR_DEVICE;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int64_t W = s->hist + s->block;
  char* win = static_cast<char*>(s->win[s->cur]);
  char* nxt = static_cast<char*>(s->win[s->cur ^ 1]);
  cudaError_t e;
  if (s->layout == DD_LAYOUT_SPECTRUM_MAJOR) {
    // per beam: [W][nchans]; history first, the block behind it
    const size_t spec = (size_t)s->nchans * s->bytes;
    e = cudaMemcpy2DAsync(win + (size_t)s->hist * spec, (size_t)W * spec, block_dev, (size_t)s->block * spec,
                          (size_t)s->block * spec, s->nbeams, cudaMemcpyDeviceToDevice, st);
  } else {
    // rows of `block` samples into rows of W samples, behind the history
    e = cudaMemcpy2DAsync(win + (size_t)s->hist * s->bytes, (size_t)W * s->bytes, block_dev, (size_t)s->block * s->bytes,
                          (size_t)s->block * s->bytes, (size_t)s->nbeams * s->nchans, cudaMemcpyDeviceToDevice, st);
  }
  if (e != cudaSuccess) return dd::cuda_fail(e, "cudaMemcpy2DAsync(block into window)");
  int rc = dd_execute(s->plan, win, out_dev, cuda_stream);
  if (rc != DD_OK) return rc;
  // carry: the last `hist` samples of this window become the head of the next one (other buffer: no overlap)
  if (s->layout == DD_LAYOUT_SPECTRUM_MAJOR) {
    const size_t spec = (size_t)s->nchans * s->bytes;
    e = cudaMemcpy2DAsync(nxt, (size_t)W * spec, win + (size_t)s->block * spec, (size_t)W * spec, (size_t)s->hist * spec,
                          s->nbeams, cudaMemcpyDeviceToDevice, st);
  } else {
    e = cudaMemcpy2DAsync(nxt, (size_t)W * s->bytes, win + (size_t)s->block * s->bytes, (size_t)W * s->bytes,
                          (size_t)s->hist * s->bytes, (size_t)s->nbeams * s->nchans, cudaMemcpyDeviceToDevice, st);
  }
  if (e != cudaSuccess) return dd::cuda_fail(e, "cudaMemcpy2DAsync(carry)");
  s->cur ^= 1;
  ++s->pushes;
  return DD_OK;
}

const dd_plan_t* dd_stream_plan(const dd_stream_t* s) { return s ? s->plan : nullptr; }

int dd_stream_info(const dd_stream_t* s, int64_t* block_samples, int64_t* hist_samples, int64_t* pushes) {
  if (!s) return DD_ERR_INVALID;
  if (block_samples) *block_samples = s->block;
  if (hist_samples) *hist_samples = s->hist;
  if (pushes) *pushes = s->pushes;
  return DD_OK;
}

int dd_stream_destroy(dd_stream_t* s) {
  if (!s) return DD_OK;
  for (int i = 0; i < 2; ++i)
    if (s->win[i]) cudaFree(s->win[i]);
  if (s->plan) dd_plan_destroy(s->plan);
  delete s;
  return DD_OK;
}

}  // extern "C"
