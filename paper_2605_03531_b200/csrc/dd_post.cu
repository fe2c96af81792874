// dd_post.cu -- pulsar-side post-processing of dedispersed time series: the steps the
// thesis applies to a dedispersed series before folding (PAPER.md:421 downsampling, :425 running-median
// de-reddening, :441-484 re-sampling with Eqs 3.1-3.6), for all rows of a DM-time plane at once.
//
// Readings (C1-C7), stated in include/dd.h with each entry point.  All three are exact: the results are
// defined operation by operation in IEEE arithmetic (double sums in index order, order statistics, explicitly
// rounded double products), so they carry the same bits as the plain definitions.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <algorithm>
#include <new>
#include <vector>

#include "dd_internal.h"

namespace dd {

// ------------------------------------------------------------------------------------------------------------
// C1: downsampling.  y[k] = fl32( sum_{i<F} (double)x[k*F+i] ), k < n/F.  One thread per output; the F loads of a
// warp cover 32*F consecutive floats, every line of which is consumed out of L1 within the loop.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dd_downsample_kernel(const float* __restrict__ in, long long in_pitch, long long m,
                                                            int F, float* __restrict__ out, long long out_pitch) {
  const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= m) return;
  const float* x = in + (long long)blockIdx.y * in_pitch + k * F;
  double s = 0.0;
  if ((F & 3) == 0 && ((reinterpret_cast<uintptr_t>(x) & 15u) == 0)) {
    for (int i = 0; i < F; i += 4) {
      const float4 v = __ldg(reinterpret_cast<const float4*>(x + i));
      s = __dadd_rn(s, (double)v.x);
      s = __dadd_rn(s, (double)v.y);
      s = __dadd_rn(s, (double)v.z);
      s = __dadd_rn(s, (double)v.w);
    }
  } else {
    for (int i = 0; i < F; ++i) s = __dadd_rn(s, (double)__ldg(x + i));
  }
  out[(long long)blockIdx.y * out_pitch + k] = __double2float_rn(s);
}

// ------------------------------------------------------------------------------------------------------------
// C2: running median of an odd window W = 2h+1, window start s(t) = min(max(t-h, 0), n-W); out = x - med.
//
// Order statistics are taken on order-preserving 32-bit keys of the floats.  A CTA stages the keys of the samples
// its outputs need (a tile of 8 warps x kMedSeg outputs plus the window halo) in shared memory.  Each warp slides
// one window over its segment and keeps the exact state
//     m = median key,  below = #{key < m},  equal = #{key == m}          (below <= h < below + equal)
// The first window is solved by a radix select on the key bits (32 counting passes over the window, the lanes
// sharing the elements).  A slide by one sample changes below / (below + equal) by at most one, so the median
// either stays or moves to the neighbouring order statistic: the largest key below m or the smallest above it,
// found with its multiplicity by ONE pass of the warp over the window.  No approximation, no assumption on the
// value range.
// ------------------------------------------------------------------------------------------------------------
constexpr int kMedWarps = 8;
constexpr int kMedSeg = 256;  // outputs per warp

__device__ __forceinline__ uint32_t f2key(float v) {
  const uint32_t b = __float_as_uint(v);
  return b ^ ((b >> 31) ? 0xffffffffu : 0x80000000u);
}
__device__ __forceinline__ float key2f(uint32_t k) {
  return __uint_as_float(k ^ ((k >> 31) ? 0x80000000u : 0xffffffffu));
}

__global__ void __launch_bounds__(kMedWarps * 32) dd_running_median_kernel(const float* __restrict__ in, long long in_pitch,
                                                                          long long n, int W, float* __restrict__ med,
                                                                          float* __restrict__ out, long long out_pitch) {
  extern __shared__ uint32_t keys[];  // keys of samples [base, base + span), then the medians of the tile's outputs
  const int h = (W - 1) / 2;
  const long long t0 = (long long)blockIdx.x * (kMedWarps * kMedSeg);
  const int nt = (int)min((long long)kMedWarps * kMedSeg, n - t0);  // outputs of this tile
  const float* x = in + (long long)blockIdx.y * in_pitch;
  // window start of output t (relative to the tile: t = t0 + r) is clamp(t - h, 0, n - W); everything below is in
  // 32-bit offsets from `base`, the window start of the tile's first output
  const long long base = min(max(t0 - h, 0LL), n - W);
  const int smax = (int)(n - W - base);                 // largest window start, relative to base
  const int off = (int)(t0 - h - base);                 // window start of output r before clamping = r + off
  const int span = min(max(nt - 1 + off, 0), smax) + W;  // samples staged
  uint32_t* meds = keys + (kMedWarps * kMedSeg + W);
  for (int i = threadIdx.x; i < span; i += blockDim.x) keys[i] = f2key(__ldg(x + base + i));
  __syncthreads();

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int rs = warp * kMedSeg, re = min(nt, rs + kMedSeg);  // this warp's outputs [rs, re) of the tile
  if (rs < re) {
    // ---- first window of the segment: radix select of the element of rank h
    int s = min(max(rs + off, 0), smax);
    const uint32_t* win = keys + s;
    uint32_t m = 0;
    for (int b = 31; b >= 0; --b) {
      const uint32_t trial = m | (1u << b);
      int c = 0;
      for (int i = lane; i < W; i += 32) c += win[i] < trial;
      c = __reduce_add_sync(0xffffffffu, c);
      if (c <= h) m = trial;  // at most h keys are below `trial`: the rank-h key is >= trial
    }
    int below = 0, equal = 0;
    for (int i = lane; i < W; i += 32) {
      const uint32_t k = win[i];
      below += k < m;
      equal += k == m;
    }
    below = __reduce_add_sync(0xffffffffu, below);
    equal = __reduce_add_sync(0xffffffffu, equal);
    if (lane == 0) meds[rs] = m;
    for (int r = rs + 1; r < re; ++r) {
      const int sn = min(max(r + off, 0), smax);
      if (sn != s) {  // the window moves by one sample: keys[s] leaves, keys[s + W] enters
        const uint32_t ko = keys[s], ki = keys[s + W];
        s = sn;
        below += (int)(ki < m) - (int)(ko < m);
        equal += (int)(ki == m) - (int)(ko == m);
        win = keys + s;
        if (below > h) {  // exactly h+1 keys below m: the median is the largest of them
          uint32_t best = 0;
          int cnt = 0;
          for (int i = lane; i < W; i += 32) {
            const uint32_t k = win[i];
            if (k < m) {
              cnt = k > best ? 1 : cnt + (k == best);
              best = max(best, k);
            }
          }
          const uint32_t all = __reduce_max_sync(0xffffffffu, best);
          cnt = __reduce_add_sync(0xffffffffu, (best == all && cnt > 0) ? cnt : 0);
          m = all;
          equal = cnt;
          below -= cnt;
        } else if (below + equal <= h) {  // exactly h keys at or below m: the median is the smallest key above m
          uint32_t best = 0xffffffffu;
          int cnt = 0;
          for (int i = lane; i < W; i += 32) {
            const uint32_t k = win[i];
            if (k > m) {
              cnt = k < best ? 1 : cnt + (k == best);
              best = min(best, k);
            }
          }
          const uint32_t all = __reduce_min_sync(0xffffffffu, best);
          cnt = __reduce_add_sync(0xffffffffu, (best == all && cnt > 0) ? cnt : 0);
          below += equal;
          m = all;
          equal = cnt;
        }
      }
      if (lane == 0) meds[r] = m;
    }
  }
  __syncthreads();
  // coalesced stores of the tile: median and sample minus median (the sample of output r sits at keys[r + t0 - base])
  float* orow = out ? out + (long long)blockIdx.y * out_pitch + t0 : nullptr;
  float* mrow = med ? med + (long long)blockIdx.y * out_pitch + t0 : nullptr;
  const int xoff = (int)(t0 - base);
  for (int r = threadIdx.x; r < nt; r += blockDim.x) {
    const float mv = key2f(meds[r]);
    if (mrow) mrow[r] = mv;
    if (orow) orow[r] = __fsub_rn(key2f(keys[r + xoff]), mv);
  }
}

// ------------------------------------------------------------------------------------------------------------
// C3-C7: re-sampling.  Bin edges u[0..M] (input-sample units) are built on the host by dd_resample_create from the
// recurrence of Eq 3.3; out[k] = fl32( sum_i x[i] * |[u_k, u_{k+1}) n [i, i+1)| ), accumulated left to right in
// double with explicitly rounded operations (no FMA).  rev: the series is read backwards and written backwards.
// ------------------------------------------------------------------------------------------------------------
constexpr int kResampleRows = 4;  // rows per thread: the bin edges (doubles, shared by all rows) are loaded once for four rows
__global__ void __launch_bounds__(256) dd_resample_kernel(const float* __restrict__ in, long long in_pitch, long long n,
                                                          const double* __restrict__ u, long long M, int rev, long long nrows,
                                                          float* __restrict__ out, long long out_pitch) {
  const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= M) return;
  const double a = u[k], b = u[k + 1];
  const long long i0 = (long long)floor(a), i1 = (long long)floor(b);
  const double f0 = i0 == i1 ? __dsub_rn(b, a) : __dsub_rn((double)(i0 + 1), a);  // weight of the first input bin
  const double f1 = __dsub_rn(b, (double)i1);                                       // weight of the last one (i1 > i0)
  const long long r0 = (long long)blockIdx.y * kResampleRows;
#pragma unroll
  for (int q = 0; q < kResampleRows; ++q) {
    const long long r = r0 + q;
    if (r >= nrows) break;
    const float* x = in + r * in_pitch;
    auto X = [&](long long i) { return (double)__ldg(x + (rev ? n - 1 - i : i)); };
    double s = __dmul_rn(X(i0), f0);
    if (i0 != i1) {
      for (long long i = i0 + 1; i < i1; ++i) s = __dadd_rn(s, X(i));
      if (i1 < n) s = __dadd_rn(s, __dmul_rn(X(i1), f1));
    }
    out[r * out_pitch + (rev ? M - 1 - k : k)] = __double2float_rn(s);
  }
}

}  // namespace dd

struct dd_resample {
  double f0 = 0, f1 = 0, f2 = 0, tsamp = 0;
  int64_t n = 0, M = 0;
  int reversed = 0;
  int device = -1;
  std::vector<double> edges;  // u[0..M]
  double* d_edges = nullptr;
};

namespace {

constexpr int64_t kMaxGridRows = 65535;
inline bool aligned4(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 3u) == 0; }

int check_device(int device) {
  int cur = -1;
  cudaError_t e = cudaGetDevice(&cur);
  if (e != cudaSuccess) return dd::cuda_fail(e, "cudaGetDevice");
  return cur == device ? DD_OK : DD_ERR_DEVICE;
}

// Eq 3.3 laid end to end (reading C3): u_0 = 0, t = u*tau0, w = (1 + (f'*t)/F0) + (f''*(t*t))/(2*F0), u += w while
// u + w <= n.  Plain IEEE double operations in this order (the translation unit is built without FMA contraction).
int build_edges(dd_resample& r) {
  double F0, fp, fpp;
  if (r.f1 > 0.0) {  // Eqs 3.5, 3.6: reversed series
    const double T = (double)r.n * r.tsamp;
    F0 = (r.f0 + r.f1 * T) + (r.f2 * (T * T)) / 2.0;
    fp = r.f1 + r.f2 * T;
    fpp = -r.f2;
    r.reversed = 1;
  } else {  // Eq 3.2
    F0 = r.f0;
    fp = -r.f1;
    fpp = -r.f2;
    r.reversed = 0;
  }
  if (!(F0 > 0.0)) return DD_ERR_INVALID;
  r.edges.clear();
  r.edges.push_back(0.0);
  volatile double u = 0.0;  // volatile: every operation is rounded to double and none is contracted
  for (;;) {
    volatile double t = u * r.tsamp;
    volatile double p1 = fp * t;
    volatile double q1 = p1 / F0;
    volatile double a1 = 1.0 + q1;
    volatile double tt = t * t;
    volatile double p2 = fpp * tt;
    volatile double q2 = p2 / (2.0 * F0);
    volatile double w = a1 + q2;
    if (!(w >= 0.5)) return DD_ERR_INVALID;  // reading C4: a bin is never shorter than half an input sample
    volatile double un = u + w;
    if (!(un <= (double)r.n)) break;
    r.edges.push_back((double)un);
    u = un;
  }
  r.M = (int64_t)r.edges.size() - 1;
  return DD_OK;
}

}  // namespace

extern "C" {

int dd_post_downsample(const float* in_dev, int64_t nrows, int64_t in_pitch, int64_t n, int32_t factor, float* out_dev,
                       int64_t out_pitch, void* cuda_stream) {
  if (!in_dev || !out_dev || nrows < 0 || n < 1 || factor < 1 || in_pitch < n || out_pitch < n / factor) return DD_ERR_INVALID;
  if (!aligned4(in_dev) || !aligned4(out_dev)) return DD_ERR_ALIGN;
  const int64_t m = n / factor;
  if (nrows == 0 || m == 0) return DD_OK;
  for (int64_t r0 = 0; r0 < nrows; r0 += kMaxGridRows) {  // grid.y holds at most 65535 rows
    dim3 grid((unsigned)((m + 255) / 256), (unsigned)std::min<int64_t>(kMaxGridRows, nrows - r0));
    dd::dd_downsample_kernel<<<grid, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        in_dev + r0 * in_pitch, in_pitch, m, factor, out_dev + r0 * out_pitch, out_pitch);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return dd::cuda_fail(e, "dd_downsample_kernel launch");
  }
  return DD_OK;
}

int dd_post_dered(const float* in_dev, int64_t nrows, int64_t in_pitch, int64_t n, int32_t window, float* median_dev,
                  float* out_dev, int64_t out_pitch, void* cuda_stream) {
  if (!in_dev || (!median_dev && !out_dev) || nrows < 0 || n < 1 || window < 1 || (window & 1) == 0 || window > n ||
      window > DD_POST_MAX_WINDOW || in_pitch < n || out_pitch < n)
    return DD_ERR_INVALID;
  if (nrows == 0) return DD_OK;
  const size_t smem = (size_t)(2 * dd::kMedWarps * dd::kMedSeg + window) * sizeof(uint32_t);
  cudaError_t e = cudaFuncSetAttribute(dd::dd_running_median_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
  if (e != cudaSuccess) return dd::cuda_fail(e, "cudaFuncSetAttribute(dd_running_median_kernel)");
  for (int64_t r0 = 0; r0 < nrows; r0 += kMaxGridRows) {
    dim3 grid((unsigned)((n + dd::kMedWarps * dd::kMedSeg - 1) / (dd::kMedWarps * dd::kMedSeg)),
              (unsigned)std::min<int64_t>(kMaxGridRows, nrows - r0));
    dd::dd_running_median_kernel<<<grid, dd::kMedWarps * 32, smem, static_cast<cudaStream_t>(cuda_stream)>>>(
        in_dev + r0 * in_pitch, in_pitch, n, window, median_dev ? median_dev + r0 * out_pitch : nullptr,
        out_dev ? out_dev + r0 * out_pitch : nullptr, out_pitch);
    e = cudaGetLastError();
    if (e != cudaSuccess) return dd::cuda_fail(e, "dd_running_median_kernel launch");
  }
  return DD_OK;
}

static int resample_create(double f0, double f1, double f2, double tsamp_s, int64_t n, bool device, dd_resample_t** out) {
  if (!out) return DD_ERR_INVALID;
  *out = nullptr;
  if (!(f0 > 0.0) || !(tsamp_s > 0.0) || n < 1 || !(f1 == f1) || !(f2 == f2)) return DD_ERR_INVALID;
  dd_resample* r = new (std::nothrow) dd_resample();
  if (!r) return DD_ERR_NOMEM;
  r->f0 = f0, r->f1 = f1, r->f2 = f2, r->tsamp = tsamp_s, r->n = n;
  int rc;
  try {
    rc = build_edges(*r);
  } catch (const std::bad_alloc&) {
    rc = DD_ERR_NOMEM;
  }
  if (rc == DD_OK && device) {
    cudaError_t e = cudaGetDevice(&r->device);
    if (e == cudaSuccess) e = cudaMalloc(&r->d_edges, r->edges.size() * sizeof(double));
    if (e == cudaSuccess)
      e = cudaMemcpy(r->d_edges, r->edges.data(), r->edges.size() * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) rc = dd::cuda_fail(e, "dd_resample_create");
  }
  if (rc != DD_OK) {
    dd_resample_destroy(r);
    return rc;
  }
  *out = r;
  return DD_OK;
}

int dd_resample_create(double f0, double f1, double f2, double tsamp_s, int64_t n, dd_resample_t** out) {
  return resample_create(f0, f1, f2, tsamp_s, n, true, out);
}
int dd_resample_create_host(double f0, double f1, double f2, double tsamp_s, int64_t n, dd_resample_t** out) {
  return resample_create(f0, f1, f2, tsamp_s, n, false, out);
}

int dd_resample_info(const dd_resample_t* r, int64_t* out_len, int32_t* reversed) {
  if (!r) return DD_ERR_INVALID;
  if (out_len) *out_len = r->M;
  if (reversed) *reversed = r->reversed;
  return DD_OK;
}

int dd_resample_get_edges(const dd_resample_t* r, double* host_buf) {
  if (!r || !host_buf) return DD_ERR_INVALID;
  for (size_t i = 0; i < r->edges.size(); ++i) host_buf[i] = r->edges[i];
  return DD_OK;
}

int dd_resample_execute(const dd_resample_t* r, const float* in_dev, int64_t nrows, int64_t in_pitch, float* out_dev,
                        int64_t out_pitch, void* cuda_stream) {
  if (!r || !in_dev || !out_dev || nrows < 0 || in_pitch < r->n || out_pitch < r->M || !r->d_edges) return DD_ERR_INVALID;
  int rc = check_device(r->device);
  if (rc != DD_OK) return rc;
  if (nrows == 0 || r->M == 0) return DD_OK;
  for (int64_t r0 = 0; r0 < nrows; r0 += kMaxGridRows * dd::kResampleRows) {
    const int64_t nr = std::min<int64_t>(kMaxGridRows * dd::kResampleRows, nrows - r0);
    dim3 grid((unsigned)((r->M + 255) / 256), (unsigned)((nr + dd::kResampleRows - 1) / dd::kResampleRows));
    dd::dd_resample_kernel<<<grid, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        in_dev + r0 * in_pitch, in_pitch, r->n, r->d_edges, r->M, r->reversed, nr, out_dev + r0 * out_pitch, out_pitch);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return dd::cuda_fail(e, "dd_resample_kernel launch");
  }
  return DD_OK;
}

int dd_resample_destroy(dd_resample_t* r) {
  if (!r) return DD_OK;
  if (r->d_edges) cudaFree(r->d_edges);
  delete r;
  return DD_OK;
}

}  // extern "C"
