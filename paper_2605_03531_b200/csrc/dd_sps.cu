// dd_sps.cu -- boxcar single-pulse search on the rows of the DM-time plane.
//
// PAPER.md:317-325 (section 2.1): "The SPS module searches for statistically significant single pulses above a
// user-specified threshold using time-domain boxcar filtering."  The readings that make this a definition are
// DESIGN.md B1-B6; per row x[0..n) (integers held in floats):
//   S1 = sum x, S2 = sum x^2 (exact), mean = S1/n, var = S2/n - mean*mean (>= 0), sigma = sqrt(var)   (IEEE double)
//   for width w = 2^k: B[t] = sum_{i<w} x[t+i]; best = max B, tmax = first t reaching it;
//   den = sigma*sqrt(w); snr = sigma > 0 ? (best - w*mean)/den : 0; count = #{t: B[t] > w*mean + threshold*den}
// Everything up to the few double operations per (row, width) is integer arithmetic, and those use explicit
// round-to-nearest intrinsics in the stated order (no FMA contraction), so the results are bit-exact.
//
// One CTA per row.  Phase A: S1, S2 with vector loads and a block reduction.  Phase B: tiles of kTile samples plus
// a halo of the widest filter are staged in shared memory with coalesced loads and turned into an exclusive prefix
// sum P (int64); every boxcar of every width is then P[t+w] - P[t].  The plane is read twice (the second pass mostly from L2): HBM-bound.
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "dd_internal.h"

namespace dd {

constexpr int kSpsThreads = 256;
constexpr int kSpsTile = 4096;   // samples per tile
constexpr int kSpsMaxK = 12;     // widths 1 .. 2048

struct SpsParams {
  const float* plane;  // beam 0 of the range
  long long beam_stride, pitch;
  int n, K;
  double threshold;
  float* snr;
  int32_t* tmax;
  int32_t* count;
  long long row0, rows_per_beam;  // output row = beam*rows_per_beam + row0 + trial
};

__device__ __forceinline__ unsigned long long shfl_down_u64(unsigned long long v, int o) {
  return __shfl_down_sync(0xffffffffu, v, o);
}
// four consecutive prefix sums starting at a multiple of four: one or two vector loads from shared memory
__device__ __forceinline__ void load4(const uint32_t* P, uint32_t (&v)[4]) {
  const uint4 q = *reinterpret_cast<const uint4*>(P);
  v[0] = q.x, v[1] = q.y, v[2] = q.z, v[3] = q.w;
}
__device__ __forceinline__ void load4(const unsigned long long* P, unsigned long long (&v)[4]) {
  const ulonglong2 a = *reinterpret_cast<const ulonglong2*>(P), b = *reinterpret_cast<const ulonglong2*>(P + 2);
  v[0] = a.x, v[1] = a.y, v[2] = b.x, v[3] = b.y;
}

// K = number of widths; WIDE = boxcar sums may reach 2^32 (64-bit prefix sums), else 32-bit modular prefix sums
// (a difference of two of them is the exact boxcar because it is below 2^32).
template <int K, bool WIDE>
__global__ void __launch_bounds__(kSpsThreads) dd_sps_kernel(const SpsParams p) {
  using acc_t = typename std::conditional<WIDE, unsigned long long, uint32_t>::type;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  acc_t* P = reinterpret_cast<acc_t*>(smem_raw);  // [kSpsTile + halo + 1]
  __shared__ unsigned long long red[2][kSpsThreads / 32];
  __shared__ unsigned long long s_thr[kSpsMaxK];  // B >= s_thr  <=>  B > w*mean + threshold*den
  __shared__ double s_wmean[kSpsMaxK], s_den[kSpsMaxK];
  __shared__ double s_sigma;
  __shared__ unsigned long long s_best[kSpsMaxK][kSpsThreads / 32];
  __shared__ int s_tb[kSpsMaxK][kSpsThreads / 32], s_cnt[kSpsMaxK][kSpsThreads / 32];
  __shared__ unsigned long long s_warp_tot[kSpsThreads / 32];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n = p.n;
  const float* x = p.plane + (long long)blockIdx.y * p.beam_stride + (long long)blockIdx.x * p.pitch;

  // ---------------- phase A: exact sums ---------------------------------------------------------------
  unsigned long long s1 = 0, s2 = 0;
  const int n4 = n / 4;  // rows start on 128-byte lines (pitch and range offsets are multiples of 32 floats)
  for (int q = tid; q < n4; q += kSpsThreads) {
    const float4 v = __ldg(reinterpret_cast<const float4*>(x) + q);
    const unsigned long long a = (unsigned long long)v.x, b = (unsigned long long)v.y, c = (unsigned long long)v.z,
                             d = (unsigned long long)v.w;
    s1 += a + b + c + d;
    s2 += a * a + b * b + c * c + d * d;
  }
  for (int t = 4 * n4 + tid; t < n; t += kSpsThreads) {
    const unsigned long long a = (unsigned long long)x[t];
    s1 += a;
    s2 += a * a;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    s1 += shfl_down_u64(s1, o);
    s2 += shfl_down_u64(s2, o);
  }
  if (lane == 0) red[0][warp] = s1, red[1][warp] = s2;
  __syncthreads();
  if (tid == 0) {
    unsigned long long t1 = 0, t2 = 0;
    for (int i = 0; i < kSpsThreads / 32; ++i) t1 += red[0][i], t2 += red[1][i];
    const double dn = (double)n;
    const double mean = __ddiv_rn(__ull2double_rn(t1), dn);
    double var = __dsub_rn(__ddiv_rn(__ull2double_rn(t2), dn), __dmul_rn(mean, mean));
    if (var < 0.0) var = 0.0;
    const double sigma = __dsqrt_rn(var);
    s_sigma = sigma;
    for (int k = 0; k < K; ++k) {
      const double w = (double)(1 << k);
      const double den = __dmul_rn(sigma, __dsqrt_rn(w));
      const double wmean = __dmul_rn(w, mean);
      const double thr = __dadd_rn(wmean, __dmul_rn(p.threshold, den));
      s_den[k] = den;
      s_wmean[k] = wmean;
      // integer form of "B > thr" for integer B: B >= floor(thr) + 1 (everything passes below 0, nothing above 2^62)
      s_thr[k] = thr < 0.0 ? 0ull : thr >= 4.0e18 ? ~0ull : (unsigned long long)floor(thr) + 1ull;
    }
  }
  __syncthreads();

  // ---------------- phase B: boxcars from a prefix sum per tile -------------------------------------------
  constexpr int halo = 1 << (K - 1);
  const int span = kSpsTile + halo;          // prefix entries P[0..span]
  const int per = ((span + kSpsThreads - 1) / kSpsThreads) | 1;
  acc_t best[K], thr[K];
  int tb[K], cnt[K];
#pragma unroll
  for (int k = 0; k < K; ++k) {
    best[k] = 0, tb[k] = 0x7fffffff, cnt[k] = 0;
    // thresholds above the reach of acc_t can never be met: 2^32-1 is below 2^32 only for sums that small
    thr[k] = WIDE ? (acc_t)s_thr[k] : (s_thr[k] > 0xffffffffull ? (acc_t)0xffffffffu : (acc_t)s_thr[k]);
  }
  bool never[K];  // (narrow sums) threshold not representable: count stays 0
#pragma unroll
  for (int k = 0; k < K; ++k) never[k] = !WIDE && s_thr[k] > 0xffffffffull;

  uint32_t* V = reinterpret_cast<uint32_t*>(smem_raw + (size_t)(span + 2) / 2 * 2 * sizeof(acc_t));  // the tile's samples, [span]
  for (int tile0 = 0; tile0 < n; tile0 += kSpsTile) {
    // stage the tile + halo with coalesced loads (samples past the end of the row count as 0)
    for (int i = tid; i < span; i += kSpsThreads) {
      const int t = tile0 + i;
      V[i] = t < n ? (uint32_t)x[t] : 0u;
    }
    __syncthreads();
    // thread-local sums of `per` consecutive samples (per is odd: conflict-free), then a block-wide exclusive
    // scan of the thread totals
    const int i0 = tid * per;
    acc_t loc = 0;
    for (int i = i0; i < i0 + per && i < span; ++i) loc += V[i];
    acc_t inc = loc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const acc_t v = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += v;
    }
    if (lane == 31) s_warp_tot[warp] = inc;
    __syncthreads();
    acc_t base = inc - loc;
    for (int wq = 0; wq < warp; ++wq) base += (acc_t)s_warp_tot[wq];
    if (tid == 0) P[0] = 0;
    for (int i = i0; i < i0 + per && i < span; ++i) {
      base += V[i];
      P[i + 1] = base;
    }
    __syncthreads();
    const bool interior = tile0 + span <= n;  // every window of every width of this tile lies inside the row
    if (interior) {
      // four consecutive samples per thread and step: the prefix sums come in vectors, the maximum of the four
      // boxcars is compared with the running best once, and only a new best looks for its position
      for (int q = tid; q < kSpsTile / 4; q += kSpsThreads) {
        const int tl = 4 * q, t = tile0 + tl;
        acc_t a[4], a4[4];
        load4(P + tl, a);
        load4(P + tl + 4, a4);
#pragma unroll
        for (int k = 0; k < K; ++k) {
          acc_t b[4];
          if (k == 0) {
            b[0] = a[1] - a[0], b[1] = a[2] - a[1], b[2] = a[3] - a[2], b[3] = a4[0] - a[3];
          } else if (k == 1) {
            b[0] = a[2] - a[0], b[1] = a[3] - a[1], b[2] = a4[0] - a[2], b[3] = a4[1] - a[3];
          } else if (k == 2) {
            b[0] = a4[0] - a[0], b[1] = a4[1] - a[1], b[2] = a4[2] - a[2], b[3] = a4[3] - a[3];
          } else {
            acc_t c[4];
            load4(P + tl + (1 << k), c);
            b[0] = c[0] - a[0], b[1] = c[1] - a[1], b[2] = c[2] - a[2], b[3] = c[3] - a[3];
          }
          if (!never[k]) cnt[k] += (b[0] >= thr[k]) + (b[1] >= thr[k]) + (b[2] >= thr[k]) + (b[3] >= thr[k]);
          const acc_t m01 = b[0] > b[1] ? b[0] : b[1], m23 = b[2] > b[3] ? b[2] : b[3], m = m01 > m23 ? m01 : m23;
          if (m > best[k] || tb[k] == 0x7fffffff) {  // rare once the row's level is reached; t increases, so the first maximum is kept
            best[k] = m;
            tb[k] = t + (b[0] == m ? 0 : b[1] == m ? 1 : b[2] == m ? 2 : 3);
          }
        }
      }
    } else {
      for (int tl = tid; tl < kSpsTile; tl += kSpsThreads) {
        const int t = tile0 + tl;
        if (t >= n) break;
        const acc_t p0 = P[tl];
#pragma unroll
        for (int k = 0; k < K; ++k) {
          const int w = 1 << k;
          if (t + w <= n) {
            const acc_t b = P[tl + w] - p0;
            if (b > best[k] || tb[k] == 0x7fffffff) best[k] = b, tb[k] = t;
            cnt[k] += (b >= thr[k]) && !never[k];
          }
        }
      }
    }
    __syncthreads();
  }

  // ---------------- reduce over the block: larger sum wins, ties go to the smaller t ----------------------
#pragma unroll
  for (int k = 0; k < K; ++k) {
    {
      unsigned long long b = best[k];
      int t = tb[k], c = cnt[k];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long ob = shfl_down_u64(b, o);
        const int ot = __shfl_down_sync(0xffffffffu, t, o);
        c += __shfl_down_sync(0xffffffffu, c, o);
        if (ot != 0x7fffffff && (t == 0x7fffffff || ob > b || (ob == b && ot < t))) b = ob, t = ot;
      }
      if (lane == 0) s_best[k][warp] = b, s_tb[k][warp] = t, s_cnt[k][warp] = c;
    }
  }
  __syncthreads();
  if (tid < K) {
    const int k = tid;
    unsigned long long b = 0;
    int t = 0x7fffffff, c = 0;
    for (int i = 0; i < kSpsThreads / 32; ++i) {
      const unsigned long long ob = s_best[k][i];
      const int ot = s_tb[k][i];
      c += s_cnt[k][i];
      if (ot != 0x7fffffff && (t == 0x7fffffff || ob > b || (ob == b && ot < t))) b = ob, t = ot;
    }
    const long long o = ((long long)blockIdx.y * p.rows_per_beam + p.row0 + blockIdx.x) * K + k;
    if (t == 0x7fffffff) {  // filter wider than the row
      p.snr[o] = 0.0f, p.tmax[o] = -1, p.count[o] = 0;
    } else {
      const double sigma = s_sigma;
      p.snr[o] = sigma > 0.0 ? (float)__ddiv_rn(__dsub_rn(__ull2double_rn(b), s_wmean[k]), s_den[k]) : 0.0f;
      p.tmax[o] = t;
      p.count[o] = c;
    }
  }
}

template <int K, bool WIDE>
static cudaError_t launch_sps(const SpsParams& sp, dim3 grid, size_t smem, cudaStream_t stream) {
  // per launch: the attribute is per device and the call is cheap (no static flag: not device- or thread-safe)
  cudaError_t e = cudaFuncSetAttribute(dd_sps_kernel<K, WIDE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
  if (e != cudaSuccess) return e;
  dd_sps_kernel<K, WIDE><<<grid, kSpsThreads, smem, stream>>>(sp);
  return cudaGetLastError();
}

}  // namespace dd

extern "C" {

int dd_sps_rows(const dd_plan_t* p, int64_t* rows) {
  if (!p || !rows) return DD_ERR_INVALID;
  int64_t n = 0;
  for (const auto& r : p->ranges) n += r.ndm;
  *rows = n * p->nbeams;
  return DD_OK;
}

int dd_sps_execute(const dd_plan_t* p, const float* plane_dev, int32_t nwidths, double threshold, float* snr_dev,
                   int32_t* tmax_dev, int32_t* count_dev, void* cuda_stream) {
  if (!p || !plane_dev || !snr_dev || !tmax_dev || !count_dev || nwidths < 1 || nwidths > dd::kSpsMaxK || p->device < 0 ||
      !(threshold >= -1.0e300 && threshold <= 1.0e300))
    return DD_ERR_INVALID;
  int64_t rows_per_beam = 0;
  for (const auto& r : p->ranges) {
    // exactness of S2 = sum x^2 in 64 bits: (largest possible sum)^2 * nout < 2^63
    const double v = (double)p->nchans * (double)((1 << p->in_bits) - 1) * (double)r.decim;
    if (v * v * (double)r.nout >= 9.2e18 || r.nout > 0x7fffffffLL) return DD_ERR_OVERFLOW;
    rows_per_beam += r.ndm;
  }
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  const size_t span = (size_t)dd::kSpsTile + ((size_t)1 << (nwidths - 1));
  int64_t row0 = 0;
  for (const auto& r : p->ranges) {
    dd::SpsParams sp;
    sp.plane = plane_dev + r.offset;
    sp.beam_stride = p->beam_stride;
    sp.pitch = r.pitch;
    sp.n = (int)r.nout;
    sp.K = nwidths;
    sp.threshold = threshold;
    sp.snr = snr_dev;
    sp.tmax = tmax_dev;
    sp.count = count_dev;
    sp.row0 = row0;
    sp.rows_per_beam = rows_per_beam;
    // 32-bit prefix sums while the widest boxcar of the largest possible samples stays below 2^32
    const double vmax = (double)p->nchans * (double)((1 << p->in_bits) - 1) * (double)r.decim;
    const bool wide = vmax * (double)(1 << (nwidths - 1)) >= 4294967296.0;
    const size_t smem = (span + 2) / 2 * 2 * (wide ? 8 : 4) + span * 4;
    const dim3 grid((unsigned)r.ndm, (unsigned)p->nbeams);
    cudaError_t e = cudaErrorInvalidValue;
#define DD_SPS(K_)                                                                                                  \
  case K_:                                                                                                          \
    e = wide ? dd::launch_sps<K_, true>(sp, grid, smem, stream) : dd::launch_sps<K_, false>(sp, grid, smem, stream); \
    break;
    switch (nwidths) {
      DD_SPS(1) DD_SPS(2) DD_SPS(3) DD_SPS(4) DD_SPS(5) DD_SPS(6) DD_SPS(7) DD_SPS(8) DD_SPS(9) DD_SPS(10) DD_SPS(11)
      DD_SPS(12)
    }
#undef DD_SPS
    if (e != cudaSuccess) return dd::cuda_fail(e, "dd_sps_kernel launch");
    row0 += r.ndm;
  }
  return DD_OK;
}

}  // extern "C"
