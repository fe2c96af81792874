// dd_sps.cu -- boxcar single-pulse search on the rows of the DM-time plane.
//
// PAPER.md:317-325 (section 2.1): "The SPS module searches for statistically significant single pulses above a
// user-specified threshold using time-domain boxcar filtering.  ...  The list of candidates thus generated is
// filtered ..."  The readings that make this a definition are DESIGN.md B1-B6; per row x[0..n) (integers in floats):
//   S1 = sum x, S2 = sum x^2 (exact), mean = S1/n, var = S2/n - mean*mean (>= 0), sigma = sqrt(var)   (IEEE double)
//   for width w = 2^k: B[t] = sum_{i<w} x[t+i]; best = max B, tmax = first t reaching it;
//   den = sigma*sqrt(w); snr = sigma > 0 ? (best - w*mean)/den : 0; count = #{t: B[t] > w*mean + threshold*den}
//   candidate list: every (row, k, t) with B[t] > w*mean + threshold*den and its snr, ordered by row, k, t.
// Everything up to the few double operations per (row, width) is integer arithmetic, and those use explicit
// round-to-nearest intrinsics in the stated order (no FMA contraction), so the results are bit-exact.
//
// dd_sps_kernel: one CTA per row.  Phase A: S1, S2 (vector loads, block reduction) -- skipped when dd_execute has
// already accumulated them in its epilogue (dd_plan_set_row_stats), which leaves ONE pass over the plane.  Phase B:
// tiles of kSpsTile samples plus a halo of the widest filter are staged in shared memory and turned into a prefix sum
// P; every boxcar of every width is P[t+w] - P[t], four consecutive samples per thread and step.  Samples above the
// threshold are rare, so the loop tests the maximum of the four against the threshold and counts one by one only then.
// dd_sps_fill_kernel: the candidate list.  Rows without a candidate leave at once; the others redo their boxcars and
// write (row, k, t, snr) in order at the offsets an exclusive scan of the counts has fixed (dd_sps_scan_kernel).
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <type_traits>
#include <vector>

#include "dd_internal.h"
#include "dd_ptx.cuh"

namespace dd {

constexpr int kSpsThreads = 256;
constexpr int kSpsTile = 4096;   // samples per tile
constexpr int kSpsMaxK = 12;     // widths 1 .. 2048
constexpr int kSpsMaxRanges = 8;  // ranges one launch of the barrier-free kernel can cover

struct SpsParams {
  const float* plane;  // beam 0 of the range
  long long beam_stride, pitch;
  int n, K;
  double threshold;
  float* snr;
  int32_t* tmax;
  int32_t* count;
  long long row0, rows_per_beam;  // output row = beam*rows_per_beam + row0 + trial
  const unsigned long long* stats;  // [rows][2] = S1, S2 per output row, or nullptr (phase A computes them)
  // dd_sps_warp_kernel: several ranges in one launch, longest rows first (blockIdx.x runs over the rows of rg[0], rg[1], ...)
  int nr;
  struct Range {
    long long plane_off, pitch, row0;  // floats from `plane` to the range's first row; row pitch; first output row
    int n, ndm;
  } rg[kSpsMaxRanges];
  // candidate list (dd_sps_fill_kernel)
  const long long* offsets;  // [rows*K + 1] exclusive scan of count
  dd_sps_cand_t* cand;
  long long max_cands;
};

// dynamic shared memory: P[span + 1] prefix sums, then (16-byte aligned) V[span] samples
__host__ __device__ inline size_t sps_v_offset(size_t span, size_t acc_bytes) { return ((span + 1) * acc_bytes + 127) / 128 * 128; }

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

// Row statistics and the per-width constants, by one thread, in the operation order of the definition.
struct SpsRowConsts {
  unsigned long long thr[kSpsMaxK];  // B >= thr  <=>  B > w*mean + threshold*den   (integer B)
  double wmean[kSpsMaxK], den[kSpsMaxK];
  double sigma;
};
__device__ __forceinline__ void sps_row_consts(unsigned long long t1, unsigned long long t2, int n, int K, double threshold,
                                               SpsRowConsts& c) {
  const double dn = (double)n;
  const double mean = __ddiv_rn(__ull2double_rn(t1), dn);
  double var = __dsub_rn(__ddiv_rn(__ull2double_rn(t2), dn), __dmul_rn(mean, mean));
  if (var < 0.0) var = 0.0;
  const double sigma = __dsqrt_rn(var);
  c.sigma = sigma;
  for (int k = 0; k < K; ++k) {
    const double w = (double)(1 << k);
    const double den = __dmul_rn(sigma, __dsqrt_rn(w));
    const double wmean = __dmul_rn(w, mean);
    const double thr = __dadd_rn(wmean, __dmul_rn(threshold, den));
    c.den[k] = den;
    c.wmean[k] = wmean;
    // integer form of "B > thr" for integer B: B >= floor(thr) + 1 (everything passes below 0, nothing above 2^62)
    c.thr[k] = thr < 0.0 ? 0ull : thr >= 4.0e18 ? ~0ull : (unsigned long long)floor(thr) + 1ull;
  }
}
__device__ __forceinline__ float sps_snr(unsigned long long b, const SpsRowConsts& c, int k) {
  return c.sigma > 0.0 ? (float)__ddiv_rn(__dsub_rn(__ull2double_rn(b), c.wmean[k]), c.den[k]) : 0.0f;
}

// Phase A: exact S1, S2 of the row (all threads call; result valid in thread 0 after the reduction through `red`).
__device__ __forceinline__ void sps_row_sums(const float* x, int n, unsigned long long (&red)[2][kSpsThreads / 32],
                                             unsigned long long& t1, unsigned long long& t2) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
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
  t1 = t2 = 0;
  if (tid == 0)
    for (int i = 0; i < kSpsThreads / 32; ++i) t1 += red[0][i], t2 += red[1][i];
}

// Stage samples [tile0, tile0 + span) of the row (zeros past its end) and build the exclusive prefix sum P[0..span].
// V: [PER * kSpsThreads] scratch (>= span); PER = odd number of consecutive samples per thread (bank-conflict free),
// compile-time so that both loops unroll and the samples stay in registers between the two.
template <typename acc_t, int PER>
__device__ __forceinline__ void sps_build_prefix(const float* x, int n, int tile0, int span, uint32_t* V, acc_t* P,
                                                 unsigned long long* warp_tot) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int padded = PER * kSpsThreads;
  if (tile0 + span <= n && (tile0 & 3) == 0) {  // interior: vector loads
    for (int q = tid; q < span / 4; q += kSpsThreads) {
      const float4 v = __ldg(reinterpret_cast<const float4*>(x + tile0) + q);
      *reinterpret_cast<uint4*>(V + 4 * q) = make_uint4((uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w);
    }
    for (int i = span / 4 * 4 + tid; i < padded; i += kSpsThreads) V[i] = i < span ? (uint32_t)x[tile0 + i] : 0u;
  } else {
    for (int i = tid; i < padded; i += kSpsThreads) {
      const int t = tile0 + i;
      V[i] = (i < span && t < n) ? (uint32_t)x[t] : 0u;
    }
  }
  __syncthreads();
  const int i0 = tid * PER;
  uint32_t v[PER];
  acc_t loc = 0;
#pragma unroll
  for (int i = 0; i < PER; ++i) {
    v[i] = V[i0 + i];
    loc += v[i];
  }
  acc_t inc = loc;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const acc_t u = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += u;
  }
  if (lane == 31) warp_tot[warp] = inc;
  __syncthreads();
  acc_t base = inc - loc;
  for (int wq = 0; wq < warp; ++wq) base += (acc_t)warp_tot[wq];
  if (tid == 0) P[0] = 0;
#pragma unroll
  for (int i = 0; i < PER; ++i) {
    base += v[i];
    if (i0 + i < span) P[i0 + i + 1] = base;
  }
  __syncthreads();
}
// The same from a tile of raw floats already in shared memory (bulk-copied there): X[i] = sample tile0 + i for
// i < loaded, anything beyond counts as zero.
template <typename acc_t, int PER>
__device__ __forceinline__ void sps_build_prefix_raw(const float* X, int valid, int span, acc_t* P, unsigned long long* warp_tot) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int i0 = tid * PER;
  uint32_t v[PER];
  acc_t loc = 0;
#pragma unroll
  for (int i = 0; i < PER; ++i) {
    v[i] = i0 + i < valid ? (uint32_t)X[i0 + i] : 0u;  // valid = samples of this tile that exist (row end) and were copied
    loc += v[i];
  }
  acc_t inc = loc;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const acc_t u = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += u;
  }
  if (lane == 31) warp_tot[warp] = inc;
  __syncthreads();
  acc_t base = inc - loc;
  for (int wq = 0; wq < warp; ++wq) base += (acc_t)warp_tot[wq];
  if (tid == 0) P[0] = 0;
#pragma unroll
  for (int i = 0; i < PER; ++i) {
    base += v[i];
    if (i0 + i < span) P[i0 + i + 1] = base;
  }
  __syncthreads();
}
// samples per thread in the prefix build: odd, PER * kSpsThreads >= kSpsTile + 2^(K-1)
__host__ __device__ constexpr int sps_per(int K) { return ((kSpsTile + (1 << (K - 1)) + kSpsThreads - 1) / kSpsThreads) | 1; }

// K = number of widths; WIDE = boxcar sums may reach 2^32 (64-bit prefix sums), else 32-bit modular prefix sums
// (a difference of two of them is the exact boxcar because it is below 2^32).
template <int K, bool WIDE>
__global__ void __launch_bounds__(kSpsThreads, WIDE ? 2 : (K <= 8 ? 4 : 3)) dd_sps_kernel(const SpsParams p) {
  using acc_t = typename std::conditional<WIDE, unsigned long long, uint32_t>::type;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  acc_t* P = reinterpret_cast<acc_t*>(smem_raw);  // [kSpsTile + halo + 1]
  __shared__ unsigned long long red[2][kSpsThreads / 32];
  __shared__ SpsRowConsts s_c;
  __shared__ __align__(8) unsigned long long s_bar[2];  // "tile landed" barriers of the two raw-sample buffers
  __shared__ unsigned long long s_best[kSpsMaxK][kSpsThreads / 32];
  __shared__ int s_tb[kSpsMaxK][kSpsThreads / 32];
  __shared__ int s_count[kSpsMaxK];  // boxcars at or above the threshold, whole row (rare: shared-memory atomics)
  __shared__ unsigned long long s_warp_tot[kSpsThreads / 32];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n = p.n;
  const float* x = p.plane + (long long)blockIdx.y * p.beam_stride + (long long)blockIdx.x * p.pitch;
  const long long orow = (long long)blockIdx.y * p.rows_per_beam + p.row0 + blockIdx.x;

  // ---------------- phase A: exact sums (or the ones dd_execute left behind) ------------------------------
  if (tid < kSpsMaxK) s_count[tid] = 0;
  if (p.stats) {
    if (tid == 0) sps_row_consts(p.stats[2 * orow], p.stats[2 * orow + 1], n, K, p.threshold, s_c);
  } else {
    unsigned long long t1, t2;
    sps_row_sums(x, n, red, t1, t2);
    if (tid == 0) sps_row_consts(t1, t2, n, K, p.threshold, s_c);
  }
  __syncthreads();

  // ---------------- phase B: boxcars from a prefix sum per tile -------------------------------------------
  constexpr int halo = 1 << (K - 1);
  const int span = kSpsTile + halo;          // prefix entries P[0..span]
  // per thread and width: best1 = (largest boxcar seen) + 1, 0 = none yet; tq >= 0: start of the group of four samples
  // that holds it, exact position still to be looked up; tq < 0: -(t + 2) with t where it was first seen (-1: nowhere)
  acc_t best1[K], thr[K];
  int tq[K];
#pragma unroll
  for (int k = 0; k < K; ++k) {
    best1[k] = 0, tq[k] = -1;
    // (narrow sums) boxcars stay below 2^32 - 1 (dd_sps_execute picks WIDE otherwise), so a threshold that does not fit
    // 32 bits is replaced by 2^32 - 1, which no boxcar reaches
    thr[k] = WIDE ? (acc_t)s_c.thr[k] : (s_c.thr[k] > 0xffffffffull ? (acc_t)0xffffffffu : (acc_t)s_c.thr[k]);
  }

  // Raw tiles (kSpsTile + halo floats, rounded up to 16 bytes, clipped to the row's pitch) are brought in by 1-D bulk
  // copies (TMA) into two buffers: the copy of tile i+1 is in flight while tile i is filtered.
  constexpr int kPer = sps_per(K);
  float* const X0 = reinterpret_cast<float*>(smem_raw + sps_v_offset(span, sizeof(acc_t)));  // buffer b at X0 + b*kXstride
  constexpr int kXstride = kPer * kSpsThreads;
  const uint32_t bar0 = smem_u32(&s_bar[0]);
  auto tile_floats = [&](int tile0) { return min((span + 3) & ~3, ((n + 3) & ~3) - tile0); };  // rows are padded to 32 floats
  if (tid == 0) {
    mbar_init(bar0, 1);
    mbar_init(bar0 + 8, 1);
    fence_barrier_init();
    const uint32_t bytes = (uint32_t)tile_floats(0) * 4u;
    mbar_arrive_expect_tx(bar0, bytes);
    bulk_copy_g2s(smem_u32(X0), x, bytes, bar0);
  }
  __syncthreads();
  uint32_t phase = 0;  // bit b: parity to wait for on buffer b
  // the four boxcars of width 2^k that start at tl .. tl+3
  auto boxcars4 = [&](int k, int tl, const acc_t (&a)[4], const acc_t (&a4)[4], acc_t (&b)[4]) {
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
  };
  int buf = 0;
  for (int tile0 = 0; tile0 < n; tile0 += kSpsTile, buf ^= 1) {
    if (tid == 0 && tile0 + kSpsTile < n) {  // next tile into the other buffer (its last readers passed the barrier below)
      const uint32_t bytes = (uint32_t)tile_floats(tile0 + kSpsTile) * 4u;
      mbar_arrive_expect_tx(bar0 + 8u * (buf ^ 1), bytes);
      bulk_copy_g2s(smem_u32(X0 + (buf ^ 1) * kXstride), x + tile0 + kSpsTile, bytes, bar0 + 8u * (buf ^ 1));
    }
    mbar_wait(bar0 + 8u * buf, (phase >> buf) & 1u);
    phase ^= 1u << buf;
    sps_build_prefix_raw<acc_t, kPer>(X0 + buf * kXstride, min(span, n - tile0), span, P, s_warp_tot);
    // groups of four samples whose windows of every width lie inside the row take the vector path; the last
    // halo + 3 samples of the row are done one by one below
    const int nfast = min(kSpsTile, max(0, n - halo - 3 - tile0 + 1)) / 4;  // groups q < nfast: tile0 + 4q + 3 + halo <= n
    {
      // Four consecutive samples per thread and step; the prefix sums come in vectors.  Only the maximum m of the four
      // boxcars is looked at in the loop: "m reaches the threshold" sets a bit (rare: those groups are counted one by
      // one after the loop) and "m beats the best" records the group (its exact position is looked up after the loop).
      uint32_t hits = 0;
      for (int q = tid; q < nfast; q += kSpsThreads) {
        const int tl = 4 * q;
        acc_t a[4], a4[4];
        load4(P + tl, a);
        load4(P + tl + 4, a4);
#pragma unroll
        for (int k = 0; k < K; ++k) {
          acc_t b[4];
          boxcars4(k, tl, a, a4, b);
          const acc_t m01 = b[0] > b[1] ? b[0] : b[1], m23 = b[2] > b[3] ? b[2] : b[3], m = m01 > m23 ? m01 : m23;
          if (m >= thr[k]) hits |= 1u << k;
          if (m >= best1[k]) {  // m > best; t increases, so the first maximum is kept
            best1[k] = m + 1;
            tq[k] = tile0 + tl;
          }
        }
      }
      if (hits) {  // count the boxcars at or above the threshold in this thread's groups of the widths that had one
        for (int q = tid; q < nfast; q += kSpsThreads) {
          const int tl = 4 * q;
          acc_t a[4], a4[4];
          load4(P + tl, a);
          load4(P + tl + 4, a4);
#pragma unroll
          for (int k = 0; k < K; ++k) {
            if (!(hits & (1u << k))) continue;
            acc_t b[4];
            boxcars4(k, tl, a, a4, b);
            const int c = (b[0] >= thr[k]) + (b[1] >= thr[k]) + (b[2] >= thr[k]) + (b[3] >= thr[k]);
            if (c) atomicAdd(&s_count[k], c);
          }
        }
      }
#pragma unroll
      for (int k = 0; k < K; ++k) {
        if (tq[k] >= 0) {  // a new best in this tile: which of the four was it
          const int tl = tq[k] - tile0;
          acc_t a[4], a4[4], b[4];
          load4(P + tl, a);
          load4(P + tl + 4, a4);
          boxcars4(k, tl, a, a4, b);
          const acc_t m = best1[k] - 1;
          tq[k] = -(tq[k] + (b[0] == m ? 0 : b[1] == m ? 1 : b[2] == m ? 2 : 3) + 2);
        }
      }
    }
    if (4 * nfast < kSpsTile) {  // the end of the row: windows checked one by one
      for (int tl = 4 * nfast + tid; tl < kSpsTile; tl += kSpsThreads) {
        const int t = tile0 + tl;
        if (t >= n) break;
        const acc_t p0 = P[tl];
#pragma unroll
        for (int k = 0; k < K; ++k) {
          const int w = 1 << k;
          if (t + w <= n) {
            const acc_t b = P[tl + w] - p0;
            if (b >= best1[k]) best1[k] = b + 1, tq[k] = -(t + 2);
            if (b >= thr[k]) atomicAdd(&s_count[k], 1);
          }
        }
      }
    }
    __syncthreads();
  }

  // ---------------- reduce over the block: larger sum wins, ties go to the smaller t ----------------------
#pragma unroll
  for (int k = 0; k < K; ++k) {
    unsigned long long b = best1[k];  // (best + 1; 0 = this thread saw no window of this width)
    int t = best1[k] ? -(tq[k] + 2) : 0x7fffffff;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const unsigned long long ob = shfl_down_u64(b, o);
      const int ot = __shfl_down_sync(0xffffffffu, t, o);
      if (ob > b || (ob == b && ot < t)) b = ob, t = ot;
    }
    if (lane == 0) s_best[k][warp] = b, s_tb[k][warp] = t;
  }
  __syncthreads();
  if (tid < K) {
    const int k = tid;
    unsigned long long b = 0;
    int t = 0x7fffffff;
    const int c = s_count[k];
    for (int i = 0; i < kSpsThreads / 32; ++i) {
      const unsigned long long ob = s_best[k][i];
      const int ot = s_tb[k][i];
      if (ob > b || (ob == b && ot < t)) b = ob, t = ot;
    }
    const long long o = orow * K + k;
    if (b == 0) {  // filter wider than the row
      p.snr[o] = 0.0f, p.tmax[o] = -1, p.count[o] = 0;
    } else {
      p.snr[o] = sps_snr(b - 1, s_c, k);
      p.tmax[o] = t;
      p.count[o] = c;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// dd_sps_warp_kernel: the search for K <= 9 widths and 32-bit sums, WITHOUT block barriers in the tile loop.  One CTA
// per row as above, but every warp works on tiles of its own (tile t of kSpsWarpTile samples goes to warp t mod 8): its
// raw samples arrive by bulk copies into one of the warp's two buffers, the warp turns them into the prefix sum IN PLACE
// (lane l owns PER consecutive samples, PER odd: conflict-free; a warp scan joins the lanes) and filters it; only
// __syncwarp orders the phases.  (ncu on the block-wide kernel: 3.1 barrier stalls per issued instruction, the shared-
// memory data pipe at 59 %.)  Same arithmetic, same results.
// ------------------------------------------------------------------------------------------------
constexpr int kSpsWarpTile = 1024;
__host__ __device__ constexpr int sps_warp_words(int K) {  // words of one warp buffer: prefix entries 0 .. span, 16-byte multiple
  return (kSpsWarpTile + (1 << (K - 1)) + 1 + 3) / 4 * 4;
}
__host__ __device__ constexpr int sps_warp_per(int K) { return ((kSpsWarpTile + (1 << (K - 1)) + 31) / 32) | 1; }

template <int K>
__global__ void __launch_bounds__(kSpsThreads, 3) dd_sps_warp_kernel(const SpsParams p) {
  using acc_t = uint32_t;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ unsigned long long red[2][kSpsThreads / 32];
  __shared__ SpsRowConsts s_c;
  __shared__ __align__(8) unsigned long long s_bar[kSpsThreads / 32][2];
  __shared__ unsigned long long s_best[kSpsMaxK][kSpsThreads / 32];
  __shared__ int s_tb[kSpsMaxK][kSpsThreads / 32];
  __shared__ int s_count[kSpsMaxK];
  __shared__ unsigned int s_blk[kSpsMaxK];  // (largest boxcar any warp has published so far) + 1, 0 = none

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // which range this row belongs to: the ranges are listed longest rows first, and CTAs start in blockIdx order, so the
  // short rows fill the end of the launch (one launch per range ends in a partial wave of CTAs each time: 10 % on config 3)
  int rr = 0, row = (int)blockIdx.x;
  while (rr + 1 < p.nr && row >= p.rg[rr].ndm) row -= p.rg[rr].ndm, ++rr;
  const int n = p.rg[rr].n;
  const float* x = p.plane + (long long)blockIdx.y * p.beam_stride + p.rg[rr].plane_off + (long long)row * p.rg[rr].pitch;
  const long long orow = (long long)blockIdx.y * p.rows_per_beam + p.rg[rr].row0 + row;

  if (tid < kSpsMaxK) s_count[tid] = 0, s_blk[tid] = 0;
  if (lane < kSpsMaxK) s_best[lane][warp] = 0, s_tb[lane][warp] = 0x7fffffff;  // this warp's record per width
  if (p.stats) {
    if (tid == 0) sps_row_consts(p.stats[2 * orow], p.stats[2 * orow + 1], n, K, p.threshold, s_c);
  } else {
    unsigned long long t1, t2;
    sps_row_sums(x, n, red, t1, t2);
    if (tid == 0) sps_row_consts(t1, t2, n, K, p.threshold, s_c);
  }
  const uint32_t bar0 = smem_u32(&s_bar[warp][0]);
  if (lane == 0) {
    mbar_init(bar0, 1);
    mbar_init(bar0 + 8, 1);
    fence_barrier_init();
  }
  __syncthreads();

  constexpr int halo = 1 << (K - 1);
  constexpr int span = kSpsWarpTile + halo;
  constexpr int kWords = sps_warp_words(K);
  constexpr int PER = sps_warp_per(K);
  uint32_t* const buf0 = reinterpret_cast<uint32_t*>(smem_raw) + (size_t)warp * 2 * kWords;

  // Records live in shared memory, one per warp and width: s_best = (largest boxcar among the warp's windows) + 1 and
  // s_tb = where it was first seen; they change a few times per row, so the filter loop carries no position.  seen[k]
  // (the same in every lane) is what a later tile of this warp has to BEAT to matter: the warp's own record (a tie with
  // it lies later in the row), or one less than the largest value it has seen published by another warp -- a tie with
  // another warp's record must still be recorded, because that warp's window may lie later in the row (warps run their
  // tiles at their own pace: a warp can be told of a record from a tile behind the one it filters next).  A stale
  // value is only smaller, i.e. costs a lookup, never a result.
  acc_t seen[K], thr[K];
#pragma unroll
  for (int k = 0; k < K; ++k) {
    seen[k] = 0;
    thr[k] = s_c.thr[k] > 0xffffffffull ? (acc_t)0xffffffffu : (acc_t)s_c.thr[k];
  }
  // publish (boxcar + 1) of a candidate record; true if no warp has published a larger one (equal ones are both kept:
  // the final reduction takes the smaller position)
  auto publish = [&](int k, acc_t w1) -> bool {
    unsigned int old = 0;
    if (lane == 0) old = atomicMax(&s_blk[k], w1);
    old = __shfl_sync(0xffffffffu, old, 0);
    seen[k] = old > w1 ? old - 1 : w1;
    return w1 >= old;
  };
  auto tile_floats = [&](int tile0) { return min((span + 3) & ~3, ((n + 3) & ~3) - tile0); };
  auto issue = [&](int tile0, int b) {  // lane 0: bulk copy of the tile's raw samples into buffer b of this warp
    const uint32_t bytes = (uint32_t)tile_floats(tile0) * 4u;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the buffer was last touched by ordinary loads / stores
    mbar_arrive_expect_tx(bar0 + 8u * b, bytes);
    bulk_copy_g2s(smem_u32(buf0 + b * kWords), x + tile0, bytes, bar0 + 8u * b);
  };
  const int ntiles = (n + kSpsWarpTile - 1) / kSpsWarpTile;
  if (lane == 0 && warp < ntiles) issue(warp * kSpsWarpTile, 0);
  auto boxcars4 = [&](const acc_t* P, int k, int tl, const acc_t (&a)[4], const acc_t (&a4)[4], acc_t (&b)[4]) {
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
  };

  int it = 0;
  for (int t = warp; t < ntiles; t += kSpsThreads / 32, ++it) {
    const int b = it & 1;
    const int tile0 = t * kSpsWarpTile;
    if (lane == 0 && t + kSpsThreads / 32 < ntiles) issue((t + kSpsThreads / 32) * kSpsWarpTile, b ^ 1);
    mbar_wait(bar0 + 8u * b, (uint32_t)(it >> 1) & 1u);
    uint32_t* const P = buf0 + b * kWords;            // raw floats now, prefix sums after the next block
    const float* const X = reinterpret_cast<const float*>(P);
    {
      const int valid = min(span, n - tile0), i0 = lane * PER;
      uint32_t v[PER];
      acc_t loc = 0;
#pragma unroll
      for (int i = 0; i < PER; ++i) {
        v[i] = i0 + i < valid ? (uint32_t)X[i0 + i] : 0u;
        loc += v[i];
      }
      acc_t inc = loc;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const acc_t u = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += u;
      }
      acc_t base = inc - loc;
      __syncwarp();  // every lane has read its samples: the prefix may overwrite them
      if (lane == 0) P[0] = 0;
#pragma unroll
      for (int i = 0; i < PER; ++i) {
        base += v[i];
        if (i0 + i < span) P[i0 + i + 1] = base;
      }
      __syncwarp();
    }
    const int nfast = min(kSpsWarpTile, max(0, n - halo - 3 - tile0 + 1)) / 4;
    if (nfast > 0) {
      // Four consecutive samples per lane and step; the loop only keeps, per width, the largest boxcar the lane has seen
      // in this tile (a fused subtract-max and a three-way max per pair).  Per tile and width the warp's maximum (REDUX)
      // then decides, uniformly, whether the lanes count windows at or above the threshold (rare) or look up the
      // position of a new record (a few times per row).
      acc_t tmax[K];
#pragma unroll
      for (int k = 0; k < K; ++k) tmax[k] = 0;
#pragma unroll 4  // (independent groups in flight: 8 widths 1.28 -> 1.22 ms)
      for (int q = lane; q < nfast; q += 32) {
        const int tl = 4 * q;
        acc_t a[4], a4[4];
        load4(P + tl, a);
        load4(P + tl + 4, a4);
#pragma unroll
        for (int k = 0; k < K; ++k) {
          acc_t bx[4];
          boxcars4(P, k, tl, a, a4, bx);
          const acc_t m01 = bx[0] > bx[1] ? bx[0] : bx[1], m23 = bx[2] > bx[3] ? bx[2] : bx[3], m = m01 > m23 ? m01 : m23;
          tmax[k] = m > tmax[k] ? m : tmax[k];
        }
      }
#pragma unroll
      for (int k = 0; k < K; ++k) {
        const acc_t wmax = __reduce_max_sync(0xffffffffu, tmax[k]);
        const bool hit = wmax >= thr[k];
        bool better = false;
        if (wmax + 1 > seen[k]) better = publish(k, wmax + 1);
        if (!(hit || better)) continue;
        int c = 0, first = 0x7fffffff;
        for (int q = lane; q < nfast; q += 32) {
          const int tl = 4 * q;
          acc_t a[4], a4[4], bx[4];
          load4(P + tl, a);
          load4(P + tl + 4, a4);
          boxcars4(P, k, tl, a, a4, bx);
          c += (bx[0] >= thr[k]) + (bx[1] >= thr[k]) + (bx[2] >= thr[k]) + (bx[3] >= thr[k]);
          if (first == 0x7fffffff && (bx[0] == wmax || bx[1] == wmax || bx[2] == wmax || bx[3] == wmax))
            first = tile0 + tl + (bx[0] == wmax ? 0 : bx[1] == wmax ? 1 : bx[2] == wmax ? 2 : 3);
        }
        if (hit && c) atomicAdd(&s_count[k], c);
        if (better) {
          first = __reduce_min_sync(0xffffffffu, first);
          if (lane == 0) s_best[k][warp] = (unsigned long long)wmax + 1ull, s_tb[k][warp] = first;
          __syncwarp();
        }
      }
    }
    if (4 * nfast < kSpsWarpTile) {  // the end of the row: windows checked one by one, then merged into the warp's record
      acc_t tb1[K];  // this lane's (largest boxcar) + 1 among them, first position
      int tt[K];
#pragma unroll
      for (int k = 0; k < K; ++k) tb1[k] = 0, tt[k] = 0x7fffffff;
      for (int tl = 4 * nfast + lane; tl < kSpsWarpTile; tl += 32) {
        const int t1 = tile0 + tl;
        if (t1 >= n) break;
        const acc_t p0 = P[tl];
#pragma unroll
        for (int k = 0; k < K; ++k) {
          const int w = 1 << k;
          if (t1 + w <= n) {
            const acc_t bb = P[tl + w] - p0;
            if (bb >= tb1[k]) tb1[k] = bb + 1, tt[k] = t1;
            if (bb >= thr[k]) atomicAdd(&s_count[k], 1);
          }
        }
      }
#pragma unroll
      for (int k = 0; k < K; ++k) {
        const acc_t wb1 = __reduce_max_sync(0xffffffffu, tb1[k]);
        // these windows lie behind every window the warp has looked at so far: only a strictly larger sum is a record
        if (wb1 > seen[k] && publish(k, wb1)) {
          const int first = __reduce_min_sync(0xffffffffu, tb1[k] == wb1 ? tt[k] : 0x7fffffff);
          if (lane == 0) s_best[k][warp] = wb1, s_tb[k][warp] = first;
          __syncwarp();
        }
      }
    }
    __syncwarp();  // all lanes are done with this buffer before lane 0 refills it two tiles later
  }

  // ---------------- reduce over the block: larger sum wins, ties go to the smaller t ----------------------
  __syncthreads();
  if (tid < K) {
    const int k = tid;
    unsigned long long bb = 0;
    int t = 0x7fffffff;
    const int c = s_count[k];
    for (int i = 0; i < kSpsThreads / 32; ++i) {
      const unsigned long long ob = s_best[k][i];
      const int ot = s_tb[k][i];
      if (ob > bb || (ob == bb && ot < t)) bb = ob, t = ot;
    }
    const long long o = orow * K + k;
    if (bb == 0) {
      p.snr[o] = 0.0f, p.tmax[o] = -1, p.count[o] = 0;
    } else {
      p.snr[o] = sps_snr(bb - 1, s_c, k);
      p.tmax[o] = t;
      p.count[o] = c;
    }
  }
}

// Exclusive scan of count[0..m) into offsets[0..m] (int64), one CTA: the list positions of every (row, width).
__global__ void __launch_bounds__(1024) dd_sps_scan_kernel(const int32_t* __restrict__ count, long long m,
                                                           long long* __restrict__ offsets) {
  __shared__ long long wsum[32];
  __shared__ long long carry;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) carry = 0;
  __syncthreads();
  for (long long base = 0; base < m; base += 1024) {
    const long long i = base + tid;
    const long long v = i < m ? (long long)count[i] : 0;
    long long inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const long long u = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += u;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    long long pre = carry;
    for (int wq = 0; wq < warp; ++wq) pre += wsum[wq];
    if (i < m) offsets[i] = pre + inc - v;
    __syncthreads();
    if (tid == 1023) carry = pre + inc;
    __syncthreads();
  }
  if (tid == 0) offsets[m] = carry;
}

// The candidate list: (row, k, t, snr) of every boxcar above the threshold, in the order row, k, t, written at
// offsets[row*K + k] + (rank of t).  One CTA per row; rows without candidates (almost all) return at once.
template <bool WIDE>
__global__ void __launch_bounds__(kSpsThreads) dd_sps_fill_kernel(const SpsParams p) {
  using acc_t = typename std::conditional<WIDE, unsigned long long, uint32_t>::type;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  acc_t* P = reinterpret_cast<acc_t*>(smem_raw);
  __shared__ unsigned long long red[2][kSpsThreads / 32];
  __shared__ SpsRowConsts s_c;
  __shared__ unsigned long long s_warp_tot[kSpsThreads / 32];
  __shared__ int s_wcnt[kSpsThreads / 32];
  __shared__ long long s_written;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n = p.n, K = p.K;
  const long long orow = (long long)blockIdx.y * p.rows_per_beam + p.row0 + blockIdx.x;
  if (p.offsets[orow * K + K] == p.offsets[orow * K]) return;  // no candidate in this row
  const float* x = p.plane + (long long)blockIdx.y * p.beam_stride + (long long)blockIdx.x * p.pitch;
  if (p.stats) {
    if (tid == 0) sps_row_consts(p.stats[2 * orow], p.stats[2 * orow + 1], n, K, p.threshold, s_c);
  } else {
    unsigned long long t1, t2;
    sps_row_sums(x, n, red, t1, t2);
    if (tid == 0) sps_row_consts(t1, t2, n, K, p.threshold, s_c);
  }
  __syncthreads();
  const int halo = 1 << (K - 1);
  const int span = kSpsTile + halo;
  uint32_t* V = reinterpret_cast<uint32_t*>(smem_raw + sps_v_offset(span, sizeof(acc_t)));
  for (int k = 0; k < K; ++k) {
    const long long o0 = p.offsets[orow * K + k], o1 = p.offsets[orow * K + k + 1];
    if (o1 == o0) continue;
    const int w = 1 << k;
    const unsigned long long thr = s_c.thr[k];
    if (tid == 0) s_written = 0;
    __syncthreads();
    for (int tile0 = 0; tile0 < n; tile0 += kSpsTile) {
      if (K <= 9)
        sps_build_prefix<acc_t, sps_per(9)>(x, n, tile0, span, V, P, s_warp_tot);
      else
        sps_build_prefix<acc_t, sps_per(12)>(x, n, tile0, span, V, P, s_warp_tot);
      for (int c0 = 0; c0 < kSpsTile && tile0 + c0 < n; c0 += kSpsThreads) {  // 256 consecutive t at a time, in order
        const int tl = c0 + tid, t = tile0 + tl;
        const bool in = t + w <= n;
        const unsigned long long b = in ? (unsigned long long)(acc_t)(P[tl + w] - P[tl]) : 0ull;
        const bool hit = in && b >= thr && (WIDE || thr <= 0xffffffffull);
        const unsigned bal = __ballot_sync(0xffffffffu, hit);
        if (lane == 0) s_wcnt[warp] = __popc(bal);
        __syncthreads();
        int before = 0, total = 0;
        for (int wq = 0; wq < kSpsThreads / 32; ++wq) {
          before += wq < warp ? s_wcnt[wq] : 0;
          total += s_wcnt[wq];
        }
        if (hit) {
          const long long pos = o0 + s_written + before + __popc(bal & ((1u << lane) - 1u));
          if (pos < p.max_cands) {
            dd_sps_cand_t c;
            c.row = (int32_t)orow, c.width_log2 = k, c.t = t, c.snr = sps_snr(b, s_c, k);
            p.cand[pos] = c;
          }
        }
        __syncthreads();
        if (tid == 0) s_written += total;
        __syncthreads();
      }
      __syncthreads();
    }
  }
}

template <int K, bool WIDE>
static cudaError_t launch_sps(const SpsParams& sp, dim3 grid, size_t smem, cudaStream_t stream) {
  // per launch: the attribute is per device and the call is cheap (no static flag: not device- or thread-safe)
  cudaError_t e = cudaFuncSetAttribute(dd_sps_kernel<K, WIDE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 128 * 1024);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(dd_sps_kernel<K, WIDE>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
  if (e != cudaSuccess) return e;
  dd_sps_kernel<K, WIDE><<<grid, kSpsThreads, smem, stream>>>(sp);
  return cudaGetLastError();
}

template <int K>
static cudaError_t launch_sps_warp(const SpsParams& sp, dim3 grid, cudaStream_t stream) {
  const size_t smem = (size_t)(kSpsThreads / 32) * 2 * sps_warp_words(K) * 4;
  cudaError_t e = cudaFuncSetAttribute(dd_sps_warp_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(dd_sps_warp_kernel<K>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
  if (e != cudaSuccess) return e;
  dd_sps_warp_kernel<K><<<grid, kSpsThreads, smem, stream>>>(sp);
  return cudaGetLastError();
}

}  // namespace dd

namespace {

// validation shared by the entry points; rows_per_beam out
int sps_check(const dd_plan_t* p, const float* plane_dev, int32_t nwidths, double threshold, int64_t* rows_per_beam) {
  if (!p || !plane_dev || nwidths < 1 || nwidths > dd::kSpsMaxK || p->device < 0 ||
      !(threshold >= -1.0e300 && threshold <= 1.0e300))
    return DD_ERR_INVALID;
  if ((reinterpret_cast<uintptr_t>(plane_dev) & 15u) != 0) return DD_ERR_ALIGN;  // rows are read with 16-byte loads
  int cur = -1;
  cudaError_t e = cudaGetDevice(&cur);
  if (e != cudaSuccess) return dd::cuda_fail(e, "cudaGetDevice");
  if (cur != p->device) return DD_ERR_DEVICE;
  *rows_per_beam = 0;
  for (const auto& r : p->ranges) {
    // exactness of S2 = sum x^2 in 64 bits: (largest possible sum)^2 * nout < 2^63
    const double v = (double)p->nchans * (double)((1 << p->in_bits) - 1) * (double)r.decim;
    if (v * v * (double)r.nout >= 9.2e18 || r.nout > 0x7fffffffLL) return DD_ERR_OVERFLOW;
    *rows_per_beam += r.ndm;
  }
  return DD_OK;
}

bool sps_wide(const dd_plan_t* p, const dd::RangePlan& r, int nwidths) {
  // 32-bit prefix sums while the widest boxcar of the largest possible samples stays below 2^32 - 1 (the kernel
  // keeps "best + 1" and uses 2^32 - 1 as the unreachable threshold)
  const double vmax = (double)p->nchans * (double)((1 << p->in_bits) - 1) * (double)r.decim;
  return vmax * (double)(1 << (nwidths - 1)) >= 4294967295.0;
}

size_t sps_smem(bool wide, int nwidths) {
  const size_t span = (size_t)dd::kSpsTile + ((size_t)1 << (nwidths - 1));
  // then two raw-sample buffers (search kernel) / one staging buffer (fill kernel), each padded to a whole number of
  // samples per thread (the larger of the kernels' choices)
  return dd::sps_v_offset(span, wide ? 8 : 4) + 2 * (size_t)dd::sps_per(nwidths <= 9 ? 9 : 12) * dd::kSpsThreads * 4;
}

}  // namespace

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
  if (!snr_dev || !tmax_dev || !count_dev) return DD_ERR_INVALID;
  int64_t rows_per_beam = 0;
  int rc = sps_check(p, plane_dev, nwidths, threshold, &rows_per_beam);
  if (rc != DD_OK) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  // The barrier-free kernel (32-bit sums, up to 9 widths) takes all the ranges it applies to in ONE launch, longest rows
  // first; the other ranges (and everything else) go range by range to the block-wide kernel below.
  std::vector<char> merged(p->ranges.size(), 0);
  if (nwidths <= 9 && p->sps_warp_kernel) {
    std::vector<int> idx;
    for (size_t i = 0; i < p->ranges.size(); ++i)
      if (!sps_wide(p, p->ranges[i], nwidths)) idx.push_back((int)i);
    std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return p->ranges[a].nout > p->ranges[b].nout; });
    for (size_t first = 0; first < idx.size(); first += dd::kSpsMaxRanges) {
      dd::SpsParams sp = {};
      sp.plane = plane_dev;
      sp.beam_stride = p->beam_stride;
      sp.K = nwidths;
      sp.threshold = threshold;
      sp.snr = snr_dev;
      sp.tmax = tmax_dev;
      sp.count = count_dev;
      sp.rows_per_beam = rows_per_beam;
      sp.stats = p->row_stats;
      long long rows = 0;
      for (size_t k = first; k < idx.size() && k < first + dd::kSpsMaxRanges; ++k) {
        const auto& r = p->ranges[idx[k]];
        auto& g = sp.rg[sp.nr++];
        g.plane_off = r.offset, g.pitch = r.pitch, g.row0 = r.row0, g.n = (int)r.nout, g.ndm = r.ndm;
        rows += r.ndm;
        merged[idx[k]] = 1;
      }
      const dim3 grid((unsigned)rows, (unsigned)p->nbeams);
      cudaError_t e = cudaErrorInvalidValue;
#define DD_SPSW(K_) case K_: e = dd::launch_sps_warp<K_>(sp, grid, stream); break;
      switch (nwidths) { DD_SPSW(1) DD_SPSW(2) DD_SPSW(3) DD_SPSW(4) DD_SPSW(5) DD_SPSW(6) DD_SPSW(7) DD_SPSW(8) DD_SPSW(9) }
#undef DD_SPSW
      if (e != cudaSuccess) return dd::cuda_fail(e, "dd_sps_warp_kernel launch");
    }
  }
  int64_t row0 = 0;
  for (const auto& r : p->ranges) {
    if (merged[&r - p->ranges.data()]) {
      row0 += r.ndm;
      continue;
    }
    dd::SpsParams sp = {};
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
    sp.stats = p->row_stats;
    const bool wide = sps_wide(p, r, nwidths);
    const size_t smem = sps_smem(wide, nwidths);
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

int dd_sps_candidates(const dd_plan_t* p, const float* plane_dev, int32_t nwidths, double threshold, const int32_t* count_dev,
                      int64_t* offsets_dev, dd_sps_cand_t* cand_dev, int64_t max_cands, void* cuda_stream) {
  if (!count_dev || !offsets_dev || max_cands < 0 || (max_cands > 0 && !cand_dev)) return DD_ERR_INVALID;
  int64_t rows_per_beam = 0;
  int rc = sps_check(p, plane_dev, nwidths, threshold, &rows_per_beam);
  if (rc != DD_OK) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  const int64_t m = rows_per_beam * p->nbeams * nwidths;
  dd::dd_sps_scan_kernel<<<1, 1024, 0, stream>>>(count_dev, m, reinterpret_cast<long long*>(offsets_dev));
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return dd::cuda_fail(e, "dd_sps_scan_kernel launch");
  int64_t row0 = 0;
  for (const auto& r : p->ranges) {
    dd::SpsParams sp = {};
    sp.plane = plane_dev + r.offset;
    sp.beam_stride = p->beam_stride;
    sp.pitch = r.pitch;
    sp.n = (int)r.nout;
    sp.K = nwidths;
    sp.threshold = threshold;
    sp.row0 = row0;
    sp.rows_per_beam = rows_per_beam;
    sp.stats = p->row_stats;
    sp.offsets = reinterpret_cast<const long long*>(offsets_dev);
    sp.cand = cand_dev;
    sp.max_cands = max_cands;
    const bool wide = sps_wide(p, r, nwidths);
    const size_t smem = sps_smem(wide, nwidths);
    const dim3 grid((unsigned)r.ndm, (unsigned)p->nbeams);
    if (wide) {
      e = cudaFuncSetAttribute(dd::dd_sps_fill_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 128 * 1024);
      if (e == cudaSuccess) dd::dd_sps_fill_kernel<true><<<grid, dd::kSpsThreads, smem, stream>>>(sp);
    } else {
      e = cudaFuncSetAttribute(dd::dd_sps_fill_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 128 * 1024);
      if (e == cudaSuccess) dd::dd_sps_fill_kernel<false><<<grid, dd::kSpsThreads, smem, stream>>>(sp);
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return dd::cuda_fail(e, "dd_sps_fill_kernel launch");
    row0 += r.ndm;
  }
  return DD_OK;
}

}  // extern "C"
