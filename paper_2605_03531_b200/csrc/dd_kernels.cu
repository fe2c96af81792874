// dd_kernels.cu -- CUDA kernels (sm_100a) of the dedispersion hot path and their launchers.
//
//   dd_pack_kernel    step a2: widen + time-decimate (a SUM over `decim` adjacent
//                     samples, reading A8) and lay the result out as 16-byte "superwords"
//                     whose lanes are NL time segments of the same channel (dd_internal.h).
//   dd_tiled_kernel   steps a3 + a4: S[j][t] = sum_c y[c][t + d(c,j)]  (Eq. 1.1 delays)
//                     staged through shared memory with 1-D TMA bulk copies (cp.async.bulk + mbarrier),
//                     register-blocked kRD trials x NL time lanes per thread, packed-lane integer adds
//                     (two 16-bit lanes per 32-bit IADD3, two channels per IADD3), reuse of the loaded
//                     superword across neighbouring trials with equal delay, fp32 DM-time writer.
//   dd_direct_kernel  the simple variant: one thread per (trial, sample), delays from a global table.
//
// Integer sums are exact, so every variant produces the same bits as the definition.
#include <cuda_runtime.h>
#include <stdint.h>

#include "dd_internal.h"

namespace dd {

// Two consecutive superwords as one 256-bit store (STG.256): a warp then writes whole 32-byte sectors.
__device__ __forceinline__ void store2(uint4* dst, const uint4& a, const uint4& b) {  // dst 32-byte aligned
  asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(dst), "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w),
               "r"(b.x), "r"(b.y), "r"(b.z), "r"(b.w)
               : "memory");
}

// ------------------------------------------------------------------------------------------------
// a2: pack + time decimation
// ------------------------------------------------------------------------------------------------
// Thread = 4 consecutive superwords i0..i0+3 of one (beam, channel) row.
//   lane m of superword i = sum_{q<K} x[K*(i + m*H) + q]  if i + m*H < ns_r, else 0.
// H is a multiple of 16, so the K*4 source elements of a lane start at a 4*K*sizeof(Tin)-aligned
// address and are fetched with one vector load per 16 bytes.
template <typename Tin, int K>
__device__ __forceinline__ void load_lane4(const Tin* __restrict__ row, int64_t s, int64_t ns_r, uint32_t v[4]) {
  // s = first decimated index; returns v[e] = y[s+e]
  constexpr int kBytes = 4 * K * (int)sizeof(Tin);
  constexpr uintptr_t kAlignMask = (kBytes > 16 ? 16 : kBytes) - 1;
  const Tin* src = row + (int64_t)K * s;
  // vector path: fully inside the row and aligned (rows are aligned whenever nsamps*sizeof(Tin) is a
  // multiple of 16, true for all power-of-two lengths of the paper's data blocks)
  if (s + 4 <= ns_r && (reinterpret_cast<uintptr_t>(src) & kAlignMask) == 0) {
    Tin buf[4 * K];
    if constexpr (kBytes == 4) {
      *reinterpret_cast<uint32_t*>(buf) = __ldg(reinterpret_cast<const uint32_t*>(src));
    } else if constexpr (kBytes == 8) {
      *reinterpret_cast<uint2*>(buf) = __ldg(reinterpret_cast<const uint2*>(src));
    } else {
#pragma unroll
      for (int q = 0; q < kBytes / 16; ++q)
        reinterpret_cast<uint4*>(buf)[q] = __ldg(reinterpret_cast<const uint4*>(src) + q);
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      uint32_t a = 0;
#pragma unroll
      for (int q = 0; q < K; ++q) a += (uint32_t)buf[e * K + q];
      v[e] = a;
    }
  } else {
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      uint32_t a = 0;
      if (s + e < ns_r) {
#pragma unroll
        for (int q = 0; q < K; ++q) a += (uint32_t)row[(int64_t)K * (s + e) + q];
      }
      v[e] = a;
    }
  }
}

template <typename Tin, int K, int NL>
__global__ void __launch_bounds__(256) dd_pack_kernel(const Tin* __restrict__ in, uint4* __restrict__ P, int nchans,
                                                      int Cpad, int64_t nsamps, int64_t ns_r, int64_t H, int64_t Wp,
                                                      int rev, int64_t off) {
  const int64_t i0 = 4 * ((int64_t)blockIdx.x * blockDim.x + threadIdx.x);
  if (i0 >= Wp) return;
  const int c = blockIdx.y;
  const int beam = blockIdx.z;
  uint4* dst = P + ((int64_t)beam * Cpad + c) * Wp + i0;
  if (c >= nchans) {  // zero rows that pad the channel count to a multiple of the stage size
    const uint4 z = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int e = 0; e < 4; ++e) dst[e] = z;
    return;
  }
  const Tin* row = in + ((int64_t)beam * nchans + (rev ? nchans - 1 - c : c)) * nsamps + off;  // rev: ascending band
  uint32_t v[NL][4];
#pragma unroll
  for (int m = 0; m < NL; ++m) load_lane4<Tin, K>(row, i0 + (int64_t)m * H, ns_r, v[m]);
  uint4 w[4];
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    if constexpr (NL == 8) {
      w[e].x = v[0][e] | (v[1][e] << 16);
      w[e].y = v[2][e] | (v[3][e] << 16);
      w[e].z = v[4][e] | (v[5][e] << 16);
      w[e].w = v[6][e] | (v[7][e] << 16);
    } else {
      w[e].x = v[0][e];
      w[e].y = v[1][e];
      w[e].z = v[2][e];
      w[e].w = v[3][e];
    }
  }
  store2(dst, w[0], w[1]);  // i0 is a multiple of 4 and Wp of 8: 64-byte aligned
  store2(dst + 2, w[2], w[3]);
}

template <typename Tin, int NL>
static cudaError_t launch_pack_t(const dd_plan* p, const RangePlan& r, const void* in_dev, cudaStream_t stream) {
  uint4* P = reinterpret_cast<uint4*>(static_cast<char*>(p->ws) + r.ws_offset);
  const int64_t quads = r.Wp / 4;
  dim3 block(256);
  dim3 grid((unsigned)((quads + 255) / 256), (unsigned)r.Cpad, (unsigned)p->nbeams);
  const Tin* in = static_cast<const Tin*>(in_dev);
#define DD_PACK(K)                                                                                              \
  dd_pack_kernel<Tin, K, NL><<<grid, block, 0, stream>>>(in, P, p->nchans, r.Cpad, p->nsamps, r.ns, r.H, r.Wp, \
                                                         p->ascending, r.in_off);                                 \
  break
  switch (r.decim) {
    case 1: DD_PACK(1);
    case 2: DD_PACK(2);
    case 4: DD_PACK(4);
    case 8: DD_PACK(8);
    default: return cudaErrorInvalidValue;
  }
#undef DD_PACK
  return cudaGetLastError();
}

// a2 for 8-bit lanes (NL = 16), undecimated input.  Thread = 4 consecutive superwords i0..i0+3 of one
// (beam, channel) row; byte k of word q of superword i is x[i + (4q+k)*H] (0 past the end of the row).  uint16
// samples go to two planes of this form: plane 0 their low bytes, plane 1 their high bytes.
template <typename Tin>
__global__ void __launch_bounds__(256) dd_pack_bytes_kernel(const Tin* __restrict__ in, uint4* __restrict__ P0,
                                                            uint4* __restrict__ P1, int nchans, int Cpad, int64_t nsamps,
                                                            int64_t ns_r, int64_t H, int64_t Wp, int rev, int64_t off) {
  const int64_t i0 = 4 * ((int64_t)blockIdx.x * blockDim.x + threadIdx.x);
  if (i0 >= Wp) return;
  const int c = blockIdx.y;
  const int beam = blockIdx.z;
  const int64_t o = ((int64_t)beam * Cpad + c) * Wp + i0;
  constexpr bool kTwo = sizeof(Tin) == 2;
  if (c >= nchans) {  // zero rows that pad the channel count to a multiple of the stage size
    const uint4 z = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      P0[o + e] = z;
      if (kTwo) P1[o + e] = z;
    }
    return;
  }
  const Tin* row = in + ((int64_t)beam * nchans + (rev ? nchans - 1 - c : c)) * nsamps + off;
  uint32_t lo[4][4] = {}, hi[4][4] = {};  // [superword e][word q]
#pragma unroll
  for (int m = 0; m < 16; ++m) {
    const int64_t s = i0 + (int64_t)m * H;
    uint32_t v[4];
    const Tin* src = row + s;
    if (s + 4 <= ns_r && (reinterpret_cast<uintptr_t>(src) & (4 * sizeof(Tin) - 1)) == 0) {
      if constexpr (kTwo) {
        const uint2 t = __ldg(reinterpret_cast<const uint2*>(src));
        v[0] = t.x & 0xffffu, v[1] = t.x >> 16, v[2] = t.y & 0xffffu, v[3] = t.y >> 16;
      } else {
        const uint32_t t = __ldg(reinterpret_cast<const uint32_t*>(src));
        v[0] = t & 0xffu, v[1] = (t >> 8) & 0xffu, v[2] = (t >> 16) & 0xffu, v[3] = t >> 24;
      }
    } else {
#pragma unroll
      for (int e = 0; e < 4; ++e) v[e] = s + e < ns_r ? (uint32_t)row[s + e] : 0u;
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      lo[e][m / 4] |= (v[e] & 0xffu) << (8 * (m % 4));
      if (kTwo) hi[e][m / 4] |= (v[e] >> 8) << (8 * (m % 4));
    }
  }
#pragma unroll
  for (int e = 0; e < 4; e += 2) {
    store2(P0 + o + e, make_uint4(lo[e][0], lo[e][1], lo[e][2], lo[e][3]),
           make_uint4(lo[e + 1][0], lo[e + 1][1], lo[e + 1][2], lo[e + 1][3]));
    if (kTwo)
      store2(P1 + o + e, make_uint4(hi[e][0], hi[e][1], hi[e][2], hi[e][3]),
             make_uint4(hi[e + 1][0], hi[e + 1][1], hi[e + 1][2], hi[e + 1][3]));
  }
}

// a2 for spectrum-major input [beam][time][channel] (the layout of the thesis's shared-memory ring buffers,
// PAPER.md:351): the corner turn is fused into the pack.  CTA = kTcCh channels x kTcTi superword indices.
// Phase 1 reads the NL*kTcTi*decim spectra slices of the tile with consecutive threads on consecutive
// channels (coalesced) and sums `decim` spectra into shared memory; phase 2 builds the superwords of every
// channel and writes them with consecutive threads on consecutive superwords.
constexpr int kTcCh = 128, kTcTi = 4;
template <typename Tin, int NL>
__global__ void __launch_bounds__(256) dd_pack_tc_kernel(const Tin* __restrict__ in, uint4* __restrict__ P0,
                                                         uint4* __restrict__ P1, int nchans, int Cpad, int64_t nsamps,
                                                         int64_t ns_r, int decim, int64_t H, int64_t Wp, int rev,
                                                         int64_t off) {
  __shared__ uint32_t vals[NL][kTcTi][kTcCh + 1];
  const int64_t i0 = (int64_t)blockIdx.x * kTcTi;
  const int c0 = blockIdx.y * kTcCh;
  const int beam = blockIdx.z;
  const Tin* x = in + (int64_t)beam * nsamps * nchans;
  if (!rev && nchans % 4 == 0) {
    // fast path: a warp reads the 128 channels of one spectrum slice with one 4-channel vector load per thread
    const int l = threadIdx.x & 31, wq = threadIdx.x >> 5;
    const int c = c0 + 4 * l;
#pragma unroll
    for (int rr = 0; rr < NL * kTcTi / 8; ++rr) {
      const int row = wq + 8 * rr, m = row / kTcTi, ti = row % kTcTi;
      const int64_t s = i0 + ti + (int64_t)m * H;  // decimated sample index
      uint32_t a[4] = {0, 0, 0, 0};
      if (c < nchans && s < ns_r) {
        const Tin* src = x + ((int64_t)decim * s + off) * nchans + c;
#pragma unroll 4
        for (int q = 0; q < decim; ++q) {
          if constexpr (sizeof(Tin) == 1) {
            const uint32_t t = __ldg(reinterpret_cast<const uint32_t*>(src + (int64_t)q * nchans));
            a[0] += t & 0xffu, a[1] += (t >> 8) & 0xffu, a[2] += (t >> 16) & 0xffu, a[3] += t >> 24;
          } else {
            const uint2 t = __ldg(reinterpret_cast<const uint2*>(src + (int64_t)q * nchans));
            a[0] += t.x & 0xffffu, a[1] += t.x >> 16, a[2] += t.y & 0xffffu, a[3] += t.y >> 16;
          }
        }
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) vals[m][ti][4 * l + k] = a[k];
    }
  } else {
    for (int idx = threadIdx.x; idx < NL * kTcTi * kTcCh; idx += blockDim.x) {
      const int cl = idx % kTcCh, ti = (idx / kTcCh) % kTcTi, m = idx / (kTcCh * kTcTi);
      const int c = c0 + cl;
      const int64_t s = i0 + ti + (int64_t)m * H;  // decimated sample index
      uint32_t a = 0;
      if (c < nchans && s < ns_r) {
        const Tin* src = x + ((int64_t)decim * s + off) * nchans + (rev ? nchans - 1 - c : c);
        for (int q = 0; q < decim; ++q) a += (uint32_t)src[(int64_t)q * nchans];
      }
      vals[m][ti][cl] = a;
    }
  }
  __syncthreads();
  for (int idx = threadIdx.x; idx < kTcTi * kTcCh; idx += blockDim.x) {
    const int ti = idx % kTcTi, cl = idx / kTcTi;
    const int c = c0 + cl;
    if (c >= Cpad || i0 + ti >= Wp) continue;
    const int64_t o = ((int64_t)beam * Cpad + c) * Wp + i0 + ti;
    uint32_t v[NL];
#pragma unroll
    for (int m = 0; m < NL; ++m) v[m] = vals[m][ti][cl];
    if constexpr (NL == 4) {
      P0[o] = make_uint4(v[0], v[1], v[2], v[3]);
    } else if constexpr (NL == 8) {
      P0[o] = make_uint4(v[0] | (v[1] << 16), v[2] | (v[3] << 16), v[4] | (v[5] << 16), v[6] | (v[7] << 16));
    } else {  // 16 byte lanes; uint16 input: low bytes to plane 0, high bytes to plane 1
      uint32_t lo[4], hi[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        lo[q] = (v[4 * q] & 0xffu) | ((v[4 * q + 1] & 0xffu) << 8) | ((v[4 * q + 2] & 0xffu) << 16) | (v[4 * q + 3] << 24);
        hi[q] = (v[4 * q] >> 8) | ((v[4 * q + 1] >> 8) << 8) | ((v[4 * q + 2] >> 8) << 16) | ((v[4 * q + 3] >> 8) << 24);
      }
      P0[o] = make_uint4(lo[0], lo[1], lo[2], lo[3]);
      if (sizeof(Tin) == 2) P1[o] = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    }
  }
}

template <typename Tin, int NL>
static cudaError_t launch_pack_tc_t(const dd_plan* p, const RangePlan& r, const void* in_dev, cudaStream_t stream) {
  uint4* P0 = reinterpret_cast<uint4*>(static_cast<char*>(p->ws) + r.ws_offset);
  uint4* P1 = reinterpret_cast<uint4*>(static_cast<char*>(p->ws) + r.ws_offset + r.plane_bytes);
  dim3 grid((unsigned)((r.Wp + kTcTi - 1) / kTcTi), (unsigned)((r.Cpad + kTcCh - 1) / kTcCh), (unsigned)p->nbeams);
  dd_pack_tc_kernel<Tin, NL><<<grid, 256, 0, stream>>>(static_cast<const Tin*>(in_dev), P0, P1, p->nchans, r.Cpad,
                                                       p->nsamps, r.ns, r.decim, r.H, r.Wp, p->ascending, r.in_off);
  return cudaGetLastError();
}

cudaError_t launch_pack(const dd_plan* p, const RangePlan& r, const void* in_dev, cudaStream_t stream) {
  if (p->layout == DD_LAYOUT_SPECTRUM_MAJOR) {
    if (p->in_bits == 8)
      return r.NL == 16 ? launch_pack_tc_t<uint8_t, 16>(p, r, in_dev, stream)
             : r.NL == 8 ? launch_pack_tc_t<uint8_t, 8>(p, r, in_dev, stream)
                         : launch_pack_tc_t<uint8_t, 4>(p, r, in_dev, stream);
    return r.NL == 16 ? launch_pack_tc_t<uint16_t, 16>(p, r, in_dev, stream)
           : r.NL == 8 ? launch_pack_tc_t<uint16_t, 8>(p, r, in_dev, stream)
                       : launch_pack_tc_t<uint16_t, 4>(p, r, in_dev, stream);
  }
  if (r.NL == 16) {
    uint4* P0 = reinterpret_cast<uint4*>(static_cast<char*>(p->ws) + r.ws_offset);
    uint4* P1 = reinterpret_cast<uint4*>(static_cast<char*>(p->ws) + r.ws_offset + r.plane_bytes);
    dim3 block(256);
    dim3 grid((unsigned)((r.Wp / 4 + 255) / 256), (unsigned)r.Cpad, (unsigned)p->nbeams);
    if (p->in_bits == 8)
      dd_pack_bytes_kernel<uint8_t><<<grid, block, 0, stream>>>(static_cast<const uint8_t*>(in_dev), P0, nullptr, p->nchans,
                                                                r.Cpad, p->nsamps, r.ns, r.H, r.Wp, p->ascending, r.in_off);
    else
      dd_pack_bytes_kernel<uint16_t><<<grid, block, 0, stream>>>(static_cast<const uint16_t*>(in_dev), P0, P1, p->nchans,
                                                                 r.Cpad, p->nsamps, r.ns, r.H, r.Wp, p->ascending, r.in_off);
    return cudaGetLastError();
  }
  if (p->in_bits == 8) {
    return r.NL == 8 ? launch_pack_t<uint8_t, 8>(p, r, in_dev, stream) : launch_pack_t<uint8_t, 4>(p, r, in_dev, stream);
  }
  return r.NL == 8 ? launch_pack_t<uint16_t, 8>(p, r, in_dev, stream) : launch_pack_t<uint16_t, 4>(p, r, in_dev, stream);
}

// ------------------------------------------------------------------------------------------------
// DD_KERNEL_SUBBAND: pair rows.  P2[beam][2v + p][i] = P[beam][2v][i] + P[beam][2v+1][i + delta_v + p], lane by lane
// (16-bit lanes: 2 * maxval < 65536, no carry between lanes).  A delay is a shift by whole superwords, so both
// terms are aligned 16-byte loads.  Thread = 4 consecutive time indices of one pair row: 4 + 5 loads, 8 stores.
// Elements past the end of the packed row (never needed by a valid output) read as zero.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 add4(const uint4& a, const uint4& b) {
  return make_uint4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w);
}
__global__ void __launch_bounds__(256) dd_pair_kernel(const uint4* __restrict__ P, uint4* __restrict__ P2,
                                                      const int32_t* __restrict__ delta, int npairs, int64_t Wp) {
  const int64_t i0 = 4 * ((int64_t)blockIdx.x * blockDim.x + threadIdx.x);
  if (i0 >= Wp) return;
  const int v = blockIdx.y;
  const int beam = blockIdx.z;
  const uint4* ra = P + ((int64_t)beam * 2 * npairs + 2 * v) * Wp;
  const uint4* rb = ra + Wp;
  const int64_t d = delta[v];
  const uint4 z = make_uint4(0, 0, 0, 0);
  uint4 b[5];
#pragma unroll
  for (int e = 0; e < 5; ++e) {
    const int64_t k = i0 + d + e;
    b[e] = (k >= 0 && k < Wp) ? __ldg(rb + k) : z;
  }
  uint4* dst0 = P2 + ((int64_t)beam * 2 * npairs + 2 * v) * Wp + i0;  // i0 is a multiple of 4 and Wp of 8: all four in range
  uint4* dst1 = dst0 + Wp;
  uint4 a[4];
#pragma unroll
  for (int e = 0; e < 4; ++e) a[e] = __ldg(ra + i0 + e);
  store2(dst0, add4(a[0], b[0]), add4(a[1], b[1]));
  store2(dst0 + 2, add4(a[2], b[2]), add4(a[3], b[3]));
  store2(dst1, add4(a[0], b[1]), add4(a[1], b[2]));
  store2(dst1 + 2, add4(a[2], b[3]), add4(a[3], b[4]));
}

cudaError_t launch_pairs(const dd_plan* p, const RangePlan& r, cudaStream_t stream) {
  const uint4* P = reinterpret_cast<const uint4*>(static_cast<const char*>(p->ws) + r.ws_offset);
  uint4* P2 = reinterpret_cast<uint4*>(static_cast<char*>(p->ws) + r.ws2_offset);
  const int npairs = r.Cpad / 2;
  dim3 grid((unsigned)((r.Wp / 4 + 255) / 256), (unsigned)npairs, (unsigned)p->nbeams);
  dd_pair_kernel<<<grid, 256, 0, stream>>>(P, P2, r.d_delta, npairs, r.Wp);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// the simple variant
// ------------------------------------------------------------------------------------------------
template <typename Tin>
__global__ void __launch_bounds__(256) dd_direct_kernel(const Tin* __restrict__ in, const int32_t* __restrict__ delays,
                                                        float* __restrict__ out, int nchans, long long nsamps, int decim,
                                                        long long nout, long long pitch, long long out_beam_stride,
                                                        long long chan_stride, long long time_stride, int rev,
                                                        long long off, unsigned long long* stats,
                                                        long long stats_beam_stride) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  const int beam = blockIdx.z;
  uint32_t s = 0;
  if (t < nout) {
    const Tin* x = in + (long long)beam * nchans * nsamps;
    const int32_t* d = delays + (long long)j * nchans;  // internal order: channel 0 = highest frequency
    for (int c = 0; c < nchans; ++c) {
      const Tin* src = x + (long long)(rev ? nchans - 1 - c : c) * chan_stride + ((long long)decim * (t + d[c]) + off) * time_stride;
      for (int q = 0; q < decim; ++q) s += (uint32_t)src[q * time_stride];
    }
    out[(long long)beam * out_beam_stride + (long long)j * pitch + t] = __uint2float_rn(s);
  }
  if (stats) {  // row statistics for the single-pulse search (dd_plan_set_row_stats): one pair of atomics per warp
    unsigned long long s1 = t < nout ? s : 0, s2 = t < nout ? (unsigned long long)s * s : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      s1 += __shfl_down_sync(0xffffffffu, s1, o);
      s2 += __shfl_down_sync(0xffffffffu, s2, o);
    }
    if ((threadIdx.x & 31) == 0) {
      unsigned long long* st = stats + (long long)beam * stats_beam_stride + 2ll * j;
      atomicAdd(st, s1);
      atomicAdd(st + 1, s2);
    }
  }
}

cudaError_t launch_direct(const dd_plan* p, const RangePlan& r, const void* in_dev, float* out_dev,
                          cudaStream_t stream) {
  dim3 block(256);
  dim3 grid((unsigned)((r.nout + 255) / 256), (unsigned)r.ndm, (unsigned)p->nbeams);
  const bool tc = p->layout == DD_LAYOUT_SPECTRUM_MAJOR;
  const long long cs = tc ? 1 : p->nsamps, ts = tc ? p->nchans : 1;
  unsigned long long* stats = p->row_stats ? p->row_stats + 2 * r.row0 : nullptr;
  if (p->in_bits == 8) {
    dd_direct_kernel<uint8_t><<<grid, block, 0, stream>>>(static_cast<const uint8_t*>(in_dev), r.d_delays,
                                                          out_dev + r.offset, p->nchans, p->nsamps, r.decim, r.nout,
                                                          r.pitch, p->beam_stride, cs, ts, p->ascending, r.in_off, stats,
                                                          2 * p->rows_per_beam);
  } else {
    dd_direct_kernel<uint16_t><<<grid, block, 0, stream>>>(static_cast<const uint16_t*>(in_dev), r.d_delays,
                                                           out_dev + r.offset, p->nchans, p->nsamps, r.decim, r.nout,
                                                           r.pitch, p->beam_stride, cs, ts, p->ascending, r.in_off, nullptr, 0);
  }
  return cudaGetLastError();
}

}  // namespace dd
