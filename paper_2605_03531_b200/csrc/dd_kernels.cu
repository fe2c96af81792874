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

// ------------------------------------------------------------------------------------------------
// PTX helpers: mbarrier + 1-D bulk async copy (TMA), shared::cta addresses are 32-bit.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void fence_barrier_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
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
                                                      int Cpad, int64_t nsamps, int64_t ns_r, int64_t H, int64_t Wp) {
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
  const Tin* row = in + ((int64_t)beam * nchans + c) * nsamps;
  uint32_t v[NL][4];
#pragma unroll
  for (int m = 0; m < NL; ++m) load_lane4<Tin, K>(row, i0 + (int64_t)m * H, ns_r, v[m]);
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    uint4 w;
    if constexpr (NL == 8) {
      w.x = v[0][e] | (v[1][e] << 16);
      w.y = v[2][e] | (v[3][e] << 16);
      w.z = v[4][e] | (v[5][e] << 16);
      w.w = v[6][e] | (v[7][e] << 16);
    } else {
      w.x = v[0][e];
      w.y = v[1][e];
      w.z = v[2][e];
      w.w = v[3][e];
    }
    dst[e] = w;
  }
}

template <typename Tin, int NL>
static cudaError_t launch_pack_t(const dd_plan* p, const RangePlan& r, const void* in_dev, cudaStream_t stream) {
  uint4* P = reinterpret_cast<uint4*>(static_cast<char*>(p->ws) + r.ws_offset);
  const int64_t quads = r.Wp / 4;
  dim3 block(256);
  dim3 grid((unsigned)((quads + 255) / 256), (unsigned)r.Cpad, (unsigned)p->nbeams);
  const Tin* in = static_cast<const Tin*>(in_dev);
#define DD_PACK(K)                                                                                              \
  dd_pack_kernel<Tin, K, NL><<<grid, block, 0, stream>>>(in, P, p->nchans, r.Cpad, p->nsamps, r.ns, r.H, r.Wp); \
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

cudaError_t launch_pack(const dd_plan* p, const RangePlan& r, const void* in_dev, cudaStream_t stream) {
  if (p->in_bits == 8) {
    return r.NL == 8 ? launch_pack_t<uint8_t, 8>(p, r, in_dev, stream) : launch_pack_t<uint8_t, 4>(p, r, in_dev, stream);
  }
  return r.NL == 8 ? launch_pack_t<uint16_t, 8>(p, r, in_dev, stream) : launch_pack_t<uint16_t, 4>(p, r, in_dev, stream);
}

// ------------------------------------------------------------------------------------------------
// a3 + a4: tiled dedispersion
// ------------------------------------------------------------------------------------------------
struct TiledParams {
  const uint4* P;        // packed input of this range [nbeams][Cpad][Wp]
  const uint32_t* meta;  // [nblocks][Cpad][Dcta] byte offsets (d - dmin)*16
  const int32_t* dmin;   // [nblocks][Cpad]
  const int32_t* span;   // [nblocks][Cpad]
  float* out;            // beam 0, this range
  long long out_beam_stride, pitch, Wp, H, nout, ntau;
  int ndm, Cpad, Dcta, T, Cc, nstages, nblocks;
  int rowpitch;      // superwords per staged row = T + Smax
  int flush_stages;  // flush the 16-bit lanes every this many stages (NL == 8)
};

__host__ __device__ inline size_t tiled_stage_bytes(int Cc, int rowpitch, int Dcta) {
  return (size_t)Cc * ((size_t)rowpitch * kSuperwordBytes + (size_t)Dcta * 4);
}
constexpr int kBarRegion = 128;  // bytes reserved for the mbarriers at the start of dynamic smem

size_t tiled_smem_bytes(const RangePlan& r) {
  return kBarRegion + (size_t)r.stages * tiled_stage_bytes(r.Cc, r.T + r.Smax, r.Dcta);
}

__device__ __forceinline__ void add_pair(uint4& acc, const uint4& a, const uint4& b) {
  // one IADD3 per 32-bit word: two channels, and (NL == 8) two 16-bit time lanes, per instruction
  acc.x = acc.x + a.x + b.x;
  acc.y = acc.y + a.y + b.y;
  acc.z = acc.z + a.z + b.z;
  acc.w = acc.w + a.w + b.w;
}

// Shared-memory superword loads of the inner loop, written in PTX so that the conditional reload
// overwrites the four registers IN PLACE (the C++ form made ptxas copy them on every trial).
__device__ __forceinline__ void lds_first(uint4& w, uint32_t base, uint32_t off) {
  asm volatile("{\n .reg .u32 a;\n add.u32 a, %4, %5;\n ld.shared.v4.u32 {%0,%1,%2,%3}, [a];\n}"
               : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w)
               : "r"(base), "r"(off));
}
template <bool REUSE>
__device__ __forceinline__ void lds_if_changed(uint4& w, uint32_t base, uint32_t off, uint32_t prev) {
  if constexpr (REUSE) {
    asm volatile(
        "{\n .reg .pred p;\n .reg .u32 a;\n setp.ne.u32 p, %5, %6;\n add.u32 a, %4, %5;\n"
        " @p ld.shared.v4.u32 {%0,%1,%2,%3}, [a];\n}"
        : "+r"(w.x), "+r"(w.y), "+r"(w.z), "+r"(w.w)
        : "r"(base), "r"(off), "r"(prev));
  } else {
    lds_first(w, base, off);
  }
}

template <int NL, bool REUSE, int NT>
__global__ void __launch_bounds__(NT, 512 / NT) dd_tiled_kernel(const TiledParams p) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int tid = threadIdx.x;
  // CTA -> (trial block fastest, time tile, beam): CTAs resident together share a time tile in L2
  const long long lin = blockIdx.x;
  const int blk = (int)(lin % p.nblocks);
  const long long rest = lin / p.nblocks;
  const long long tau = rest % p.ntau;
  const int beam = (int)(rest / p.ntau);

  const uint32_t bar_base = smem_u32(smem);  // full[s] at +8*s, empty[s] at +8*(nstages+s)
  const int nstages = p.nstages;
  const size_t stage_bytes = tiled_stage_bytes(p.Cc, p.rowpitch, p.Dcta);
  const uint32_t row_bytes = (uint32_t)p.rowpitch * kSuperwordBytes;
  const uint32_t data_bytes = (uint32_t)p.Cc * row_bytes;
  const uint32_t meta_bytes = (uint32_t)p.Cc * (uint32_t)p.Dcta * 4u;
  const int nchunks = p.Cpad / p.Cc;

  if (tid == 0) {
    for (int s = 0; s < nstages; ++s) {
      mbar_init(bar_base + 8u * s, 1);                    // full: one arrive.expect_tx by the producer
      mbar_init(bar_base + 8u * (nstages + s), NT / 32);  // empty: one arrive per consumer warp
    }
    fence_barrier_init();
  }
  __syncthreads();

  // ---------------- producer role, rotated over the warps ---------------------------------------------
  // Chunk k (channels k*Cc .. k*Cc+Cc-1) is issued by warp k % nwarps: one bulk copy per channel row plus
  // one for the offsets, landing in stage k % nstages and signalling full[stage] with the byte count.
  // A warp issues chunk k when it starts iteration k - ahead (ahead = nstages - 2): the stage it refills
  // was consumed two iterations ago, so the wait on its empty barrier is normally already satisfied.
  // Row start and length of the warp's NEXT chunk are fetched one turn early (pf_d0 / pf_bytes).
  const uint4* Pbeam = p.P + (long long)beam * p.Cpad * p.Wp + tau * p.T;
  const long long tab = (long long)blk * p.Cpad;
  const int lane = tid & 31;
  const int warp = tid >> 5;
  constexpr int kWarps = NT / 32;
  const int ahead = nstages - 2;
  int pf_d0 = 0;
  uint32_t pf_bytes = 0;
  auto prefetch = [&](int k) {
    pf_bytes = 0;
    if (k < nchunks && lane < p.Cc) {
      const int c = k * p.Cc + lane;
      pf_d0 = __ldg(p.dmin + tab + c);
      pf_bytes = (uint32_t)(p.T + __ldg(p.span + tab + c)) * kSuperwordBytes;
    }
  };
  auto produce = [&](int k) {
    const int s = k % nstages;
    if (k >= nstages) mbar_wait(bar_base + 8u * (nstages + s), ((uint32_t)(k / nstages) & 1u) ^ 1u);
    const uint32_t sbase = smem_u32(smem + kBarRegion + (size_t)s * stage_bytes);
    const uint32_t full = bar_base + 8u * s;
    uint32_t total = pf_bytes;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) total += __shfl_xor_sync(0xffffffffu, total, o);
    if (lane == 0) {
      mbar_arrive_expect_tx(full, total + meta_bytes);
      bulk_copy_g2s(sbase + data_bytes, p.meta + (tab + (long long)k * p.Cc) * p.Dcta, meta_bytes, full);
    }
    __syncwarp();
    if (lane < p.Cc)
      bulk_copy_g2s(sbase + lane * row_bytes, Pbeam + (long long)(k * p.Cc + lane) * p.Wp + pf_d0, pf_bytes, full);
  };
  // prologue: chunks 0 .. ahead-1
  for (int k = warp; k < ahead && k < nchunks; k += kWarps) {
    prefetch(k);
    produce(k);
  }
  {  // first chunk this warp issues inside the loop
    int k = warp;
    while (k < ahead) k += kWarps;
    prefetch(k);
  }

  // ---------------- consumers: kRD trials x one superword (NL time lanes) per thread --------------
  const int g = tid / p.T;       // trial group inside the CTA (warp-uniform: T is a multiple of 32)
  const int ti = tid - g * p.T;  // superword inside the time tile
  uint4 acc[kRD];
  uint32_t wide[kRD][NL == 8 ? 8 : 1];
#pragma unroll
  for (int j = 0; j < kRD; ++j) {
    acc[j] = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int m = 0; m < (NL == 8 ? 8 : 1); ++m) wide[j][m] = 0;
  }
  const uint32_t thread_off = (uint32_t)ti * kSuperwordBytes;
  const uint32_t group_off = (uint32_t)g * kRD * 4u;
  const uint32_t meta_row = (uint32_t)p.Dcta * 4u;
  int since_flush = 0;

  for (int it = 0; it < nchunks; ++it) {
    const int s = it % nstages;
    const uint32_t ph = (uint32_t)(it / nstages) & 1u;
    {  // producer turn: chunk it + ahead belongs to warp (it + ahead) % kWarps
      const int k = it + ahead;
      if (k < nchunks && (k % kWarps) == warp) {
        produce(k);
        prefetch(k + kWarps);
      }
    }
    mbar_wait(bar_base + 8u * s, ph);
    const unsigned char* sdata = smem + kBarRegion + (size_t)s * stage_bytes + thread_off;
    const unsigned char* smeta = smem + kBarRegion + (size_t)s * stage_bytes + data_bytes + group_off;
#pragma unroll 2
    for (int cc = 0; cc < p.Cc; cc += 2) {
      const uint4 oa = *reinterpret_cast<const uint4*>(smeta + (uint32_t)cc * meta_row);
      const uint4 ob = *reinterpret_cast<const uint4*>(smeta + (uint32_t)(cc + 1) * meta_row);
      const unsigned char* ra = sdata + (uint32_t)cc * row_bytes;
      const unsigned char* rb = ra + row_bytes;
      const uint32_t aa = smem_u32(ra), ab = smem_u32(rb);
      uint4 wa, wb;
      lds_first(wa, aa, oa.x);
      lds_first(wb, ab, ob.x);
      add_pair(acc[0], wa, wb);
      lds_if_changed<REUSE>(wa, aa, oa.y, oa.x);
      lds_if_changed<REUSE>(wb, ab, ob.y, ob.x);
      add_pair(acc[1], wa, wb);
      lds_if_changed<REUSE>(wa, aa, oa.z, oa.y);
      lds_if_changed<REUSE>(wb, ab, ob.z, ob.y);
      add_pair(acc[2], wa, wb);
      lds_if_changed<REUSE>(wa, aa, oa.w, oa.z);
      lds_if_changed<REUSE>(wb, ab, ob.w, ob.z);
      add_pair(acc[3], wa, wb);
    }
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(bar_base + 8u * (nstages + s));  // stage may be refilled
    if constexpr (NL == 8) {
      if (++since_flush == p.flush_stages) {  // 16-bit lanes would overflow next: widen to 32 bits
        since_flush = 0;
#pragma unroll
        for (int j = 0; j < kRD; ++j) {
          wide[j][0] += acc[j].x & 0xffffu;
          wide[j][1] += acc[j].x >> 16;
          wide[j][2] += acc[j].y & 0xffffu;
          wide[j][3] += acc[j].y >> 16;
          wide[j][4] += acc[j].z & 0xffffu;
          wide[j][5] += acc[j].z >> 16;
          wide[j][6] += acc[j].w & 0xffffu;
          wide[j][7] += acc[j].w >> 16;
          acc[j] = make_uint4(0, 0, 0, 0);
        }
      }
    }
  }

  // ---------------- a4: DM-time writer, fp32 (I2F rounds to nearest even) -------------------------
  const long long i = tau * p.T + ti;
  if (i >= p.H) return;
  float* obase = p.out + (long long)beam * p.out_beam_stride;
#pragma unroll
  for (int j = 0; j < kRD; ++j) {
    const int jj = blk * p.Dcta + g * kRD + j;
    if (jj >= p.ndm) break;
    float* orow = obase + (long long)jj * p.pitch;
    uint32_t v[NL];
    if constexpr (NL == 8) {
      v[0] = wide[j][0] + (acc[j].x & 0xffffu);
      v[1] = wide[j][1] + (acc[j].x >> 16);
      v[2] = wide[j][2] + (acc[j].y & 0xffffu);
      v[3] = wide[j][3] + (acc[j].y >> 16);
      v[4] = wide[j][4] + (acc[j].z & 0xffffu);
      v[5] = wide[j][5] + (acc[j].z >> 16);
      v[6] = wide[j][6] + (acc[j].w & 0xffffu);
      v[7] = wide[j][7] + (acc[j].w >> 16);
    } else {
      v[0] = acc[j].x;
      v[1] = acc[j].y;
      v[2] = acc[j].z;
      v[3] = acc[j].w;
    }
#pragma unroll
    for (int m = 0; m < NL; ++m) {
      const long long t = i + (long long)m * p.H;
      if (t < p.nout) orow[t] = __uint2float_rn(v[m]);  // consecutive threads -> consecutive floats
    }
  }
}

template <int NL, bool REUSE, int NT>
static cudaError_t launch_tiled_t(const TiledParams& tp, long long nctas, size_t smem, cudaStream_t stream) {
  dd_tiled_kernel<NL, REUSE, NT><<<(unsigned)nctas, NT, smem, stream>>>(tp);
  return cudaGetLastError();
}

template <int NL, bool REUSE, int NT>
static cudaError_t set_smem_t() {
  return cudaFuncSetAttribute(dd_tiled_kernel<NL, REUSE, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
}

cudaError_t configure_kernels(const dd_plan*) {
  cudaError_t e;
#define DD_CFG(NL, RE, NT) \
  if ((e = set_smem_t<NL, RE, NT>()) != cudaSuccess) return e;
  DD_CFG(8, false, 256) DD_CFG(8, true, 256) DD_CFG(8, false, 512) DD_CFG(8, true, 512)
  DD_CFG(4, false, 256) DD_CFG(4, true, 256) DD_CFG(4, false, 512) DD_CFG(4, true, 512)
#undef DD_CFG
  return cudaSuccess;
}

cudaError_t launch_tiled(const dd_plan* p, const RangePlan& r, float* out_dev, cudaStream_t stream) {
  TiledParams tp;
  tp.P = reinterpret_cast<const uint4*>(static_cast<const char*>(p->ws) + r.ws_offset);
  tp.meta = r.d_meta;
  tp.dmin = r.d_dmin;
  tp.span = r.d_span;
  tp.out = out_dev + r.offset;
  tp.out_beam_stride = p->beam_stride;
  tp.pitch = r.pitch;
  tp.Wp = r.Wp;
  tp.H = r.H;
  tp.nout = r.nout;
  tp.ntau = r.ntau;
  tp.ndm = r.ndm;
  tp.Cpad = r.Cpad;
  tp.Dcta = r.Dcta;
  tp.T = r.T;
  tp.Cc = r.Cc;
  tp.nstages = r.stages;
  tp.nblocks = r.nblocks;
  tp.rowpitch = r.T + r.Smax;
  tp.flush_stages = r.flush > 0 ? r.flush / r.Cc : 0;
  const long long nctas = (long long)r.nblocks * r.ntau * p->nbeams;
  if (nctas <= 0 || nctas > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
  const size_t smem = tiled_smem_bytes(r);
  const int nt = r.G * r.T;
#define DD_GO(NL, RE, NT) return launch_tiled_t<NL, RE, NT>(tp, nctas, smem, stream)
  if (r.NL == 8) {
    if (nt == 512) { if (r.reuse) DD_GO(8, true, 512); else DD_GO(8, false, 512); }
    if (nt == 256) { if (r.reuse) DD_GO(8, true, 256); else DD_GO(8, false, 256); }
  } else {
    if (nt == 512) { if (r.reuse) DD_GO(4, true, 512); else DD_GO(4, false, 512); }
    if (nt == 256) { if (r.reuse) DD_GO(4, true, 256); else DD_GO(4, false, 256); }
  }
#undef DD_GO
  return cudaErrorInvalidConfiguration;
}

// ------------------------------------------------------------------------------------------------
// the simple variant
// ------------------------------------------------------------------------------------------------
template <typename Tin>
__global__ void __launch_bounds__(256) dd_direct_kernel(const Tin* __restrict__ in, const int32_t* __restrict__ delays,
                                                        float* __restrict__ out, int nchans, long long nsamps, int decim,
                                                        long long nout, long long pitch, long long out_beam_stride) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nout) return;
  const int j = blockIdx.y;
  const int beam = blockIdx.z;
  const Tin* x = in + (long long)beam * nchans * nsamps;
  const int32_t* d = delays + (long long)j * nchans;
  uint32_t s = 0;
  for (int c = 0; c < nchans; ++c) {
    const Tin* src = x + (long long)c * nsamps + (long long)decim * (t + d[c]);
    for (int q = 0; q < decim; ++q) s += (uint32_t)src[q];
  }
  out[(long long)beam * out_beam_stride + (long long)j * pitch + t] = __uint2float_rn(s);
}

cudaError_t launch_direct(const dd_plan* p, const RangePlan& r, const void* in_dev, float* out_dev,
                          cudaStream_t stream) {
  dim3 block(256);
  dim3 grid((unsigned)((r.nout + 255) / 256), (unsigned)r.ndm, (unsigned)p->nbeams);
  if (p->in_bits == 8) {
    dd_direct_kernel<uint8_t><<<grid, block, 0, stream>>>(static_cast<const uint8_t*>(in_dev), r.d_delays,
                                                          out_dev + r.offset, p->nchans, p->nsamps, r.decim, r.nout,
                                                          r.pitch, p->beam_stride);
  } else {
    dd_direct_kernel<uint16_t><<<grid, block, 0, stream>>>(static_cast<const uint16_t*>(in_dev), r.d_delays,
                                                           out_dev + r.offset, p->nchans, p->nsamps, r.decim, r.nout,
                                                           r.pitch, p->beam_stride);
  }
  return cudaGetLastError();
}

}  // namespace dd
