// dd_tiled.cu -- steps a3 + a4 of the hot path: the tiled dedispersion kernel and its
// launcher.
//
//   S[j][t] = sum_c y[c][t + d(c,j)]      (PAPER.md:421 brute-force O(m x N) sum; delays of Eq. 1.1)
//
// CTA tile = Dcta trials x T superwords x all channels.  Thread = kRD (8) neighbouring trials x one
// superword (NL time lanes, dd_internal.h).  Channel rows are staged into a shared-memory ring by 1-D TMA
// bulk copies (cp.async.bulk + mbarrier).  The adder is integer and packed: one IADD3 adds two channels
// into two 16-bit time lanes (NL == 8), i.e. four algorithmic adds per instruction.  Packed lanes are kept
// exact by a two-level carry-save scheme: every `flush` channels the upper bytes of the 16-bit lanes are
// moved into a second packed accumulator (sum = lo + 256*hi), so the accumulators of a trial are 8
// registers and never overflow.  Part of the adds are issued as IMADs on the FMA-side pipe, which the ALU-pipe
// instructions of the adder would otherwise leave idle.  Neighbouring trials that share a delay reuse the superword
// held in registers (delta, reuse and hybrid table forms, dd_internal.h).  The DM-time writer converts once (I2F.RN)
// and stores fp32.
//
// Integer sums are exact, so the result has the same bits as the definition whatever the order.
#include <cuda_runtime.h>
#include <stdint.h>

#include "dd_internal.h"
#include "dd_ptx.cuh"

namespace dd {

// Shared-memory superword loads of the inner loop, written in PTX so that a conditional reload overwrites
// the four registers IN PLACE (the C++ form makes ptxas copy them on every trial).
__device__ __forceinline__ void lds_sw(uint4& w, uint32_t addr) {
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w) : "r"(addr));
}
// general modes: reload iff this trial's offset differs from the previous trial's
__device__ __forceinline__ void lds_if_ne(uint4& w, uint32_t addr, uint32_t off, uint32_t prev) {
  asm volatile(
      "{\n .reg .pred p;\n setp.ne.u32 p, %5, %6;\n"
      " @p ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];\n}"
      : "+r"(w.x), "+r"(w.y), "+r"(w.z), "+r"(w.w)
      : "r"(addr), "r"(off), "r"(prev));
}
// delta mode: if bit BIT of m is set, step one superword forward and reload in place
template <int BIT>
__device__ __forceinline__ void lds_if_bit(uint4& w, uint32_t& addr, uint32_t m) {
  asm volatile(
      "{\n .reg .pred p;\n .reg .b32 t;\n and.b32 t, %5, %6;\n setp.ne.u32 p, t, 0;\n"
      " @p add.u32 %4, %4, 16;\n"
      " @p ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];\n}"
      : "+r"(w.x), "+r"(w.y), "+r"(w.z), "+r"(w.w), "+r"(addr)
      : "r"(m), "n"(1u << BIT));
}

// pair mode: if bit BIT of m is set (the pair row of this trial differs from the previous trial's: its delay
// stepped or the other pre-summed row is needed), reload from the byte offset the table gives for this trial
template <int BIT>
__device__ __forceinline__ void lds_pair_if(uint4& w, uint32_t sdata, uint32_t off, uint32_t m) {
  asm volatile(
      "{\n .reg .pred p;\n .reg .b32 t;\n and.b32 t, %6, %7;\n setp.ne.u32 p, t, 0;\n"
      " add.u32 t, %4, %5;\n"
      " @p ld.shared.v4.u32 {%0,%1,%2,%3}, [t];\n}"
      : "+r"(w.x), "+r"(w.y), "+r"(w.z), "+r"(w.w)
      : "r"(sdata), "r"(off), "r"(m), "n"(1u << BIT));
}

__device__ __forceinline__ void add_pair(uint4& acc, const uint4& a, const uint4& b) {
  // one IADD3 per 32-bit word: two channels, and (NL == 8) two 16-bit time lanes, per instruction
  acc.x = acc.x + a.x + b.x;
  acc.y = acc.y + a.y + b.y;
  acc.z = acc.z + a.z + b.z;
  acc.w = acc.w + a.w + b.w;
}
// The delta kernel was bound by the ALU pipe (IADD3, LOP3, R2P, the predicated address steps: 79 % busy) while the
// FMA-side pipe idled, so part of the adds of every trial step go there as IMADs (two per IADD3 they replace: more issue
// slots, fewer ALU slots).  Words per quad and trial step (of 8) moved, config 3: 0: 111.8 ms, 1: 110.8, 2: 109.2,
// 3: 109.1, 4: 112.6 (issue slots and shared memory take over); with the channels dealt to quads by phase (dd_plan.cu
// build_tables) 1: 103.5, 2: 102.1, 3: 100.7, 4: 104.1, 5: 109.2; with the final tile and the padded trial groups
// skipped 0: 97.8, 1: 95.1, 2: 95.1, 3: 95.5, 4: 99.8.
constexpr int kDeltaFmaWords = 2;
// acc += t on the FMA-side pipe: IMAD with a multiplier of one that ptxas cannot fold (a kernel parameter)
__device__ __forceinline__ uint32_t mad1(uint32_t t, uint32_t one, uint32_t e) {
  uint32_t d;
  asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(t), "r"(one), "r"(e));
  return d;
}
// add_pair with the first NW words of the superword added by two IMADs each instead of one IADD3
template <int NW>
__device__ __forceinline__ void add_pair_mix(uint4& acc, const uint4& a, const uint4& b, uint32_t one) {
  acc.x = NW > 0 ? mad1(b.x, one, mad1(a.x, one, acc.x)) : acc.x + a.x + b.x;
  acc.y = NW > 1 ? mad1(b.y, one, mad1(a.y, one, acc.y)) : acc.y + a.y + b.y;
  acc.z = NW > 2 ? mad1(b.z, one, mad1(a.z, one, acc.z)) : acc.z + a.z + b.z;
  acc.w = NW > 3 ? mad1(b.w, one, mad1(a.w, one, acc.w)) : acc.w + a.w + b.w;
}
struct TiledParams {
  const uint4* P;       // packed input of this range [nbeams][Cpad][Wp]
  const uint4* meta;    // per trial block: offsets / changed bits (dd_internal.h RangePlan::d_meta)
  const int32_t* dmin;  // [nblocks][Cpad] first delay of the block = start of the staged row
  const int32_t* span;  // [nblocks][Cpad] delay spread of the block = staged row length beyond T
  const int32_t* chan;  // [nblocks][Cpad] channel (row of P) staged in that row, or nullptr: the row index itself
  float* out;           // beam 0, this range
  long long out_beam_stride, pitch, Wp, H, nout, ntau;
  int ndm, Cpad, G, T, Cc, nstages;
  int nd;            // hybrid modes: leading channel chunks that carry the delta table
  int blk0, nblk;    // trial blocks of this launch: blk0 .. blk0 + nblk - 1
  int rowpitch;      // superwords per staged row = T + Smax
  int flush_stages;  // move the upper bytes of the packed lanes away every this many stages (NL == 8, 16)
  uint32_t one;       // 1: a multiplier ptxas cannot fold, keeps integer adds on the FMA-side pipe as IMAD (add_bytes)
  float accum_scale;  // 0: store; else out = value * accum_scale + out (high byte plane of uint16 input)
  unsigned long long* stats;  // nullptr, or [beam][trial of this range][2]: sum x and sum x^2 of the rows written (dd_plan_set_row_stats)
  long long stats_beam_stride;
};

__host__ __device__ inline size_t tiled_stage_bytes(int mode, int NL, int Cc, int rowpitch, int G) {
  return ((size_t)Cc * (size_t)rowpitch * kSuperwordBytes + tiled_meta_bytes(mode, NL, Cc, G) + 127) / 128 * 128;
}
constexpr int kBarRegion = 128;  // bytes reserved for the mbarriers at the start of dynamic smem

size_t tiled_smem_bytes(const RangePlan& r) {
  // + 512: delta mode prefetches one table row (G <= 16 entries of 16 bytes) past the last quad of a stage
  return kBarRegion + (size_t)r.stages * tiled_stage_bytes(r.mode, r.NL, r.Cc, r.T + r.Smax, r.G) + 512;
}

// ------------------------------------------------------------------------------------------------
// consumer bodies: one pipeline stage (Cc channels) accumulated into the kRD trials of this thread
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t off16(const uint4& m, int j) {  // j-th 16-bit field of a meta entry
  const uint32_t w = (j >> 1) == 0 ? m.x : (j >> 1) == 1 ? m.y : (j >> 1) == 2 ? m.z : m.w;
  return (j & 1) ? (w >> 16) : (w & 0xffffu);
}

// general modes (kModeGeneral, kModeGeneralReuse, kModeWide): channels in pairs; per channel and trial group the table
// holds kRD 32-bit byte offsets inside the stage, row of the channel included (two 16-byte entries), so an address is one
// add.  REUSE: a trial whose offset equals the previous trial's keeps the registers (one compare, the load predicated
// off).  WIDE: uint16 samples in the 16-bit lanes (add_wide), else packed lanes with headroom (add_pair).
__device__ __forceinline__ uint32_t word_of(const uint4& m, int j) { return j == 0 ? m.x : j == 1 ? m.y : j == 2 ? m.z : m.w; }

// uint16 lanes (kModeWide, NL = 8): a word w holds two uint16 samples with no headroom.  E += w (mod 2^32; one IADD3 for
// two channels) and O += w >> 16 (one LEA.HI per channel) give the lane sums E - (O << 16) and O, exact while the channel
// sum fits 32 bits (checked at plan creation).  Bound by shared memory: 2 bytes per add.
// words of E added by IMADs on the FMA-side pipe (the ALU pipe also carries the shift-adds and the offset compares; the
// kernel is bound by shared memory, 92 % of the wavefront peak): config 4, 0: 256.5 ms, 2: 251.8, 4: 250.7
constexpr int kWideFmaWords = 4;
// (the packed adder of the offsets forms gains nothing from it: reuse form on a coarsened config 3, 84.5 -> 85.4 ms)
__device__ __forceinline__ void add_wide(uint4& E, uint4& O, const uint4& a, const uint4& b, uint32_t one) {
  add_pair_mix<kWideFmaWords>(E, a, b, one);
  O.x += a.x >> 16, O.y += a.y >> 16, O.z += a.z >> 16, O.w += a.w >> 16;
  asm volatile("" : "+r"(O.x), "+r"(O.y), "+r"(O.z), "+r"(O.w));  // keeps each shift-add one LEA.HI
  O.x += b.x >> 16, O.y += b.y >> 16, O.z += b.z >> 16, O.w += b.w >> 16;
}

template <bool REUSE, bool WIDE>
__device__ __forceinline__ void stage_general(uint4 (&acc)[kRD], uint4 (&hi)[kRD], uint32_t sdata, uint32_t smeta, int Cc,
                                              uint32_t meta_row, uint32_t one) {
#pragma unroll 1
  for (int cc = 0; cc < Cc; cc += 2) {
    uint4 ma[2], mb[2];
    lds_sw(ma[0], smeta), lds_sw(ma[1], smeta + 16);
    lds_sw(mb[0], smeta + meta_row), lds_sw(mb[1], smeta + meta_row + 16);
    smeta += 2 * meta_row;
    uint4 wa, wb;
    uint32_t pa = ma[0].x, pb = mb[0].x;
    lds_sw(wa, sdata + pa);
    lds_sw(wb, sdata + pb);
    if constexpr (WIDE) add_wide(acc[0], hi[0], wa, wb, one); else add_pair(acc[0], wa, wb);
#pragma unroll
    for (int j = 1; j < kRD; ++j) {
      const uint32_t oa = word_of(ma[j >> 2], j & 3), ob = word_of(mb[j >> 2], j & 3);
      if constexpr (REUSE) {
        lds_if_ne(wa, sdata + oa, oa, pa);
        lds_if_ne(wb, sdata + ob, ob, pb);
        pa = oa, pb = ob;
      } else {
        lds_sw(wa, sdata + oa);
        lds_sw(wb, sdata + ob);
      }
      if constexpr (WIDE) add_wide(acc[j], hi[j], wa, wb, one); else add_pair(acc[j], wa, wb);
    }
  }
}

// delta mode: channels in quads A..D; one table entry per quad =
//   {changed bits (delta_bit), offA | offB<<16, offC | offD<<16, bit j: some channel of the quad changes at trial step j}
// off = byte offset of the superword of the group's first trial, counted from the start of the stage
__device__ __forceinline__ void sum4(uint4& t, const uint4& a, const uint4& b, const uint4& c, const uint4& d) {
  t.x = a.x + b.x + c.x + d.x;
  t.y = a.y + b.y + c.y + d.y;
  t.z = a.z + b.z + c.z + d.z;
  t.w = a.w + b.w + c.w + d.w;
}
__device__ __forceinline__ void add1(uint4& acc, const uint4& t) {
  acc.x += t.x;
  acc.y += t.y;
  acc.z += t.z;
  acc.w += t.w;
}

template <int J, bool SHARE, bool WIDE>
__device__ __forceinline__ void delta_steps(uint4 (&acc)[kRD], uint4 (&hi)[kRD], uint4& wa, uint4& wb, uint4& wc, uint4& wd, uint4& t4,
                                            uint32_t& aa, uint32_t& ab, uint32_t& ac, uint32_t& ad, uint32_t bits,
                                            uint32_t any, uint32_t one) {
  if constexpr (J < kRD) {
    // A predicated-off LDS still occupies a slot of the shared-memory data pipe (ncu: one wavefront per
    // skipped load, 36 % of the pipe in the first version), so the whole trial step of the quad is skipped
    // by ONE branch on its "any channel changed" bit: neighbouring channels have nearly the same delay
    // curve and often change at the same trial.  `any` sits in a uniform register (stage_delta),
    // which makes this a branch without reconvergence bookkeeping.
    if constexpr (SHARE) {
      if (any & (1u << J)) {
        lds_if_bit<delta_bit(J, 0)>(wa, aa, bits);
        lds_if_bit<delta_bit(J, 1)>(wb, ab, bits);
        lds_if_bit<delta_bit(J, 2)>(wc, ac, bits);
        lds_if_bit<delta_bit(J, 3)>(wd, ad, bits);
        sum4(t4, wa, wb, wc, wd);
      }
    } else {
      // (measured: one uniform branch per channel PAIR instead of per quad skips more predicated-off loads but
      // costs more than it saves: 116.2 vs 111.7 ms on config 3; 109.7 vs 107.0 ms in the SHARE variant.  Staggering
      // the two pairs of the quad by half a trial step, so that a reload is followed by the other pair's adds before
      // its words are needed, doubles the branches and R2Ps: 108.4 vs 100.7 ms.)
      if (any & (1u << J)) {
        lds_if_bit<delta_bit(J, 0)>(wa, aa, bits);
        lds_if_bit<delta_bit(J, 1)>(wb, ab, bits);
        lds_if_bit<delta_bit(J, 2)>(wc, ac, bits);
        lds_if_bit<delta_bit(J, 3)>(wd, ad, bits);
      }
    }
    if constexpr (SHARE) {
      add1(acc[J], t4);  // the quad's sum is unchanged since the last taken step: one term per word
    } else if constexpr (WIDE) {
      add_wide(acc[J], hi[J], wa, wb, one);
      add_wide(acc[J], hi[J], wc, wd, one);
    } else {
      add_pair_mix<kDeltaFmaWords - 4>(acc[J], wa, wb, one);
      add_pair_mix<kDeltaFmaWords>(acc[J], wc, wd, one);
    }
    delta_steps<J + 1, SHARE, WIDE>(acc, hi, wa, wb, wc, wd, t4, aa, ab, ac, ad, bits, any, one);
  }
}

// (the entries of a trial group's quads follow each other: the table pointer advances by a constant)
template <bool SHARE, bool WIDE = false>
__device__ __forceinline__ void stage_delta(uint4 (&acc)[kRD], uint4 (&hi)[kRD], uint32_t sdata, uint32_t smeta, int Cc,
                                            uint32_t one) {
  uint4 m;
  lds_sw(m, smeta);
#pragma unroll 1
  for (int cc = 0; cc < Cc; cc += 4) {
    // byte offsets inside the stage, row of the channel included (16 bits each: choose_tile keeps the data
    // of a delta-mode stage below 64 KB)
    uint32_t aa = sdata + (m.y & 0xffffu);
    uint32_t ab = sdata + (m.y >> 16);
    uint32_t ac = sdata + (m.z & 0xffffu);
    uint32_t ad = sdata + (m.z >> 16);
    const uint32_t bits = m.x;
    // the table entry is the same for the whole warp: a warp reduction hands it over in a uniform register
    const uint32_t any = __reduce_or_sync(0xffffffffu, m.w);
    uint4 wa, wb, wc, wd, t4;
    lds_sw(wa, aa);
    lds_sw(wb, ab);
    lds_sw(wc, ac);
    lds_sw(wd, ad);
    // next quad's entry (the last one reads the first entry of the following stage slot or the pad: unused),
    // fetched now so that its latency hides behind this quad's adds
    smeta += 16;
    lds_sw(m, smeta);
    if constexpr (SHARE) {
      sum4(t4, wa, wb, wc, wd);
      add1(acc[0], t4);
    } else if constexpr (WIDE) {
      add_wide(acc[0], hi[0], wa, wb, one);
      add_wide(acc[0], hi[0], wc, wd, one);
    } else {
      add_pair_mix<kDeltaFmaWords - 4>(acc[0], wa, wb, one);
      add_pair_mix<kDeltaFmaWords>(acc[0], wc, wd, one);
    }
    delta_steps<1, SHARE, WIDE>(acc, hi, wa, wb, wc, wd, t4, aa, ab, ac, ad, bits, any, one);
  }
}

// pair mode (kModeDeltaPair): the packed array holds, per pair v of channels, the two pre-summed rows U_0, U_1 (rows
// 2v, 2v+1).  Per quad A..D of pairs and trial group the table has five 16-byte entries:
//   {changed bits (delta_bit layout), any bits (bit j: some pair of the quad changes at trial step j), 0, 0}
//   then for each pair of the quad eight 16-bit byte offsets (inside the stage, row and U_p selection included), one
//   per trial.  A trial whose bit is clear reuses the registers of the previous trial.
template <int J>
__device__ __forceinline__ void pair_steps(uint4 (&acc)[kRD], uint4& wa, uint4& wb, uint4& wc, uint4& wd, uint32_t sdata,
                                           const uint4& oa, const uint4& ob, const uint4& oc, const uint4& od, uint32_t bits,
                                           uint32_t any) {
  if constexpr (J < kRD) {
    if (any & (1u << J)) {  // uniform (stage_pairs)
      lds_pair_if<delta_bit(J, 0)>(wa, sdata, off16(oa, J), bits);
      lds_pair_if<delta_bit(J, 1)>(wb, sdata, off16(ob, J), bits);
      lds_pair_if<delta_bit(J, 2)>(wc, sdata, off16(oc, J), bits);
      lds_pair_if<delta_bit(J, 3)>(wd, sdata, off16(od, J), bits);
    }
    add_pair(acc[J], wa, wb);
    add_pair(acc[J], wc, wd);
    pair_steps<J + 1>(acc, wa, wb, wc, wd, sdata, oa, ob, oc, od, bits, any);
  }
}

// (Adds on the FMA-side pipe as in the delta form do not pay here: the pair mode is bound by shared memory, 72.2 -> 80.8 ms.)
__device__ __forceinline__ void stage_pairs(uint4 (&acc)[kRD], uint32_t sdata, uint32_t smeta, int Cc, uint32_t meta_row) {
  // Cc = rows of the stage = 2 per pair; a quad of pairs = 8 rows
#pragma unroll 1
  for (int cc = 0; cc < Cc; cc += 8) {
    uint4 m, oa, ob, oc, od;
    lds_sw(m, smeta);
    lds_sw(oa, smeta + 16);
    lds_sw(ob, smeta + 32);
    lds_sw(oc, smeta + 48);
    lds_sw(od, smeta + 64);
    smeta += meta_row;
    const uint32_t any = __reduce_or_sync(0xffffffffu, m.y);
    uint4 wa, wb, wc, wd;
    lds_sw(wa, sdata + off16(oa, 0));
    lds_sw(wb, sdata + off16(ob, 0));
    lds_sw(wc, sdata + off16(oc, 0));
    lds_sw(wd, sdata + off16(od, 0));
    add_pair(acc[0], wa, wb);
    add_pair(acc[0], wc, wd);
    pair_steps<1>(acc, wa, wb, wc, wd, sdata, oa, ob, oc, od, m.x, any);
  }
}

// 8-bit lanes (NL = 16): channels in pairs, one table entry (kRD16 32-bit byte offsets) per channel.
// A loaded word w holds the bytes b0..b3 of four time lanes.  Two accumulators per word:
//   e += w & 0x00ff00ff            two 16-bit lanes: A0 | A2 << 16 (sums of b0 and b2)   LOP3 (ALU pipe) + IMAD (FMA-side pipe)
//   r += w >> 8                    = A1 + 2^8 A2 + 2^16 A3  (mod 2^32)                    one LEA.HI (ALU pipe)
// A2 is known from e, so r - (A2 << 8) = A1 + 2^16 A3 separates exactly as long as every lane sum stays below
// 2^16 (upper bytes moved out every 256 channels, as for the 16-bit lanes); wrap-around of r is harmless.
// The kernel is bound by the ALU pipe (LOP3, LEA.HI, IADD3 all issue there at 2 warp-instructions / clk / SM), so the
// add of the masked word runs on the otherwise idle FMA-side pipe as an IMAD whose multiplier is a kernel parameter
// holding 1 (ptxas folds a literal 1 back into an IADD3): 2 ALU + 1 FMA instruction per word instead of 2.5 ALU.
// Measured (configs 2 / 5): 5.73 -> 5.08 ms / 336.7 -> 297.8 ms; with the two shift-adds forced to stay LEA.HI
// (ptxas otherwise forms SHF + LEA.HI + IMAD.IADD, one more issue slot per pair of words) 4.90 / 286.6 ms.
// (Measured alternatives: the shift-add as IMAD.HI or IMAD.WIDE is slower -- ptxas adds register moves or splits it
// into a multiply plus 64-bit adds; lanes 1 and 3 of one word in four by IDP4A with one-hot selectors into plain
// 32-bit sums, which takes two more instructions off the ALU pipe, is slower too: 5.03 / 294.0 ms.)
__device__ __forceinline__ void add_bytes(uint4& e, uint4& r, const uint4& a, const uint4& b, uint32_t one) {
  e.x = mad1(b.x & 0x00ff00ffu, one, mad1(a.x & 0x00ff00ffu, one, e.x));
  e.y = mad1(b.y & 0x00ff00ffu, one, mad1(a.y & 0x00ff00ffu, one, e.y));
  e.z = mad1(b.z & 0x00ff00ffu, one, mad1(a.z & 0x00ff00ffu, one, e.z));
  e.w = mad1(b.w & 0x00ff00ffu, one, mad1(a.w & 0x00ff00ffu, one, e.w));
  // two dependent (x >> 8) + r steps, kept apart so that each stays one LEA.HI
  r.x += a.x >> 8, r.y += a.y >> 8, r.z += a.z >> 8, r.w += a.w >> 8;
  asm volatile("" : "+r"(r.x), "+r"(r.y), "+r"(r.z), "+r"(r.w));
  r.x += b.x >> 8, r.y += b.y >> 8, r.z += b.z >> 8, r.w += b.w >> 8;
}

__device__ __forceinline__ void stage_bytes(uint4 (&e)[kRD16], uint4 (&r)[kRD16], uint32_t sdata, uint32_t smeta, int Cc,
                                            uint32_t meta_row, uint32_t one) {
#pragma unroll 1
  for (int cc = 0; cc < Cc; cc += 2) {
    uint4 ma, mb;  // byte offsets of the four trials inside the stage (row included): one add per address
    lds_sw(ma, smeta);
    lds_sw(mb, smeta + meta_row);
    smeta += 2 * meta_row;
    uint4 xa, xb;
    lds_sw(xa, sdata + ma.x), lds_sw(xb, sdata + mb.x), add_bytes(e[0], r[0], xa, xb, one);
    lds_sw(xa, sdata + ma.y), lds_sw(xb, sdata + mb.y), add_bytes(e[1], r[1], xa, xb, one);
    lds_sw(xa, sdata + ma.z), lds_sw(xb, sdata + mb.z), add_bytes(e[2], r[2], xa, xb, one);
    lds_sw(xa, sdata + ma.w), lds_sw(xb, sdata + mb.w), add_bytes(e[3], r[3], xa, xb, one);
  }
}

// ------------------------------------------------------------------------------------------------
// per-thread accumulators of the three lane widths
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void carry_save(uint32_t& lo, uint32_t& hi) {  // 16-bit lanes: hi += lo >> 8, lo &= 0xff
  hi += __byte_perm(lo, 0u, 0x4341u);  // bytes 1 and 3 moved down in one PRMT (a shift and a mask are two ALU instructions)
  lo &= 0x00ff00ffu;
}
__device__ __forceinline__ void carry_save(uint4& lo, uint4& hi) {
  carry_save(lo.x, hi.x);
  carry_save(lo.y, hi.y);
  carry_save(lo.z, hi.z);
  carry_save(lo.w, hi.w);
}

template <int NL>
struct Lanes;

template <>
struct Lanes<4> {  // four 32-bit lanes: plain sums
  uint4 acc[kRD];
  __device__ __forceinline__ void init() {
#pragma unroll
    for (int j = 0; j < kRD; ++j) acc[j] = make_uint4(0, 0, 0, 0);
  }
  template <int MODE>
  __device__ __forceinline__ void stage(uint32_t sdata, uint32_t smeta, int Cc, uint32_t meta_row, uint32_t one) {
    if constexpr (is_delta(MODE) || MODE == kModeHybrid)  // (a hybrid range: this call is one of its delta-coded chunks)
      stage_delta<MODE == kModeDeltaShare>(acc, acc, sdata, smeta, Cc, one);
    else
      stage_general<MODE == kModeGeneralReuse, false>(acc, acc, sdata, smeta, Cc, meta_row, one);
  }
  template <int MODE>
  __device__ __forceinline__ void stage_rest(uint32_t sdata, uint32_t smeta, int Cc, uint32_t meta_row, uint32_t one) {  // hybrid: the other chunks
    stage_general<true, false>(acc, acc, sdata, smeta, Cc, meta_row, one);
  }
  __device__ __forceinline__ void flush() {}
  template <int MODE>
  __device__ __forceinline__ void values(int j, uint32_t (&v)[4]) const {
    v[0] = acc[j].x, v[1] = acc[j].y, v[2] = acc[j].z, v[3] = acc[j].w;
  }
};

template <>
struct Lanes<8> {  // eight 16-bit lanes, value = lo + 256*hi
  uint4 acc[kRD], hi[kRD];
  __device__ __forceinline__ void init() {
#pragma unroll
    for (int j = 0; j < kRD; ++j) acc[j] = hi[j] = make_uint4(0, 0, 0, 0);
  }
  template <int MODE>
  __device__ __forceinline__ void stage(uint32_t sdata, uint32_t smeta, int Cc, uint32_t meta_row, uint32_t one) {
    if constexpr (MODE == kModeWide)
      stage_general<true, true>(acc, hi, sdata, smeta, Cc, meta_row, one);  // acc = E, hi = O
    else if constexpr (MODE == kModeDeltaPair)
      stage_pairs(acc, sdata, smeta, Cc, meta_row);
    else if constexpr (is_delta(MODE) || is_hybrid(MODE))  // (a hybrid range: this call is one of its delta-coded chunks)
      stage_delta<MODE == kModeDeltaShare, MODE == kModeWideHybrid>(acc, hi, sdata, smeta, Cc, one);
    else
      stage_general<MODE == kModeGeneralReuse, false>(acc, hi, sdata, smeta, Cc, meta_row, one);
  }
  template <int MODE>
  __device__ __forceinline__ void stage_rest(uint32_t sdata, uint32_t smeta, int Cc, uint32_t meta_row, uint32_t one) {  // hybrid: the other chunks
    stage_general<true, MODE == kModeWideHybrid>(acc, hi, sdata, smeta, Cc, meta_row, one);
  }
  __device__ __forceinline__ void flush() {
#pragma unroll
    for (int j = 0; j < kRD; ++j) carry_save(acc[j], hi[j]);
  }
  template <int MODE>
  __device__ __forceinline__ void values(int j, uint32_t (&v)[8]) const {
    const uint32_t lo[4] = {acc[j].x, acc[j].y, acc[j].z, acc[j].w}, up[4] = {hi[j].x, hi[j].y, hi[j].z, hi[j].w};
    if constexpr (is_wide(MODE)) {  // acc = E = sum of the words, hi = O = sum of their upper halves
#pragma unroll
      for (int q = 0; q < 4; ++q) v[2 * q] = lo[q] - (up[q] << 16), v[2 * q + 1] = up[q];
    } else {
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        v[2 * q] = (lo[q] & 0xffffu) + ((up[q] & 0xffffu) << 8);
        v[2 * q + 1] = (lo[q] >> 16) + ((up[q] >> 16) << 8);
      }
    }
  }
};

template <>
struct Lanes<16> {  // sixteen 8-bit lanes: e, r as in add_bytes; he, hq the upper bytes moved out at each flush
  uint4 e[kRD16], r[kRD16], he[kRD16], hq[kRD16];
  __device__ __forceinline__ void init() {
#pragma unroll
    for (int j = 0; j < kRD16; ++j) e[j] = r[j] = he[j] = hq[j] = make_uint4(0, 0, 0, 0);
  }
  template <int MODE>
  __device__ __forceinline__ void stage(uint32_t sdata, uint32_t smeta, int Cc, uint32_t meta_row, uint32_t one) {
    stage_bytes(e, r, sdata, smeta, Cc, meta_row, one);
  }
  template <int MODE>
  __device__ __forceinline__ void stage_rest(uint32_t, uint32_t, int, uint32_t, uint32_t) {}  // (no hybrid form on 8-bit lanes)
  // invariant: e = A0 | A2 << 16,  r = A1 + 2^8 A2 + 2^16 A3 (mod 2^32),  lane sum = A + 256 * (he | hq lane)
  static __device__ __forceinline__ void flush_word(uint32_t& e, uint32_t& r, uint32_t& he, uint32_t& hq) {
    uint32_t q = r - ((e >> 16) << 8);  // A1 | A3 << 16
    carry_save(e, he);
    carry_save(q, hq);
    r = q + ((e >> 16) << 8);
  }
  __device__ __forceinline__ void flush() {
#pragma unroll
    for (int j = 0; j < kRD16; ++j) {
      flush_word(e[j].x, r[j].x, he[j].x, hq[j].x);
      flush_word(e[j].y, r[j].y, he[j].y, hq[j].y);
      flush_word(e[j].z, r[j].z, he[j].z, hq[j].z);
      flush_word(e[j].w, r[j].w, he[j].w, hq[j].w);
    }
  }
  template <int MODE>
  __device__ __forceinline__ void values(int j, uint32_t (&v)[16]) const {
    const uint32_t ew[4] = {e[j].x, e[j].y, e[j].z, e[j].w}, rw[4] = {r[j].x, r[j].y, r[j].z, r[j].w};
    const uint32_t hew[4] = {he[j].x, he[j].y, he[j].z, he[j].w}, hqw[4] = {hq[j].x, hq[j].y, hq[j].z, hq[j].w};
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const uint32_t q = rw[w] - ((ew[w] >> 16) << 8);
      v[4 * w + 0] = (ew[w] & 0xffffu) + ((hew[w] & 0xffffu) << 8);
      v[4 * w + 1] = (q & 0xffffu) + ((hqw[w] & 0xffffu) << 8);
      v[4 * w + 2] = (ew[w] >> 16) + ((hew[w] >> 16) << 8);
      v[4 * w + 3] = (q >> 16) + ((hqw[w] >> 16) << 8);
    }
  }
};

// ------------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------------
// STATS: also accumulate sum x and sum x^2 of every row written (dd_plan_set_row_stats); a separate instantiation so
// that the default kernel keeps its register allocation (measured: 0.4 % on config 3 with a run-time flag)
template <int NL, int MODE, int NT, bool STATS = false>
__global__ void __launch_bounds__(NT, 512 / NT) dd_tiled_kernel(const TiledParams p) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int tid = threadIdx.x;
  // CTA -> (trial block fastest, time tile, beam): CTAs resident together share a time tile in L2
  const long long lin = blockIdx.x;
  const int blk = p.blk0 + (int)(lin % p.nblk);
  const long long rest = lin / p.nblk;
  const long long tau = rest % p.ntau;
  const int beam = (int)(rest / p.ntau);

  const uint32_t bar_base = smem_u32(smem);  // full[s] at +8*s, empty[s] at +8*(nstages+s)
  const int nstages = p.nstages;
  const uint32_t row_bytes = (uint32_t)p.rowpitch * kSuperwordBytes;
  const uint32_t data_bytes = (uint32_t)p.Cc * row_bytes;
  const uint32_t meta_bytes = (uint32_t)tiled_meta_bytes(MODE, NL, p.Cc, p.G);
  // hybrid ranges: chunks 0 .. nd-1 (the highest channels, whose delay steps never exceed 1) carry the delta table, the
  // others the offsets table; a trial block's slices lie in that order
  const uint32_t meta_bytes_d = (uint32_t)tiled_meta_bytes(kModeDelta, NL, p.Cc, p.G);
  const int nd = is_hybrid(MODE) ? p.nd : 0;
  const uint32_t stage_bytes = (uint32_t)tiled_stage_bytes(MODE, NL, p.Cc, p.rowpitch, p.G);
  const uint32_t stage0 = bar_base + kBarRegion;
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
  // one for the chunk's table slice, landing in stage k % nstages and signalling full[stage] with the
  // byte count.  A warp issues chunk k when it starts iteration k - ahead (ahead = nstages - 2): the
  // stage it refills was consumed two iterations ago, so the wait on its empty barrier is normally
  // already satisfied.  Row start and length of the warp's NEXT chunk are fetched one turn early.
  const uint4* Pbeam = p.P + (long long)beam * p.Cpad * p.Wp + tau * p.T;
  const long long tab = (long long)blk * p.Cpad;
  const char* meta_blk = reinterpret_cast<const char*>(p.meta) +
                         (size_t)blk * ((size_t)nd * meta_bytes_d + (size_t)(nchunks - nd) * meta_bytes);
  const int lane = tid & 31;
  const int warp = tid >> 5;
  constexpr int kWarps = NT / 32;
  const int ahead = nstages - 2;
  int pf_d0 = 0, pf_row = 0;
  uint32_t pf_bytes = 0;
  auto prefetch = [&](int k) {
    pf_bytes = 0;
    if (k < nchunks && lane < p.Cc) {
      const int c = k * p.Cc + lane;
      pf_d0 = __ldg(p.dmin + tab + c);
      pf_bytes = (uint32_t)(p.T + __ldg(p.span + tab + c)) * kSuperwordBytes;
      pf_row = p.chan ? __ldg(p.chan + tab + c) : c;
    }
  };
  // stage and wrap count of a chunk index are tracked incrementally (no divisions in the main loop)
  auto produce = [&](int k, int s, uint32_t wraps) {  // s = k % nstages, wraps = k / nstages
    if (wraps > 0) mbar_wait(bar_base + 8u * (nstages + s), (wraps & 1u) ^ 1u);
    const uint32_t sbase = stage0 + (uint32_t)s * stage_bytes;
    const uint32_t full = bar_base + 8u * s;
    uint32_t total = pf_bytes;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) total += __shfl_xor_sync(0xffffffffu, total, o);
    if (lane == 0) {
      const uint32_t mb = k < nd ? meta_bytes_d : meta_bytes;
      const size_t moff = k < nd ? (size_t)k * meta_bytes_d : (size_t)nd * meta_bytes_d + (size_t)(k - nd) * meta_bytes;
      mbar_arrive_expect_tx(full, total + mb);
      bulk_copy_g2s(sbase + data_bytes, meta_blk + moff, mb, full);
    }
    __syncwarp();
    if (lane < p.Cc)
      bulk_copy_g2s(sbase + lane * row_bytes, Pbeam + (long long)pf_row * p.Wp + pf_d0, pf_bytes, full);
  };
  // this warp's chunks are warp, warp + kWarps, ...; (my_k, my_s, my_w) is the next one it has to issue
  int my_k = warp, my_s = warp % nstages;
  uint32_t my_w = (uint32_t)(warp / nstages);
  const int s_step = kWarps % nstages;
  const uint32_t w_step = (uint32_t)(kWarps / nstages);
  auto advance = [&]() {
    my_k += kWarps;
    my_s += s_step;
    my_w += w_step;
    if (my_s >= nstages) {
      my_s -= nstages;
      ++my_w;
    }
  };
  // prologue: chunks 0 .. ahead-1
  while (my_k < ahead && my_k < nchunks) {
    prefetch(my_k);
    produce(my_k, my_s, my_w);
    advance();
  }
  prefetch(my_k);  // first chunk this warp issues inside the loop

  // ---------------- consumers: RD trials x one superword (NL time lanes) per thread --------------
  constexpr int RD = trials_per_thread(NL);
  const int g = tid / p.T;       // trial group inside the CTA (warp-uniform: T is a multiple of 32)
  const int ti = tid - g * p.T;  // superword inside the time tile
  Lanes<NL> lanes;
  lanes.init();
  const uint32_t thread_off = (uint32_t)ti * kSuperwordBytes;
  const uint32_t entry_bytes = MODE == kModeDeltaPair ? 80u : (!is_delta(MODE) && NL != 16) ? 32u : 16u;  // table bytes per (channel | quad, trial group)
  const uint32_t meta_row = (uint32_t)p.G * entry_bytes;             // bytes between consecutive channels (quads)
  // delta form: [trial group][quad] entries of 16 bytes; the other forms: [channel | quad of pairs][trial group]
  const uint32_t meta_off_d = data_bytes + (uint32_t)g * (uint32_t)(p.Cc / 4) * 16u;
  const uint32_t meta_off = (is_delta(MODE) && MODE != kModeDeltaPair) ? meta_off_d : data_bytes + (uint32_t)g * entry_bytes;
  int since_flush = 0;
  // The last trial block of a range is padded to the block size (2000 trials = 31 blocks of 64 + 16): the trial groups of
  // a CTA that hold no real trial (warp-uniform: T is a multiple of 32) skip the adds, which leaves the SM's issue slots
  // to the others (config 3: 99.0 -> 95.6 ms).
  // (Not in the pair mode: there the extra live value costs a register spill in the loop, 71.4 -> 79.4 ms.)
  const bool group_live = MODE == kModeDeltaPair || (blk * p.G + g) * RD < p.ndm;

  int s = 0;        // stage of the chunk being consumed
  uint32_t ph = 0;  // its full-barrier parity
  for (int it = 0; it < nchunks; ++it) {
    if (it + ahead == my_k && my_k < nchunks) {  // producer turn of this warp
      produce(my_k, my_s, my_w);
      advance();
      prefetch(my_k);
    }
    const uint32_t sbase = stage0 + (uint32_t)s * stage_bytes;
    if (group_live) {
      mbar_wait(bar_base + 8u * s, ph);
      if constexpr (is_hybrid(MODE)) {
        if (it < nd)
          lanes.template stage<MODE>(sbase + thread_off, sbase + meta_off_d, p.Cc, meta_row, p.one);
        else
          lanes.template stage_rest<MODE>(sbase + thread_off, sbase + meta_off, p.Cc, meta_row, p.one);
      } else {
        lanes.template stage<MODE>(sbase + thread_off, sbase + meta_off, p.Cc, meta_row, p.one);
      }
    } else {
      mbar_wait_relaxed(bar_base + 8u * s, ph);  // keeps the barrier protocol and its producer turns only
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_base + 8u * (nstages + s));  // stage may be refilled
    if (++s == nstages) {
      s = 0;
      ph ^= 1u;
    }
    if (NL != 4 && !is_wide(MODE) && ++since_flush == p.flush_stages) {  // packed lanes could overflow next: move their upper bytes
      since_flush = 0;
      lanes.flush();
    }
  }

  // ---------------- a4: DM-time writer, fp32 (I2F rounds to nearest even) -------------------------
  const long long i = tau * p.T + ti;
  const bool active = i < p.H;  // (with STATS threads past the lane segment keep running: the sums reduce over whole warps)
  if (!active && !STATS) return;
  float* obase = p.out + (long long)beam * p.out_beam_stride;
#pragma unroll
  for (int j = 0; j < RD; ++j) {
    const int jj = (blk * p.G + g) * RD + j;
    if (jj >= p.ndm) break;  // warp-uniform
    float* orow = obase + (long long)jj * p.pitch;
    uint32_t v[NL];
    lanes.template values<MODE>(j, v);
    unsigned long long s1 = 0, s2 = 0;
#pragma unroll
    for (int m = 0; m < NL; ++m) {
      const long long t = i + (long long)m * p.H;  // consecutive threads -> consecutive floats
      if ((!STATS || active) && t < p.nout) {
        // second byte plane of uint16 input: S = S_lo + 256*S_hi.  Both plane sums are < 2^24, hence exact
        // floats, and the fused multiply-add rounds the exact total once: fl32(S), as the definition asks.
        if (p.accum_scale != 0.0f)
          orow[t] = __fmaf_rn(__uint2float_rn(v[m]), p.accum_scale, orow[t]);
        else
          orow[t] = __uint2float_rn(v[m]);
        if constexpr (STATS) {
          s1 += v[m];
          s2 += (unsigned long long)v[m] * v[m];
        }
      }
    }
    if constexpr (STATS) {  // sum x, sum x^2 of this row's piece: one pair of atomics per warp and trial (exact integers)
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        s1 += __shfl_down_sync(0xffffffffu, s1, o);
        s2 += __shfl_down_sync(0xffffffffu, s2, o);
      }
      if (lane == 0) {
        unsigned long long* st = p.stats + (long long)beam * p.stats_beam_stride + 2ll * jj;
        atomicAdd(st, s1);
        atomicAdd(st + 1, s2);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// launcher
// ------------------------------------------------------------------------------------------------
template <int NL, int MODE, int NT>
static cudaError_t launch_tiled_t(const TiledParams& tp, long long nctas, size_t smem, cudaStream_t stream) {
  if (tp.stats) {
    if constexpr (NL != 16)  // (row statistics are offered for uint8 input only, whose byte-lane ranges have one plane)
      dd_tiled_kernel<NL, MODE, NT, true><<<(unsigned)nctas, NT, smem, stream>>>(tp);
    else
      dd_tiled_kernel<16, MODE, NT, true><<<(unsigned)nctas, NT, smem, stream>>>(tp);
  } else {
    dd_tiled_kernel<NL, MODE, NT><<<(unsigned)nctas, NT, smem, stream>>>(tp);
  }
  return cudaGetLastError();
}

template <int NL, int MODE, int NT>
static cudaError_t set_smem_t() {
  cudaError_t e = cudaFuncSetAttribute(dd_tiled_kernel<NL, MODE, NT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(dd_tiled_kernel<NL, MODE, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
}

#define DD_FOR_ALL_TILED(X)                                                                    \
  X(8, kModeGeneral, 256) X(8, kModeGeneralReuse, 256) X(8, kModeDelta, 256)                   \
  X(8, kModeGeneral, 512) X(8, kModeGeneralReuse, 512) X(8, kModeDelta, 512)                   \
  X(8, kModeDeltaShare, 256) X(8, kModeDeltaShare, 512) X(4, kModeDeltaShare, 256) X(4, kModeDeltaShare, 512) \
  X(8, kModeDeltaPair, 256) X(8, kModeDeltaPair, 512) X(8, kModeWide, 256) X(8, kModeWide, 512)  \
  X(8, kModeHybrid, 256) X(8, kModeHybrid, 512) X(4, kModeHybrid, 256) X(4, kModeHybrid, 512)   \
  X(8, kModeWideHybrid, 256) X(8, kModeWideHybrid, 512)                                        \
  X(4, kModeGeneral, 256) X(4, kModeGeneralReuse, 256) X(4, kModeDelta, 256)                   \
  X(4, kModeGeneral, 512) X(4, kModeGeneralReuse, 512) X(4, kModeDelta, 512)                   \
  X(16, kModeGeneral, 256) X(16, kModeGeneral, 512)

cudaError_t configure_kernels(const dd_plan*) {
  cudaError_t e;
#define DD_CFG(NL, MODE, NT) \
  if ((e = set_smem_t<NL, MODE, NT>()) != cudaSuccess) return e;
  DD_FOR_ALL_TILED(DD_CFG)
#undef DD_CFG
  return cudaSuccess;
}

cudaError_t launch_tiled(const dd_plan* p, const RangePlan& r, float* out_dev, cudaStream_t stream, int blk0, int nblk) {
  if (nblk <= 0) nblk = r.nblocks - blk0;
  if (blk0 < 0 || nblk <= 0 || blk0 + nblk > r.nblocks) return cudaErrorInvalidValue;
  const bool pairs = use_pairs(p, r);
  TiledParams tp;
  tp.meta = pairs ? r.d_meta2 : r.d_meta;
  tp.dmin = pairs ? r.d_dmin2 : r.d_dmin;
  tp.span = pairs ? r.d_span2 : r.d_span;
  tp.chan = pairs ? r.d_chan2 : r.d_chan;
  tp.out = out_dev + r.offset;
  tp.out_beam_stride = p->beam_stride;
  tp.pitch = r.pitch;
  tp.Wp = r.Wp;
  tp.H = r.H;
  tp.nout = r.nout;
  tp.ntau = r.ntau;
  tp.ndm = r.ndm;
  tp.Cpad = r.Cpad;  // rows of the packed array the kernel walks (pairs: the two pre-summed rows of each pair)
  tp.G = r.G;
  tp.T = r.T;
  tp.Cc = r.Cc;
  tp.nstages = pairs ? r.stages2 : r.stages;
  tp.nd = r.nd;
  tp.blk0 = blk0;
  tp.nblk = nblk;
  tp.rowpitch = pairs ? r.T + r.Smax2 : r.T + r.Smax;
  tp.stats = (p->row_stats && r.planes == 1) ? p->row_stats + 2 * r.row0 : nullptr;
  tp.stats_beam_stride = 2 * p->rows_per_beam;
  tp.one = 1u;
  tp.flush_stages = r.flush > 0 ? r.flush / r.Cc : 0;  // pairs: a stage holds Cc/2 pair sums of twice the size: same interval
  const long long nctas = (long long)nblk * r.ntau * p->nbeams;
  if (nctas <= 0 || nctas > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
  const size_t smem = pairs ? kBarRegion + (size_t)r.stages2 * tiled_stage_bytes(kModeDeltaPair, r.NL, r.Cc, tp.rowpitch, r.G) + 512
                            : tiled_smem_bytes(r);
  const int nt = r.G * r.T;
  const int mode = pairs ? (int)kModeDeltaPair
                   : (r.mode == kModeDelta && (p->variant == DD_KERNEL_SHARED || p->variant == DD_KERNEL_SUBBAND))
                       ? (int)kModeDeltaShare
                       : r.mode;
  // one launch per byte plane: low bytes stored, high bytes added with weight 256
  for (int plane = 0; plane < r.planes; ++plane) {
    tp.P = reinterpret_cast<const uint4*>(static_cast<const char*>(p->ws) + (pairs ? r.ws2_offset : r.ws_offset + plane * r.plane_bytes));
    tp.accum_scale = plane == 0 ? 0.0f : 256.0f;
    cudaError_t e = cudaErrorInvalidConfiguration;
#define DD_GO(NL_, MODE_, NT_) \
  if (r.NL == NL_ && mode == MODE_ && nt == NT_) e = launch_tiled_t<NL_, MODE_, NT_>(tp, nctas, smem, stream);
    DD_FOR_ALL_TILED(DD_GO)
#undef DD_GO
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace dd
