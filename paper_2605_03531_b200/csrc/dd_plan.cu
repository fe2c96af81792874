// dd_plan.cu -- host side of libdd: the C ABI of include/dd.h, the plan / delay-table builder
// (step a1 of SURVEY.md 8(a)) and the execute sequencing.  No torch types, no exceptions across
// the boundary.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <limits.h>

#include <algorithm>
#include <new>
#include <string>
#include <vector>

#include "dd_internal.h"

namespace {

thread_local std::string g_last_cuda_error;

}  // namespace

// Records the text dd_last_cuda_error() returns (per thread) and yields DD_ERR_CUDA; shared by every source file.
int dd::cuda_fail(cudaError_t e, const char* what) {
  g_last_cuda_error = std::string(what) + ": " + cudaGetErrorString(e);
  return DD_ERR_CUDA;
}

namespace {
using dd::cuda_fail;
#define DD_CUDA(call)                                      \
  do {                                                     \
    cudaError_t e__ = (call);                              \
    if (e__ != cudaSuccess) return cuda_fail(e__, #call);  \
  } while (0)

// Dispersion constant of the north_star, s MHz^2 cm^3 / pc  (PAPER.md:258 prints 4.14881 ms GHz^2).
constexpr double kDispersion = 4.148808e3;
constexpr int kSmCount = 148;  // B200 (the library is built for sm_100a only); used by the tile cost model

inline int64_t round_up(int64_t a, int64_t b) { return (a + b - 1) / b * b; }

// a1: d_r(c,j) = round(K * DM_j * (f_c^-2 - f_top^-2) / (tsamp*decim)), double precision, half away
// from zero (the argument is never negative).  PAPER.md:258 Eq. 1.1; readings A1, A4, A6.
bool build_delays(const dd_plan& p, dd::RangePlan& r) {
  const double ts = p.tsamp * (double)r.decim;
  const double inv_top = 1.0 / (p.f_top * p.f_top);
  r.delays.resize((size_t)r.ndm * p.nchans);
  for (int j = 0; j < r.ndm; ++j) {
    const double dm = r.dm_lo + (double)j * r.dm_step;
    for (int c = 0; c < p.nchans; ++c) {
      const double f = p.f_top + (double)c * p.cw;
      const double x = kDispersion * dm * (1.0 / (f * f) - inv_top) / ts;
      const double d = floor(x + 0.5);
      if (!(d >= 0.0) || d > 2.0e9) return false;
      r.delays[(size_t)j * p.nchans + c] = (int32_t)d;
    }
  }
  return true;
}

struct TileChoice {
  int G, T, Cc, stages;
};

// "auto" tuning: what dd_plan_create uses (dd_plan_create_tuned passes the caller's overrides instead)
const dd_tuning_t kAutoTuning = {-1, -1, 0, 0, 0, 0};

// Delay spread of one trial block: d(c, last) - d(c, first); delays are non-decreasing in j.
inline int block_spread(const dd_plan& p, const dd::RangePlan& r, int blk, int Dcta, int c) {
  const int j0 = blk * Dcta;
  const int j1 = std::min(r.ndm - 1, j0 + Dcta - 1);
  return r.delays[(size_t)j1 * p.nchans + c] - r.delays[(size_t)j0 * p.nchans + c];
}

// Superwords a staged row of (trial block, channel) holds beyond the time tile: rows start at the block's first
// delay rounded DOWN to a 128-byte line (8 superwords) and end on a line (build_tables computes the same value).
inline int block_span(const dd_plan& p, const dd::RangePlan& r, int blk, int Dcta, int c) {
  const int j0 = blk * Dcta;
  const int j1 = std::min(r.ndm - 1, j0 + Dcta - 1);
  const int d0 = r.delays[(size_t)j0 * p.nchans + c] & ~7;
  return (int)round_up(r.delays[(size_t)j1 * p.nchans + c] - d0, 8);
}

// Largest block_span over ALL (trial block, channel): the row pitch of the staged rows is T + this.  Delays are
// rounded per channel, so the widest row is not always the lowest channel's (its spread can be one sample short of
// a neighbour's, and the start alignment d0 & 7 differs per channel).
int max_block_span(const dd_plan& p, const dd::RangePlan& r, int Dcta) {
  const int nblocks = (r.ndm + Dcta - 1) / Dcta;
  int smax = 0;
  for (int b = 0; b < nblocks; ++b)
    for (int c = 0; c < p.nchans; ++c) smax = std::max(smax, block_span(p, r, b, Dcta, c));
  return smax;
}

// Which table form the tiled kernel uses for this range (dd_internal.h TiledMode).  Trial groups are the
// kRD-aligned runs of trials counted from the start of the range.  *delta_prefix = number of leading channels
// (highest frequencies) none of whose delay steps inside a trial group exceeds 1: the whole range is delta-coded when
// that is every channel, and a hybrid range delta-codes the channel chunks inside that prefix.
int choose_mode(const dd_plan& p, const dd::RangePlan& r, const dd_tuning_t& tune, int* delta_prefix) {
  int64_t same = 0, total = 0;
  int prefix = p.nchans;  // first channel with a step above 1 (delays grow with the channel index, so do their steps)
  for (int j = 0; j + 1 < r.ndm; ++j) {
    if ((j + 1) % dd::kRD == 0) continue;  // first trial of a group always loads
    const int32_t* d0 = &r.delays[(size_t)j * p.nchans];
    const int32_t* d1 = d0 + p.nchans;
    for (int c = 0; c < p.nchans; ++c) {
      const int32_t inc = d1[c] - d0[c];
      same += inc == 0;
      if (inc > 1 && c < prefix) prefix = c;
    }
    total += p.nchans;
  }
  const bool delta = prefix == p.nchans;
  *delta_prefix = prefix;
  int mode = delta ? dd::kModeDelta : (total > 0 && (double)same / (double)total >= 0.25) ? dd::kModeGeneralReuse
                                                                                         : dd::kModeGeneral;
  if (tune.mode >= 0 && tune.mode <= 2) mode = tune.mode;  // dd_plan_create_tuned; delta is refused when it does not apply
  if (mode == dd::kModeDelta && !delta) mode = dd::kModeGeneral;
  return mode;
}

// Pick the tile shape of the tiled kernel for one range: more trials per CTA amortise the
// L2 -> shared-memory fill of a channel row over more adds, but widen the staged window by the delay
// spread of the block.  Cost model: staged bytes per add; constraint: >= 3 stages in 200 KB.
void choose_tile(const dd_plan& p, dd::RangePlan& r, const dd_tuning_t& tune) {
  // 16-bit lanes hold lo + 256*hi exactly when (a) 255 + flush*maxval <= 65535 between flushes and (b) the
  // hi lanes, which gain at most 255 per flush, stay below 65536: at most 256 flushes.
  const int maxval = ((1 << p.in_bits) - 1) * r.decim;
  const int flush0 = 65280 / maxval;
  if (maxval <= 4095 && (int64_t)p.nchans <= (int64_t)120 * flush0) {
    r.NL = 8;
    r.flush = flush0;
  } else {
    r.NL = 4;
    r.flush = 0;
  }
  int delta_prefix = 0;
  r.mode = choose_mode(p, r, tune, &delta_prefix);
  r.nd = 0;
  // Hybrid (dd_internal.h kModeHybrid): not delta-codable as a whole, but a leading part of the channels is.  Taken
  // automatically for DECIMATED ranges when that part is at least a tenth of the channels: there the alternative is the
  // offsets table alone (measured on config 3 with DM steps 0.22 / 0.45 / 0.9, lowest-channel delay steps of 1.06-1.09
  // samples per trial, 96 % of the channels delta-coded: x2 21.1 -> 18.4 ms, x4 17.9 -> 15.7 ms; config 4's x8 range,
  // 40 % delta-coded: 21.1 -> 19.6 ms).  Undecimated ranges keep the 8-bit-lane kernel (uint8; 35.6 ms against 36.6 ms
  // hybrid in the same experiment: near the limit of the delta form half of all trial steps reload, and it is bound by
  // shared memory like the offsets form) or the uint16-lane kernel (uint16; config 4 range 0: 236.3 against 236.1 ms).
  // dd_tuning_t::mode = 6 asks for it wherever a chunk qualifies.
  bool hybrid = false;
  if (r.mode != dd::kModeDelta && (tune.mode < 0 || tune.mode == 6) && delta_prefix >= 4)
    hybrid = tune.mode == 6 || (r.decim > 1 && (double)delta_prefix >= 0.10 * (double)p.nchans);
  // Undecimated ranges that cannot use the delta table run on 8-bit lanes: half the shared-memory traffic per
  // sample (the bound of the offsets-table modes), uint16 input as two byte planes.  dd_tuning_t::byte_lanes = 0
  // switches it off.
  const int flush16 = 65280 / 255;
  if (hybrid && !(p.in_bits == 16 && r.decim == 1 && tune.byte_lanes < 0)) {
    r.mode = dd::kModeHybrid;  // lanes as chosen above (16-bit with headroom, or 32-bit)
  } else if (p.in_bits == 16 && r.decim == 1 && r.mode != dd::kModeDelta && tune.byte_lanes < 0) {
    // undecimated uint16 input on a coarse grid: the samples themselves in 16-bit lanes (kModeWide).  Shared memory
    // delivers 2 bytes per add either way, but one pass with 1.5 ALU instructions per two adds replaces two byte-plane
    // passes of the 8-bit-lane kernel.  dd_tuning_t::byte_lanes = 1 keeps the two byte planes, 0 the 32-bit lanes.
    r.NL = 8;
    r.flush = 0;
    r.mode = hybrid ? dd::kModeWideHybrid : dd::kModeWide;
  } else if (r.decim == 1 && r.mode != dd::kModeDelta && (int64_t)p.nchans <= (int64_t)120 * flush16 && tune.byte_lanes != 0) {
    r.NL = 16;
    r.flush = flush16;
    r.mode = dd::kModeGeneral;
    r.planes = p.in_bits / 8;
  }
  r.RD = dd::trials_per_thread(r.NL);
  static const int cand[][2] = {{16, 32}, {8, 64}, {4, 128}, {2, 256}, {1, 512}, {8, 32}, {4, 64}, {2, 128}, {1, 256}};
  const size_t budget = 200 * 1024;
  // One candidate shape: does it fit (16-bit offsets, 64 KB of delta byte offsets, >= min_stages ring slots in
  // `budget`), with how many stages, at what cost.  The automatic choice and a forced tile (dd_tuning_t) go
  // through the same checks.
  auto evaluate = [&](int G, int T, int Cc, int smax, double smean, int nblocks, int min_stages, int* stages_out,
                      double* cost_out) -> bool {
    const int D = G * r.RD;
    if (T + smax > 65535) return false;  // 16-bit offsets
    if (r.flush > 0 && Cc > r.flush) return false;
    if ((r.mode == dd::kModeDelta || dd::is_hybrid(r.mode)) && (size_t)Cc * (size_t)(T + smax) * 16 > 65536)
      return false;  // 16-bit byte offsets of the delta table
    const size_t stage = (size_t)Cc * (size_t)(T + smax) * 16 + dd::tiled_meta_bytes(r.mode, r.NL, Cc, G);
    const int stages = (int)std::min<size_t>(6, budget / stage);
    if (stages < min_stages) return false;
    // bytes staged per add: row (T + mean spread) superwords + the table row, over T*NL*D adds
    double cost = ((T + smean) * 16.0 + dd::tiled_meta_bytes(r.mode, r.NL, 4, G) / 4.0) / ((double)T * r.NL * D);
    // The delta form is not bound by the fill of its stages (config 3: 0.02 - 0.04 staged bytes per add, 1 - 1.5 TB/s out
    // of L2) but by issue slots and shared-memory wavefronts, which grow with the share of quad steps that reload; shorter
    // trial blocks let the channel dealing of build_tables match delay phases over fewer trials and halve the table.  So
    // below a floor the staged bytes do not count and the shorter block wins.  Measured, 64 x 64 against 128 x 32 trials x
    // superwords: config 3 99.1 / 100.5 ms, 2048 channels 50.7 / 52.4, 327 us sampling 95.5 / 98.8, a 300-500 MHz band
    // 77.9 / 78.9 (32 x 128 needs 16-channel stages for its 16-bit offsets: 105.1).
    if (r.mode == dd::kModeDelta || dd::is_hybrid(r.mode)) cost = std::max(cost, 0.05) * (1.0 + 0.02 * (double)D / 128.0);
    // trials past the end of the last block are computed and dropped
    cost *= (double)nblocks * D / (double)r.ndm;
    if (G * T == 256) cost *= 1.02;  // mild preference for the 512-thread CTA at equal cost
    if (Cc < 16) cost *= 1.0 + 0.05 * (16 / Cc - 1);  // shorter stages synchronise more often
    {
      // wave quantisation: a grid that is not a multiple of the SM count leaves SMs idle in its last wave.  It only
      // matters for short rows (the tail plans of dd_stream_push at 800-spectra blocks: a few dozen CTAs).
      const int64_t H = round_up((r.nout + r.NL - 1) / r.NL, 16);
      const int64_t nctas = (int64_t)nblocks * ((H + T - 1) / T) * p.nbeams;
      const int64_t slots = (int64_t)kSmCount * (G * T == 256 ? 2 : 1);
      cost *= (double)((nctas + slots - 1) / slots * slots) / (double)nctas;
    }
    *stages_out = stages;
    *cost_out = cost;
    return true;
  };
  auto spreads = [&](int D, int* smax, double* smean) {
    const int nblocks = (r.ndm + D - 1) / D;
    double ssum = 0;
    const int cstep = std::max(1, p.nchans / 64);
    int nsamp = 0;
    for (int b = 0; b < nblocks; ++b)
      for (int c = 0; c < p.nchans; c += cstep, ++nsamp) ssum += block_spread(p, r, b, D, c);
    *smax = max_block_span(p, r, D);
    *smean = ssum / std::max(1, nsamp) + 7.0;  // rows start and end on 128-byte lines
    return nblocks;
  };
  double best = 1e300;
  TileChoice bc = {1, 256, 4, 2};
  bool found = false;
  const bool forced = tune.trial_groups > 0 || tune.words_per_cta > 0 || tune.chans_per_stage > 0 || tune.stages > 0;
  if (forced) {
    // dd_plan_create_tuned: a caller-chosen shape, accepted only if it is a shape the kernels are built for and it
    // passes the checks of the automatic path (the ring depth may be lowered to what fits)
    const int G = tune.trial_groups, T = tune.words_per_cta, Cc = tune.chans_per_stage;
    if (G >= 1 && T >= 32 && T % 32 == 0 && (G * T == 256 || G * T == 512) && Cc >= 4 && Cc <= 32 && Cc % 4 == 0 &&
        tune.stages >= 2 && tune.stages <= 8) {
      int smax, stages;
      double smean, cost;
      const int nblocks = spreads(G * r.RD, &smax, &smean);
      if (evaluate(G, T, Cc, smax, smean, nblocks, 2, &stages, &cost)) {
        bc = {G, T, Cc, std::min(stages, tune.stages)};
        found = true;
      }
    }
  } else {
    for (auto& gt : cand) {
      const int G = gt[0], T = gt[1];
      int smax;
      double smean;
      const int nblocks = spreads(G * r.RD, &smax, &smean);
      for (int Cc : {32, 16, 8, 4}) {
        int stages;
        double cost;
        if (!evaluate(G, T, Cc, smax, smean, nblocks, Cc >= 8 ? 3 : 2, &stages, &cost)) continue;
        if (cost < best) {
          best = cost;
          bc = {G, T, Cc, stages};
          found = true;
        }
      }
    }
  }
  r.tiled_ok = found ? 1 : 0;  // otherwise the delay spread of one trial group exceeds shared memory: direct kernel
  r.G = bc.G;
  r.T = bc.T;
  r.Cc = bc.Cc;
  r.stages = bc.stages;
  r.Dcta = r.G * r.RD;
  r.nblocks = (r.ndm + r.Dcta - 1) / r.Dcta;
  r.Cpad = (int)round_up(p.nchans, r.Cc);
  if (dd::is_hybrid(r.mode)) {
    r.nd = found ? delta_prefix / r.Cc : 0;  // whole chunks inside the delta-codable prefix
    if (r.nd == 0) r.mode = r.mode == dd::kModeWideHybrid ? dd::kModeWide : dd::kModeGeneralReuse;
  }
  if (r.flush > 0) r.flush = r.flush / r.Cc * r.Cc;
  r.Smax = max_block_span(p, r, r.Dcta);  // the true maximum over every (trial block, channel)
  if (r.T + r.Smax > 65535) r.tiled_ok = 0;
  while (r.stages > 2 && dd::tiled_smem_bytes(r) > (size_t)227 * 1024) --r.stages;
  r.H = round_up((r.nout + r.NL - 1) / r.NL, 16);
  r.ntau = (r.H + r.T - 1) / r.T;
  r.Wp = round_up(r.ntau * r.T + r.maxd + 8, 8);  // rows are 128-byte multiples; +8: staged rows end on a line
  r.plane_bytes = round_up((int64_t)p.nbeams * r.Cpad * r.Wp * dd::kSuperwordBytes, 256);
  r.ws_bytes = r.plane_bytes * r.planes;
  r.smem_bytes = dd::tiled_smem_bytes(r);
  if (r.smem_bytes > (size_t)227 * 1024) r.tiled_ok = 0;
  if (!r.tiled_ok) r.ws_bytes = 0;
}

// Device tables of the tiled kernel: per trial block and channel the start of the staged row (the first
// delay of the block rounded down to a 128-byte line: bulk copies whose source and destination are both
// line-aligned fill shared memory a line per wavefront, misaligned ones 16 bytes at a time -- ncu,
// profiles/) and its length beyond T (rounded up likewise); per trial group the offsets into the row in
// the form the range's mode wants (dd_internal.h).  Trials past the end of the range repeat the last one.
void build_tables(const dd_plan& p, dd::RangePlan& r) {
  const size_t nbc = (size_t)r.nblocks * r.Cpad;
  std::vector<int32_t>& dmin = r.h_dmin;
  std::vector<int32_t>& span = r.h_span;
  dmin.assign(nbc, 0);
  span.assign(nbc, 0);
  const bool delta = r.mode == dd::kModeDelta;
  // words of one chunk's table slice in the delta form (one 4-word entry per quad and trial group) and in the general
  // forms (one 32-bit byte offset per channel and trial); a trial block holds its chunks' slices one after the other,
  // a hybrid range its nd delta slices first
  const size_t nchunks = (size_t)r.Cpad / r.Cc;
  const size_t wd = (size_t)(r.Cc / 4) * r.G * 4, wg = (size_t)r.Cc * r.G * r.RD;
  const size_t nd = delta ? nchunks : (size_t)r.nd;
  const size_t words_per_block = nd * wd + (nchunks - nd) * wg;
  std::vector<uint32_t>& meta = r.h_meta;
  meta.assign((size_t)r.nblocks * words_per_block, 0);
  // rows past nchans are the zero rows of the packed input: delay 0 for every trial
  auto delay = [&](int j, int c) { return c < p.nchans ? r.delays[(size_t)std::min(r.ndm - 1, j) * p.nchans + c] : 0; };
  // Which channel sits in which row of a stage.  The sum runs over all channels, so their order is free, per trial
  // block.  In the delta form a trial step of a channel QUAD costs shared-memory slots and issue slots as soon as one
  // of its four channels changes its delay, so the channels of a chunk are dealt to quads by the fractional part of
  // their (unrounded) delay at the middle trial of the block: channels that cross a rounding boundary at the same
  // trials share a quad.  Config 3: quad steps with a change 42 / 54 / 57 % -> 27 / 28 / 33 % (ranges 0 / 1 / 2).
  std::vector<int32_t>& chan = r.h_chan;
  chan.resize(nbc);
  for (int b = 0; b < r.nblocks; ++b)
    for (int c = 0; c < r.Cpad; ++c) chan[(size_t)b * r.Cpad + c] = c;
  if (nd > 0) {
    const double ts = p.tsamp * (double)r.decim, inv_top = 1.0 / (p.f_top * p.f_top);
    std::vector<double> phase(r.Cc);
    std::vector<int32_t> order(r.Cc);
    for (int b = 0; b < r.nblocks; ++b) {
      const int jm = std::min(r.ndm - 1, b * r.Dcta + r.Dcta / 2);
      const double dm = r.dm_lo + (double)jm * r.dm_step;
      for (size_t k = 0; k < nd; ++k) {
        for (int i = 0; i < r.Cc; ++i) {
          const int c = (int)k * r.Cc + i;
          order[i] = c;
          if (c < p.nchans) {
            const double f = p.f_top + (double)c * p.cw;
            const double x = kDispersion * dm * (1.0 / (f * f) - inv_top) / ts + 0.5;
            phase[i] = x - floor(x);
          } else {
            phase[i] = -1.0;  // zero rows never change: last
          }
        }
        std::stable_sort(order.begin(), order.end(), [&](int32_t u, int32_t v) {
          return phase[u - (int)k * r.Cc] > phase[v - (int)k * r.Cc];
        });
        for (int i = 0; i < r.Cc; ++i) chan[(size_t)b * r.Cpad + k * r.Cc + i] = order[i];
      }
    }
  }
  for (int b = 0; b < r.nblocks; ++b) {
    const int j0 = b * r.Dcta;
    for (int s = 0; s < r.Cpad; ++s) {  // s = row of the staged chunk sequence, c = the channel that sits there
      const int c = chan[(size_t)b * r.Cpad + s];
      const int32_t d0 = delay(j0, c) & ~7;  // delays are non-decreasing in j
      dmin[(size_t)b * r.Cpad + s] = d0;
      span[(size_t)b * r.Cpad + s] = (int32_t)round_up(delay(j0 + r.Dcta - 1, c) - d0, 8);
      if (span[(size_t)b * r.Cpad + s] > r.Smax) r.tiled_ok = 0;  // cannot happen (Smax is this maximum); never overrun a row
      for (int g = 0; g < r.G; ++g) {
        const int jg = j0 + g * r.RD;
        const size_t k = (size_t)s / r.Cc, si = (size_t)s % r.Cc;
        if (k < nd) {
          uint32_t* e = &meta[(size_t)b * words_per_block + k * wd + ((size_t)g * (r.Cc / 4) + si / 4) * 4];  // [group][quad]
          const int q = s % 4;
          const uint32_t off = ((uint32_t)si * (uint32_t)(r.T + r.Smax) + (uint32_t)(delay(jg, c) - d0)) * 16u;
          e[1 + q / 2] |= off << (16 * (q % 2));  // byte offset inside the stage, < 64 KB (choose_tile)
          for (int j = 1; j < r.RD; ++j)
            if (delay(jg + j, c) != delay(jg + j - 1, c)) {
              e[0] |= 1u << dd::delta_bit(j, q);
              e[3] |= 1u << j;  // some channel of the quad changes at this trial step
            }
        } else {
          uint32_t* e = &meta[(size_t)b * words_per_block + nd * wd + (k - nd) * wg + (si * r.G + g) * r.RD];
          for (int j = 0; j < r.RD; ++j)  // byte offsets inside the stage, row of the channel included
            e[j] = ((uint32_t)si * (uint32_t)(r.T + r.Smax) + (uint32_t)(delay(jg + j, c) - d0)) * 16u;
        }
      }
    }
  }
}

int upload_tables(dd::RangePlan& r) {
  DD_CUDA(cudaMalloc(&r.d_meta, r.h_meta.size() * sizeof(uint32_t)));
  DD_CUDA(cudaMalloc(&r.d_dmin, r.h_dmin.size() * sizeof(int32_t)));
  DD_CUDA(cudaMalloc(&r.d_span, r.h_span.size() * sizeof(int32_t)));
  DD_CUDA(cudaMemcpy(r.d_meta, r.h_meta.data(), r.h_meta.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
  DD_CUDA(cudaMemcpy(r.d_dmin, r.h_dmin.data(), r.h_dmin.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
  DD_CUDA(cudaMemcpy(r.d_span, r.h_span.data(), r.h_span.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
  DD_CUDA(cudaMalloc(&r.d_chan, r.h_chan.size() * sizeof(int32_t)));
  DD_CUDA(cudaMemcpy(r.d_chan, r.h_chan.data(), r.h_chan.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
  return DD_OK;
}

// ---- two-channel sub-bands (kModeDeltaPair, variant DD_KERNEL_SUBBAND) ---------------------------------------------
// Delay of internal channel row c for the pair tables: rows past nchans are zero rows, so any delay is correct for
// them; the pad partner of the last real channel copies it (delta = 0), all-pad pairs stay at 0.
inline int32_t pair_delay(const dd_plan& p, const dd::RangePlan& r, int j, int c) {
  j = std::min(r.ndm - 1, j);
  if (c < p.nchans) return r.delays[(size_t)j * p.nchans + c];
  if ((c & 1) && c - 1 < p.nchans) return r.delays[(size_t)j * p.nchans + c - 1];
  return 0;
}

// Decide whether range r can run on pair rows and build its tables (host).  Conditions: delta-coded 16-bit-lane
// range, an even number of channel rows per stage quad, every pair's delay difference takes at most two
// neighbouring values over ALL trials of the range, and the doubled rows fit the 16-bit byte offsets and shared memory.
void build_pair_tables(const dd_plan& p, dd::RangePlan& r) {
  r.pair_ok = 0;
  if (!r.tiled_ok || r.mode != dd::kModeDelta || r.NL != 8 || r.Cc % 8 != 0 || r.planes != 1) return;
  const int nvc = r.Cpad / 2;
  r.Cc2 = r.Cc / 2;
  r.h_delta.assign(nvc, 0);
  for (int v = 0; v < nvc; ++v) {
    int32_t lo = INT32_MAX, hi = INT32_MIN;
    for (int j = 0; j < r.ndm; ++j) {
      const int32_t d = pair_delay(p, r, j, 2 * v + 1) - pair_delay(p, r, j, 2 * v);
      lo = std::min(lo, d);
      hi = std::max(hi, d);
    }
    if (hi - lo > 1) return;  // a third row would be needed: not this range
    r.h_delta[v] = lo;
  }
  const size_t nbc = (size_t)r.nblocks * r.Cpad;
  // Which pair sits in which double row of a stage: as for the delta table (build_tables), the pairs of a chunk are
  // dealt to quads by the delay phase of their first channel at the block's middle trial, per trial block.  h_chan2
  // holds the source ROW (2v + p) of every staged row.
  std::vector<int32_t> pairsrc(nbc / 2);  // [block][slot pair] -> pair
  r.h_chan2.assign(nbc, 0);
  {
    const double ts = p.tsamp * (double)r.decim, inv_top = 1.0 / (p.f_top * p.f_top);
    std::vector<double> phase(r.Cc2);
    std::vector<int32_t> order(r.Cc2);
    for (int b = 0; b < r.nblocks; ++b) {
      const int jm = std::min(r.ndm - 1, b * r.Dcta + r.Dcta / 2);
      const double dm = r.dm_lo + (double)jm * r.dm_step;
      for (int k = 0; k < nvc / r.Cc2; ++k) {
        for (int i = 0; i < r.Cc2; ++i) {
          const int v = k * r.Cc2 + i, c = 2 * v;
          order[i] = v;
          if (c < p.nchans) {
            const double f = p.f_top + (double)c * p.cw;
            const double x = kDispersion * dm * (1.0 / (f * f) - inv_top) / ts + 0.5;
            phase[i] = x - floor(x);
          } else {
            phase[i] = -1.0;
          }
        }
        std::stable_sort(order.begin(), order.end(), [&](int32_t u, int32_t v) { return phase[u - k * r.Cc2] > phase[v - k * r.Cc2]; });
        for (int i = 0; i < r.Cc2; ++i) {
          const size_t u = (size_t)k * r.Cc2 + i;
          pairsrc[(size_t)b * nvc + u] = order[i];
          r.h_chan2[(size_t)b * r.Cpad + 2 * u] = 2 * order[i];
          r.h_chan2[(size_t)b * r.Cpad + 2 * u + 1] = 2 * order[i] + 1;
        }
      }
    }
  }
  r.h_dmin2.assign(nbc, 0);
  r.h_span2.assign(nbc, 0);
  r.Smax2 = 0;
  for (int b = 0; b < r.nblocks; ++b)
    for (int u = 0; u < nvc; ++u) {  // u = slot pair, v = the pair staged there
      const int v = pairsrc[(size_t)b * nvc + u];
      const int j0 = b * r.Dcta;
      const int32_t d0 = pair_delay(p, r, j0, 2 * v) & ~7;
      const int32_t sp = (int32_t)round_up(pair_delay(p, r, j0 + r.Dcta - 1, 2 * v) - d0, 8);
      for (int q = 0; q < 2; ++q) {  // both pre-summed rows of the pair are staged over the span of channel 2v
        r.h_dmin2[(size_t)b * r.Cpad + 2 * u + q] = d0;
        r.h_span2[(size_t)b * r.Cpad + 2 * u + q] = sp;
      }
      r.Smax2 = std::max(r.Smax2, (int)sp);
    }
  const size_t rowbytes = (size_t)(r.T + r.Smax2) * 16;
  if ((size_t)r.Cc * rowbytes > 65536) return;  // 16-bit byte offsets inside a stage
  const size_t stage = (r.Cc * rowbytes + dd::tiled_meta_bytes(dd::kModeDeltaPair, r.NL, r.Cc, r.G) + 127) / 128 * 128;
  r.stages2 = (int)std::min<size_t>(6, ((size_t)227 * 1024 - 128 - 512) / stage);
  if (r.stages2 < 2) return;
  // table: five 16-byte entries per quad of pairs and trial group (dd_tiled.cu stage_pairs)
  r.h_meta2.assign((size_t)r.nblocks * (nvc / 4) * r.G * 20, 0);
  for (int b = 0; b < r.nblocks; ++b)
    for (int u = 0; u < nvc; ++u) {
      const int v = pairsrc[(size_t)b * nvc + u];
      const int32_t d0 = r.h_dmin2[(size_t)b * r.Cpad + 2 * u];
      const int q = u % 4;
      for (int g = 0; g < r.G; ++g) {
        const int jg = b * r.Dcta + g * r.RD;
        uint32_t* e = &r.h_meta2[(((size_t)b * (nvc / 4) + u / 4) * r.G + g) * 20];
        auto D = [&](int j) { return pair_delay(p, r, j, 2 * v); };
        auto P = [&](int j) { return pair_delay(p, r, j, 2 * v + 1) - D(j) - r.h_delta[v]; };
        for (int j = 0; j < r.RD; ++j) {
          const uint32_t off = ((uint32_t)((2 * u + P(jg + j)) % r.Cc) * (uint32_t)(r.T + r.Smax2) + (uint32_t)(D(jg + j) - d0)) * 16u;
          e[4 + 4 * q + j / 2] |= off << (16 * (j % 2));
          if (j > 0 && (D(jg + j) != D(jg + j - 1) || P(jg + j) != P(jg + j - 1))) {
            e[0] |= 1u << dd::delta_bit(j, q);
            e[1] |= 1u << j;  // some pair of the quad changes at this trial step
          }
        }
      }
    }
  r.ws2_bytes = round_up((int64_t)p.nbeams * r.Cpad * r.Wp * dd::kSuperwordBytes, 256);
  // executed adds per beam: one per (trial, sample, pair) + two pre-sums per packed pair-row element
  r.adds_pair = (int64_t)r.ndm * r.nout * (p.nchans + 1) / 2 + (int64_t)2 * ((p.nchans + 1) / 2) * r.ns;
  r.pair_ok = 1;
}

int upload_pair_tables(dd::RangePlan& r) {
  if (r.d_meta2) return DD_OK;
  DD_CUDA(cudaMalloc(&r.d_meta2, r.h_meta2.size() * sizeof(uint32_t)));
  DD_CUDA(cudaMalloc(&r.d_dmin2, r.h_dmin2.size() * sizeof(int32_t)));
  DD_CUDA(cudaMalloc(&r.d_span2, r.h_span2.size() * sizeof(int32_t)));
  DD_CUDA(cudaMalloc(&r.d_delta, r.h_delta.size() * sizeof(int32_t)));
  DD_CUDA(cudaMemcpy(r.d_meta2, r.h_meta2.data(), r.h_meta2.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
  DD_CUDA(cudaMemcpy(r.d_dmin2, r.h_dmin2.data(), r.h_dmin2.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
  DD_CUDA(cudaMemcpy(r.d_span2, r.h_span2.data(), r.h_span2.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
  DD_CUDA(cudaMemcpy(r.d_delta, r.h_delta.data(), r.h_delta.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
  DD_CUDA(cudaMalloc(&r.d_chan2, r.h_chan2.size() * sizeof(int32_t)));
  DD_CUDA(cudaMemcpy(r.d_chan2, r.h_chan2.data(), r.h_chan2.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
  return DD_OK;
}

int ensure_direct_tables(dd_plan* p, bool only_untiled) {
  for (auto& r : p->ranges) {
    if (r.d_delays || (only_untiled && r.tiled_ok)) continue;
    DD_CUDA(cudaMalloc(&r.d_delays, r.delays.size() * sizeof(int32_t)));
    DD_CUDA(cudaMemcpy(r.d_delays, r.delays.data(), r.delays.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
  }
  return DD_OK;
}

int ensure_workspace(dd_plan* p) {
  const int64_t need = p->ws_bytes + p->ws_pair_bytes;
  if (need == 0 || (p->ws && p->ws_have >= need)) return DD_OK;
  if (p->ws && !p->ws_owned) return DD_ERR_NOMEM;  // a caller-owned workspace that is too small: set a larger one
  if (p->ws) cudaFree(p->ws);
  p->ws = nullptr;
  p->ws_have = 0;
  cudaError_t e = cudaMalloc(&p->ws, (size_t)need);
  if (e != cudaSuccess) {
    cuda_fail(e, "cudaMalloc(workspace)");
    p->ws = nullptr;
    return DD_ERR_NOMEM;
  }
  p->ws_owned = true;
  p->ws_have = need;
  return DD_OK;
}

inline bool aligned16(const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15u) == 0; }

}  // namespace

extern "C" {

int dd_version(void) { return DD_VERSION; }

const char* dd_strerror(int code) {
  switch (code) {
    case DD_OK: return "ok";
    case DD_ERR_INVALID: return "invalid argument";
    case DD_ERR_TOO_SHORT: return "input too short for the largest delay of a range";
    case DD_ERR_OVERFLOW: return "channel sum does not fit 32 bits";
    case DD_ERR_ALIGN: return "buffer not 16-byte aligned";
    case DD_ERR_CUDA: return "CUDA error (see dd_last_cuda_error)";
    case DD_ERR_NOMEM: return "out of memory or workspace too small";
    case DD_ERR_DEVICE: return "current CUDA device is not the plan's device";
    default: return "unknown dd_status";
  }
}

const char* dd_last_cuda_error(void) { return g_last_cuda_error.c_str(); }

// Host half of a plan: validation, delay tables, tile shapes, the tables of the tiled kernel.  No CUDA call.
static int plan_create_host(const dd_config_t* cfg, dd_plan_t** plan_out, int64_t tail_new = 0,
                            const dd_tuning_t* tune = nullptr) {
  if (!cfg || !plan_out) return DD_ERR_INVALID;
  *plan_out = nullptr;
  if (cfg->nchans < 1 || !(cfg->chan_width_mhz != 0.0) || !(cfg->tsamp_s > 0.0) || cfg->nsamps < 1 ||
      (cfg->in_layout != DD_LAYOUT_CHANNEL_MAJOR && cfg->in_layout != DD_LAYOUT_SPECTRUM_MAJOR) ||
      cfg->nbeams < 1 || !(cfg->in_bits == 8 || cfg->in_bits == 16) || cfg->nranges < 1 || !cfg->ranges ||
      !(cfg->f_top_mhz > 0.0) || cfg->nchans > 65535 || cfg->nbeams > 65535)
    return DD_ERR_INVALID;
  const double f_last = cfg->f_top_mhz + (double)(cfg->nchans - 1) * cfg->chan_width_mhz;
  if (!(f_last > 0.0)) return DD_ERR_INVALID;
  for (int r = 0; r < cfg->nranges; ++r) {
    const dd_range_t& q = cfg->ranges[r];
    if (!(q.decim == 1 || q.decim == 2 || q.decim == 4 || q.decim == 8) || q.ndm < 1 || q.ndm > 65535 ||
        !(q.dm_lo >= 0.0) || !(q.dm_step >= 0.0))
      return DD_ERR_INVALID;
    const double bound = (double)cfg->nchans * (double)((1 << cfg->in_bits) - 1) * (double)q.decim;
    if (bound >= 4294967296.0) return DD_ERR_OVERFLOW;
  }
  dd_plan* p = new (std::nothrow) dd_plan();
  if (!p) return DD_ERR_NOMEM;
  int rc = DD_OK;
  try {
    // internally channel 0 is always the highest frequency (the reference of Eq. 1.1); an ascending band is
    // the same band read backwards, and the pack / direct kernels reverse the channel index while loading
    p->ascending = cfg->chan_width_mhz > 0.0;
    p->f_top = p->ascending ? f_last : cfg->f_top_mhz;
    p->cw = -fabs(cfg->chan_width_mhz);
    p->layout = cfg->in_layout;
    p->tsamp = cfg->tsamp_s;
    p->nchans = cfg->nchans;
    p->nbeams = cfg->nbeams;
    p->in_bits = cfg->in_bits;
    p->nsamps = cfg->nsamps;
    p->tail_new = tail_new;
    p->ranges.resize(cfg->nranges);
    int64_t offset = 0;
    for (int i = 0; i < cfg->nranges && rc == DD_OK; ++i) {
      dd::RangePlan& r = p->ranges[i];
      r.dm_lo = cfg->ranges[i].dm_lo;
      r.dm_step = cfg->ranges[i].dm_step;
      r.ndm = cfg->ranges[i].ndm;
      r.decim = cfg->ranges[i].decim;
      if (!build_delays(*p, r)) { rc = DD_ERR_TOO_SHORT; break; }
      r.maxd = r.delays[(size_t)(r.ndm - 1) * p->nchans + (p->nchans - 1)];
      // a tail plan skips the input this range does not need for its last tail_new/decim outputs (16-sample
      // granularity keeps the vector loads of the pack kernels aligned)
      if (tail_new > 0) r.in_off = std::max<int64_t>(0, (p->nsamps - tail_new - r.maxd * r.decim) / 16 * 16);
      r.ns = (p->nsamps - r.in_off) / r.decim;
      r.nout = r.ns - r.maxd;
      if (r.nout < 1) { rc = DD_ERR_TOO_SHORT; break; }
      // a tail plan promises the last tail_new/decim outputs of every range: the window must hold their delays
      if (tail_new > 0 && r.nout < tail_new / r.decim) { rc = DD_ERR_TOO_SHORT; break; }
      r.pitch = round_up(r.nout, 32);
      r.offset = offset;
      r.row0 = p->rows_per_beam;
      p->rows_per_beam += r.ndm;
      offset += (int64_t)r.ndm * r.pitch;
      p->dm_samples += (int64_t)p->nbeams * r.ndm * r.nout;
      choose_tile(*p, r, tune ? *tune : kAutoTuning);
      // every range packs into the same scratch: a range is packed right before its dedispersion kernel (dd_execute), so
      // the workspace is the largest packed copy, not their sum (config 3: 2.2 GB instead of 4.0 GB)
      r.ws_offset = 0;
      p->ws_bytes = std::max<int64_t>(p->ws_bytes, round_up(r.ws_bytes, 256));
    }
    if (rc == DD_OK) {
      p->beam_stride = offset;
      p->out_elems = offset * p->nbeams;
      p->adds = p->dm_samples * p->nchans;
    }
  } catch (const std::bad_alloc&) {
    rc = DD_ERR_NOMEM;
  }
  if (rc != DD_OK) {
    delete p;
    return rc;
  }
  try {
    for (auto& r : p->ranges)
      if (r.tiled_ok) build_tables(*p, r);
  } catch (const std::bad_alloc&) {
    delete p;
    return DD_ERR_NOMEM;
  }
  p->device = -1;  // host only until dd_plan_create puts it on a device
  *plan_out = p;
  return DD_OK;
}

int dd_plan_create_host(const dd_config_t* cfg, dd_plan_t** plan_out) { return plan_create_host(cfg, plan_out); }

static int plan_create_device(const dd_config_t* cfg, dd_plan_t** plan_out, int64_t tail_new,
                              const dd_tuning_t* tune = nullptr);

int dd_plan_create(const dd_config_t* cfg, dd_plan_t** plan_out) { return plan_create_device(cfg, plan_out, 0); }

int dd_plan_create_tuned(const dd_config_t* cfg, const dd_tuning_t* tuning, int32_t host_only, dd_plan_t** plan_out) {
  if (tuning && (tuning->mode < -1 || (tuning->mode > 2 && tuning->mode != 6) || tuning->byte_lanes < -1 || tuning->byte_lanes > 1))
    return DD_ERR_INVALID;
  return host_only ? plan_create_host(cfg, plan_out, 0, tuning) : plan_create_device(cfg, plan_out, 0, tuning);
}

int dd_plan_create_tail(const dd_config_t* cfg, int64_t new_samps, dd_plan_t** plan_out) {
  if (new_samps < 1 || !cfg || new_samps > cfg->nsamps) return DD_ERR_INVALID;
  return plan_create_device(cfg, plan_out, new_samps);
}

static int plan_create_device(const dd_config_t* cfg, dd_plan_t** plan_out, int64_t tail_new, const dd_tuning_t* tune) {
  if (!plan_out) return DD_ERR_INVALID;
  dd_plan* p = nullptr;
  int rc = plan_create_host(cfg, &p, tail_new, tune);
  if (rc != DD_OK) return rc;
  *plan_out = nullptr;
  cudaError_t e = cudaGetDevice(&p->device);
  if (e != cudaSuccess) {
    delete p;
    return cuda_fail(e, "cudaGetDevice");
  }
  e = dd::configure_kernels(p);
  if (e != cudaSuccess) {
    delete p;
    return cuda_fail(e, "cudaFuncSetAttribute");
  }
  for (auto& r : p->ranges) {
    rc = r.tiled_ok ? upload_tables(r) : DD_OK;
    if (rc != DD_OK) break;
  }
  if (rc == DD_OK) rc = ensure_direct_tables(p, /*only_untiled=*/true);
  if (rc == DD_OK) rc = ensure_workspace(p);
  if (rc == DD_OK) {
    e = cudaDeviceSynchronize();
    if (e != cudaSuccess) rc = cuda_fail(e, "cudaDeviceSynchronize");
  }
  if (rc != DD_OK) {
    dd_plan_destroy(p);
    return rc;
  }
  *plan_out = p;
  return DD_OK;
}

int dd_plan_destroy(dd_plan_t* p) {
  if (!p) return DD_OK;
  for (auto& r : p->ranges) {
    if (r.d_meta) cudaFree(r.d_meta);
    if (r.d_dmin) cudaFree(r.d_dmin);
    if (r.d_span) cudaFree(r.d_span);
    if (r.d_chan) cudaFree(r.d_chan);
    if (r.d_delays) cudaFree(r.d_delays);
    if (r.d_meta2) cudaFree(r.d_meta2);
    if (r.d_dmin2) cudaFree(r.d_dmin2);
    if (r.d_span2) cudaFree(r.d_span2);
    if (r.d_delta) cudaFree(r.d_delta);
    if (r.d_chan2) cudaFree(r.d_chan2);
  }
  for (cudaEvent_t e : p->prof_events) cudaEventDestroy(e);
  if (p->ws && p->ws_owned) cudaFree(p->ws);
  for (int s = 0; s < 2; ++s) {
    if (p->h_in_dev[s]) cudaFree(p->h_in_dev[s]);
    if (p->h_out_dev[s]) cudaFree(p->h_out_dev[s]);
    if (p->ev_in_ready[s]) cudaEventDestroy(p->ev_in_ready[s]);
    if (p->ev_in_free[s]) cudaEventDestroy(p->ev_in_free[s]);
    if (p->ev_out_free[s]) cudaEventDestroy(p->ev_out_free[s]);
  }
  for (cudaEvent_t e : p->host_events) cudaEventDestroy(e);
  if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
  if (p->h2d_stream) cudaStreamDestroy(p->h2d_stream);
  delete p;
  return DD_OK;
}

int dd_execute(const dd_plan_t* plan, const void* in_dev, float* out_dev, void* cuda_stream) {
  if (!plan || !in_dev || !out_dev || plan->device < 0) return DD_ERR_INVALID;
  if (!aligned16(in_dev) || !aligned16(out_dev)) return DD_ERR_ALIGN;
  {  // the tables and the workspace live on the device the plan was created on
    int cur = -1;
    DD_CUDA(cudaGetDevice(&cur));
    if (cur != plan->device) return DD_ERR_DEVICE;
  }
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  const bool all_direct = plan->variant == DD_KERNEL_DIRECT;
  // optional per-launch events (measurement hook)
  const int max_launch = 3 * (int)plan->ranges.size();
  const int slot = plan->prof_slots > 0 ? (int)(plan->prof_calls++ % plan->prof_slots) : -1;
  int nl = 0;
  auto ev_before = [&](int kind, int range) -> cudaError_t {
    if (slot < 0) return cudaSuccess;
    plan->prof_kind[(size_t)slot * max_launch + nl] = kind;
    plan->prof_range[(size_t)slot * max_launch + nl] = range;
    return cudaEventRecord(plan->prof_events[((size_t)slot * max_launch + nl) * 2], stream);
  };
  auto ev_after = [&]() -> cudaError_t {
    if (slot < 0) return cudaSuccess;
    cudaError_t e = cudaEventRecord(plan->prof_events[((size_t)slot * max_launch + nl) * 2 + 1], stream);
    plan->prof_count[slot] = ++nl;
    return e;
  };
  if (plan->row_stats)  // row statistics for the single-pulse search: the kernels' epilogues add into zeroed sums
    DD_CUDA(cudaMemsetAsync(plan->row_stats, 0, (size_t)plan->nbeams * plan->rows_per_beam * 2 * sizeof(unsigned long long), stream));
  // Range by range: a2 (pack), then a3+a4.  The packed copies of all ranges share one scratch; the pack kernel of the
  // next range (0.4 - 1 ms) starts in the tail of the dedispersion kernel before it, where SMs idle anyway.
  for (const auto& r : plan->ranges) {
    const int ri = (int)(&r - plan->ranges.data());
    if (all_direct || !r.tiled_ok) {
      if (!r.d_delays) return DD_ERR_INVALID;  // uploaded by dd_plan_create / dd_plan_set_kernel
      DD_CUDA(ev_before(2, ri));
      DD_CUDA(dd::launch_direct(plan, r, in_dev, out_dev, stream));
      DD_CUDA(ev_after());
      continue;
    }
    if (!plan->ws || plan->ws_have < plan->ws_bytes + plan->ws_pair_bytes) return DD_ERR_NOMEM;
    DD_CUDA(ev_before(0, ri));
    DD_CUDA(dd::launch_pack(plan, r, in_dev, stream));
    DD_CUDA(ev_after());
    if (dd::use_pairs(plan, r)) {  // DD_KERNEL_SUBBAND: pre-sum the packed rows into the pair rows
      DD_CUDA(ev_before(3, ri));
      DD_CUDA(dd::launch_pairs(plan, r, stream));
      DD_CUDA(ev_after());
    }
    DD_CUDA(ev_before(1, ri));
    DD_CUDA(dd::launch_tiled(plan, r, out_dev, stream));
    DD_CUDA(ev_after());
  }
  return DD_OK;
}

// Everything a host call enqueues, for staging slot `slot`.  Any failure is returned to the caller below, which drains
// all streams before handing the error on (the caller's buffers must not be touched by copies still in flight).
//   h2d_stream : in_host -> h_in_dev[slot], once the kernels of the call that used this slot before have read it
//   stream     : pack kernels (wait for the upload), then the dedispersion kernels a few trial blocks at a time (the first
//                waits until the slot's previous output has been copied back)
//   copy_stream: each finished piece -> out_host while the next blocks are computed
static int execute_host_enqueue(dd_plan_t* plan, const void* in_host, float* out_host, cudaStream_t stream, int slot) {
  const size_t in_bytes = (size_t)plan->nbeams * plan->nchans * plan->nsamps * (plan->in_bits / 8);
  const bool all_direct = plan->variant == DD_KERNEL_DIRECT;
  void* const in_dev = plan->h_in_dev[slot];
  float* const out_dev = plan->h_out_dev[slot];
  // The DM-time plane is 3.6x the input: its copy back is the larger half of the transfer time.  Every range is
  // dedispersed in a few launches of consecutive trial blocks; as soon as one is done (event), its rows -- one
  // contiguous piece per beam -- go back on the copy stream while the next blocks are computed.
  // per range: pieces of >= 1 trial block.  Config 3, ms per step synchronous / queued back to back: 1 piece 152.5 / 116.0,
  // 2: 140.4 / 116.4, 4: 137.4 / 117.4, 8: 138.8 / 120.0, 16: 143.0 / 124.2 (every launch ends in a partial wave)
  const int kPieces = plan->host_pieces;
  size_t nev = 0;
  auto next_event = [&](cudaEvent_t* ev) -> cudaError_t {
    if (nev == plan->host_events.size()) {
      cudaEvent_t e;
      cudaError_t rc = cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
      if (rc != cudaSuccess) return rc;
      plan->host_events.push_back(e);
    }
    *ev = plan->host_events[nev++];
    return cudaSuccess;
  };
  auto copy_rows = [&](const dd::RangePlan& r, int j0, int j1) -> cudaError_t {  // trials j0 .. j1-1, all beams
    cudaEvent_t ev;
    cudaError_t rc = next_event(&ev);
    if (rc != cudaSuccess) return rc;
    if ((rc = cudaEventRecord(ev, stream)) != cudaSuccess) return rc;
    if ((rc = cudaStreamWaitEvent(plan->copy_stream, ev, 0)) != cudaSuccess) return rc;
    for (int b = 0; b < plan->nbeams; ++b) {
      const size_t off = (size_t)b * plan->beam_stride + r.offset + (size_t)j0 * r.pitch;
      rc = cudaMemcpyAsync(out_host + off, out_dev + off, (size_t)(j1 - j0) * r.pitch * sizeof(float),
                           cudaMemcpyDeviceToHost, plan->copy_stream);
      if (rc != cudaSuccess) return rc;
    }
    return cudaSuccess;
  };
  DD_CUDA(cudaStreamWaitEvent(plan->h2d_stream, plan->ev_in_free[slot], 0));  // (never recorded yet: no wait)
  DD_CUDA(cudaMemcpyAsync(in_dev, in_host, in_bytes, cudaMemcpyHostToDevice, plan->h2d_stream));
  DD_CUDA(cudaEventRecord(plan->ev_in_ready[slot], plan->h2d_stream));
  DD_CUDA(cudaStreamWaitEvent(stream, plan->ev_in_ready[slot], 0));
  DD_CUDA(cudaStreamWaitEvent(stream, plan->ev_out_free[slot], 0));
  for (const auto& r : plan->ranges) {  // range by range, as dd_execute: the packed copies share one scratch
    if (all_direct || !r.tiled_ok) {
      DD_CUDA(dd::launch_direct(plan, r, in_dev, out_dev, stream));
      DD_CUDA(copy_rows(r, 0, r.ndm));
      continue;
    }
    DD_CUDA(dd::launch_pack(plan, r, in_dev, stream));
    if (dd::use_pairs(plan, r)) DD_CUDA(dd::launch_pairs(plan, r, stream));
    const int per = std::max(1, (r.nblocks + kPieces - 1) / kPieces);
    for (int b0 = 0; b0 < r.nblocks; b0 += per) {
      const int nb = std::min(per, r.nblocks - b0);
      DD_CUDA(dd::launch_tiled(plan, r, out_dev, stream, b0, nb));
      DD_CUDA(copy_rows(r, b0 * r.Dcta, std::min(r.ndm, (b0 + nb) * r.Dcta)));
    }
  }
  DD_CUDA(cudaEventRecord(plan->ev_in_free[slot], stream));  // the last range's pack / direct kernel has read the input
  DD_CUDA(cudaEventRecord(plan->ev_out_free[slot], plan->copy_stream));
  return DD_OK;
}

static void host_drain(dd_plan_t* plan) {
  if (plan->h2d_stream) cudaStreamSynchronize(plan->h2d_stream);
  cudaStreamSynchronize(plan->host_stream);
  if (plan->copy_stream) cudaStreamSynchronize(plan->copy_stream);
}

int dd_execute_host_async(dd_plan_t* plan, const void* in_host, float* out_host, void* cuda_stream) {
  if (!plan || !in_host || !out_host || plan->device < 0) return DD_ERR_INVALID;
  {
    int cur = -1;
    DD_CUDA(cudaGetDevice(&cur));
    if (cur != plan->device) return DD_ERR_DEVICE;
  }
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  const size_t in_bytes = (size_t)plan->nbeams * plan->nchans * plan->nsamps * (plan->in_bits / 8);
  const size_t out_bytes = (size_t)plan->out_elems * sizeof(float);
  // everything that can be refused is checked before the first copy or launch is enqueued
  const bool all_direct = plan->variant == DD_KERNEL_DIRECT;
  for (const auto& r : plan->ranges) {
    if (all_direct || !r.tiled_ok) {
      if (!r.d_delays) return DD_ERR_INVALID;  // uploaded by dd_plan_create / dd_plan_set_kernel
    } else if (!plan->ws || plan->ws_have < plan->ws_bytes + plan->ws_pair_bytes) {
      return DD_ERR_NOMEM;
    }
  }
  const int slot = (int)(plan->host_calls % 2);
  if (!plan->h_in_dev[slot]) {
    if (cudaMalloc(&plan->h_in_dev[slot], in_bytes) != cudaSuccess) { plan->h_in_dev[slot] = nullptr; cudaGetLastError(); return DD_ERR_NOMEM; }
  }
  if (!plan->h_out_dev[slot]) {
    if (cudaMalloc(&plan->h_out_dev[slot], out_bytes) != cudaSuccess) { plan->h_out_dev[slot] = nullptr; cudaGetLastError(); return DD_ERR_NOMEM; }
  }
  if (!plan->copy_stream) DD_CUDA(cudaStreamCreateWithFlags(&plan->copy_stream, cudaStreamNonBlocking));
  if (!plan->h2d_stream) DD_CUDA(cudaStreamCreateWithFlags(&plan->h2d_stream, cudaStreamNonBlocking));
  for (int s = 0; s < 2; ++s) {
    if (!plan->ev_in_ready[s]) DD_CUDA(cudaEventCreateWithFlags(&plan->ev_in_ready[s], cudaEventDisableTiming));
    if (!plan->ev_in_free[s]) DD_CUDA(cudaEventCreateWithFlags(&plan->ev_in_free[s], cudaEventDisableTiming));
    if (!plan->ev_out_free[s]) DD_CUDA(cudaEventCreateWithFlags(&plan->ev_out_free[s], cudaEventDisableTiming));
  }
  if (plan->host_calls > 0 && plan->host_stream != stream) host_drain(plan);  // a change of stream breaks the stream order the slots rely on
  plan->host_stream = stream;
  const int rc = execute_host_enqueue(plan, in_host, out_host, stream, slot);
  ++plan->host_calls;
  if (rc != DD_OK) {  // drain what was enqueued: no copy may still read or write the caller's buffers after we return
    host_drain(plan);
    return rc;
  }
  return DD_OK;
}

int dd_plan_set_host_pieces(dd_plan_t* plan, int32_t pieces) {
  if (!plan || pieces < 1 || pieces > 64) return DD_ERR_INVALID;
  plan->host_pieces = pieces;
  return DD_OK;
}

int dd_host_wait(dd_plan_t* plan) {
  if (!plan || plan->device < 0) return DD_ERR_INVALID;
  if (plan->host_calls == 0) return DD_OK;
  {
    int cur = -1;
    DD_CUDA(cudaGetDevice(&cur));
    if (cur != plan->device) return DD_ERR_DEVICE;
  }
  DD_CUDA(cudaStreamSynchronize(plan->h2d_stream));
  DD_CUDA(cudaStreamSynchronize(plan->host_stream));
  DD_CUDA(cudaStreamSynchronize(plan->copy_stream));
  return DD_OK;
}

int dd_execute_host(dd_plan_t* plan, const void* in_host, float* out_host, void* cuda_stream) {
  const int rc = dd_execute_host_async(plan, in_host, out_host, cuda_stream);
  return rc != DD_OK ? rc : dd_host_wait(plan);
}

int dd_plan_out_elems(const dd_plan_t* p, int64_t* total_floats) {
  if (!p || !total_floats) return DD_ERR_INVALID;
  *total_floats = p->out_elems;
  return DD_OK;
}

int dd_plan_beam_stride(const dd_plan_t* p, int64_t* floats) {
  if (!p || !floats) return DD_ERR_INVALID;
  *floats = p->beam_stride;
  return DD_OK;
}

int dd_plan_range_info(const dd_plan_t* p, int32_t r, int64_t* ns_r, int64_t* maxd_r, int64_t* nout_r,
                       int64_t* pitch_floats, int64_t* offset_floats) {
  if (!p || r < 0 || r >= (int)p->ranges.size()) return DD_ERR_INVALID;
  const auto& q = p->ranges[r];
  if (ns_r) *ns_r = q.ns;
  if (maxd_r) *maxd_r = q.maxd;
  if (nout_r) *nout_r = q.nout;
  if (pitch_floats) *pitch_floats = q.pitch;
  if (offset_floats) *offset_floats = q.offset;
  return DD_OK;
}

int dd_plan_get_delays(const dd_plan_t* p, int32_t r, int32_t* host_buf) {
  if (!p || !host_buf || r < 0 || r >= (int)p->ranges.size()) return DD_ERR_INVALID;
  const auto& q = p->ranges[r];
  memcpy(host_buf, q.delays.data(), q.delays.size() * sizeof(int32_t));
  return DD_OK;
}

int dd_plan_work(const dd_plan_t* p, int64_t* dm_samples, int64_t* adds) {
  if (!p) return DD_ERR_INVALID;
  if (dm_samples) *dm_samples = p->dm_samples;
  if (adds) *adds = p->adds;
  return DD_OK;
}

int dd_plan_launches(const dd_plan_t* p, int32_t* n) {
  if (!p || !n) return DD_ERR_INVALID;
  int k = 0;
  for (const auto& r : p->ranges)
    k += (p->variant == DD_KERNEL_DIRECT || !r.tiled_ok) ? 1 : 1 + r.planes + (dd::use_pairs(p, r) ? 1 : 0);
  *n = k;
  return DD_OK;
}

int dd_plan_executed_adds(const dd_plan_t* p, int64_t* adds) {
  if (!p || !adds) return DD_ERR_INVALID;
  int64_t total = 0;
  for (const auto& r : p->ranges) {
    const int64_t brute = (int64_t)r.ndm * r.nout * p->nchans;
    if (dd::use_pairs(p, r)) {
      total += r.adds_pair;
    } else if ((p->variant == DD_KERNEL_SHARED || p->variant == DD_KERNEL_SUBBAND) && r.tiled_ok && r.mode == dd::kModeDelta) {
      // quad sums shared while no channel of the quad changes: a trial step costs 1 add per sample if unchanged,
      // else 3 (the new quad sum) + 1; the first trial of a group always 3 + 1.  Counted from the table.
      int64_t units = 0;  // adds per (time sample) summed over (block, quad, group, trial)
      const size_t nent = r.h_meta.size() / 4;
      for (size_t i = 0; i < nent; ++i) {
        const uint32_t any = r.h_meta[i * 4 + 3];
        units += 4;
        for (int j = 1; j < r.RD; ++j) units += ((any >> j) & 1u) ? 4 : 1;
      }
      // the table covers padded trials and channel rows; scale to the real (trial, channel) count
      const double scale = (double)brute / ((double)r.nblocks * r.Dcta * r.Cpad * (double)r.nout);
      total += (int64_t)((double)units * (double)r.nout * scale);
    } else {
      total += brute;
    }
  }
  *adds = total * p->nbeams;
  return DD_OK;
}

int dd_plan_pair_info(const dd_plan_t* p, int32_t r, int32_t* enabled, int32_t* pairs_per_stage, int32_t* row_superwords,
                      int32_t* npairs) {
  if (!p || r < 0 || r >= (int)p->ranges.size()) return DD_ERR_INVALID;
  const auto& q = p->ranges[r];
  if (enabled) *enabled = dd::use_pairs(p, q) ? 1 : 0;
  if (pairs_per_stage) *pairs_per_stage = q.Cc2;
  if (row_superwords) *row_superwords = q.T + q.Smax2;
  if (npairs) *npairs = q.Cpad / 2;
  return DD_OK;
}

int dd_plan_workspace_bytes(const dd_plan_t* p, int64_t* bytes) {
  if (!p || !bytes) return DD_ERR_INVALID;
  *bytes = p->ws_bytes + p->ws_pair_bytes;
  return DD_OK;
}

int dd_plan_set_workspace(dd_plan_t* p, void* dev, int64_t bytes) {
  if (!p) return DD_ERR_INVALID;
  if (dev) {
    if (!aligned16(dev)) return DD_ERR_ALIGN;
    if (bytes < p->ws_bytes + p->ws_pair_bytes) return DD_ERR_NOMEM;
    if (p->ws && p->ws_owned) cudaFree(p->ws);
    p->ws = dev;
    p->ws_owned = false;
    p->ws_have = bytes;
    return DD_OK;
  }
  if (p->ws && !p->ws_owned) p->ws = nullptr, p->ws_have = 0;
  return ensure_workspace(p);
}

int dd_plan_set_row_stats(dd_plan_t* p, uint64_t* stats_dev) {
  if (!p) return DD_ERR_INVALID;
  if (stats_dev && (p->in_bits != 8 || (reinterpret_cast<uintptr_t>(stats_dev) & 7u))) return DD_ERR_INVALID;
  p->row_stats = reinterpret_cast<unsigned long long*>(stats_dev);
  return DD_OK;
}

int dd_plan_set_kernel(dd_plan_t* p, int32_t variant) {
  if (!p) return DD_ERR_INVALID;
  if (variant != DD_KERNEL_AUTO && variant != DD_KERNEL_DIRECT && variant != DD_KERNEL_TILED &&
      variant != DD_KERNEL_SHARED && variant != DD_KERNEL_SUBBAND)
    return DD_ERR_INVALID;
  if (variant == DD_KERNEL_DIRECT && p->device >= 0) {
    int rc = ensure_direct_tables(p, false);
    if (rc != DD_OK) return rc;
  }
  if (variant == DD_KERNEL_SUBBAND && p->ws_pair_bytes == 0) {
    // first use: pair tables of every range that qualifies, their device copies, and room for the pair arrays
    try {
      int64_t pair_bytes = 0;
      for (auto& r : p->ranges) {
        build_pair_tables(*p, r);
        if (!r.pair_ok) continue;
        r.ws2_offset = p->ws_bytes;  // behind the packed copy; shared by the ranges like the packed copy itself
        pair_bytes = std::max(pair_bytes, r.ws2_bytes);
      }
      p->ws_pair_bytes = pair_bytes;
    } catch (const std::bad_alloc&) {
      return DD_ERR_NOMEM;
    }
    if (p->device >= 0) {
      for (auto& r : p->ranges)
        if (r.pair_ok) {
          int rc = upload_pair_tables(r);
          if (rc != DD_OK) return rc;
        }
      if (p->ws_owned || !p->ws) {
        int rc = ensure_workspace(p);
        if (rc != DD_OK) return rc;
      }
    }
  }
  p->variant = variant;
  return DD_OK;
}

int dd_plan_set_profiling(dd_plan_t* p, int32_t max_executes) {
  if (!p || max_executes < 0 || max_executes > 4096) return DD_ERR_INVALID;
  for (cudaEvent_t e : p->prof_events) cudaEventDestroy(e);
  p->prof_events.clear();
  p->prof_slots = 0;
  p->prof_calls = 0;
  const size_t max_launch = 3 * p->ranges.size();
  try {
    p->prof_kind.assign(max_launch * max_executes, 0);
    p->prof_range.assign(max_launch * max_executes, 0);
    p->prof_count.assign(max_executes, 0);
    p->prof_events.reserve(max_launch * max_executes * 2);
  } catch (const std::bad_alloc&) {
    return DD_ERR_NOMEM;
  }
  for (size_t i = 0; i < max_launch * max_executes * 2; ++i) {
    cudaEvent_t e;
    DD_CUDA(cudaEventCreate(&e));
    p->prof_events.push_back(e);
  }
  p->prof_slots = max_executes;
  return DD_OK;
}

int dd_plan_kernel_times(const dd_plan_t* p, int32_t slot, int32_t cap, float* ms, int32_t* kind, int32_t* range,
                         int32_t* n) {
  if (!p || !ms || !n || slot < 0 || slot >= p->prof_slots || cap < 0) return DD_ERR_INVALID;
  const size_t max_launch = 3 * p->ranges.size();
  const int cnt = std::min<int>(cap, p->prof_count[slot]);
  for (int i = 0; i < cnt; ++i) {
    const size_t k = (size_t)slot * max_launch + i;
    DD_CUDA(cudaEventElapsedTime(&ms[i], p->prof_events[2 * k], p->prof_events[2 * k + 1]));
    if (kind) kind[i] = p->prof_kind[k];
    if (range) range[i] = p->prof_range[k];
  }
  *n = cnt;
  return DD_OK;
}

int dd_plan_table(const dd_plan_t* p, int32_t r, int32_t which, void* host_buf, int64_t cap_bytes, int64_t* bytes) {
  if (!p || r < 0 || r >= (int)p->ranges.size() || !bytes || which < 0 || which > 8) return DD_ERR_INVALID;
  const auto& q = p->ranges[r];
  const void* srcs[9] = {q.h_meta.data(), q.h_dmin.data(), q.h_span.data(), q.h_meta2.data(), q.h_dmin2.data(),
                         q.h_span2.data(), q.h_delta.data(), q.h_chan.data(), q.h_chan2.data()};
  const size_t sizes[9] = {q.h_meta.size(), q.h_dmin.size(), q.h_span.size(), q.h_meta2.size(), q.h_dmin2.size(),
                           q.h_span2.size(), q.h_delta.size(), q.h_chan.size(), q.h_chan2.size()};
  if (which >= 3 && which != 7 && !q.pair_ok) return DD_ERR_INVALID;
  const void* src = srcs[which];
  const size_t n = sizes[which] * 4;
  *bytes = (int64_t)n;
  if (host_buf) {
    if (cap_bytes < (int64_t)n) return DD_ERR_NOMEM;
    memcpy(host_buf, src, n);
  }
  return DD_OK;
}

int dd_plan_tile_shape(const dd_plan_t* p, int32_t r, int32_t* trial_groups, int32_t* chans_per_stage, int32_t* stages,
                       int32_t* row_superwords, int32_t* cpad, int32_t* nblocks, int32_t* tiled) {
  if (!p || r < 0 || r >= (int)p->ranges.size()) return DD_ERR_INVALID;
  const auto& q = p->ranges[r];
  if (trial_groups) *trial_groups = q.G;
  if (chans_per_stage) *chans_per_stage = q.Cc;
  if (stages) *stages = q.stages;
  if (row_superwords) *row_superwords = q.T + q.Smax;
  if (cpad) *cpad = q.Cpad;
  if (nblocks) *nblocks = q.nblocks;
  if (tiled) *tiled = q.tiled_ok;
  return DD_OK;
}

int dd_plan_delta_chunks(const dd_plan_t* p, int32_t r, int32_t* chunks) {
  if (!p || !chunks || r < 0 || r >= (int)p->ranges.size()) return DD_ERR_INVALID;
  const auto& q = p->ranges[r];
  *chunks = !q.tiled_ok ? 0 : q.mode == dd::kModeDelta ? q.Cpad / q.Cc : q.nd;
  return DD_OK;
}

int dd_plan_tile_info(const dd_plan_t* p, int32_t r, int32_t* dm_per_cta, int32_t* words_per_cta, int32_t* lanes,
                      int32_t* flush_chans, int32_t* mode) {
  if (!p || r < 0 || r >= (int)p->ranges.size()) return DD_ERR_INVALID;
  const auto& q = p->ranges[r];
  if (dm_per_cta) *dm_per_cta = q.Dcta;
  if (words_per_cta) *words_per_cta = q.T;
  if (lanes) *lanes = q.NL;
  if (flush_chans) *flush_chans = q.flush;
  if (mode) *mode = q.mode;
  return DD_OK;
}

}  // extern "C"
