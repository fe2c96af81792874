// dd_internal.h -- private declarations shared by dd_plan.cu (host plan builder + C ABI) and
// dd_kernels.cu (CUDA kernels + launchers).  Not part of the public boundary (include/dd.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "dd.h"

namespace dd {

// Packed time word ("superword"): 16 bytes holding NL time lanes of one channel.
//   lane m of superword i is the decimated sample y[i + m*H]   (H = lane segment length)
//   NL = 16: sixteen 8-bit lanes (byte k of word q holds lane 4q+k); undecimated uint8 ranges whose delay steps
//            are too coarse for the delta table.  (On request, dd_tuning_t::byte_lanes = 1, uint16 input is split into
//            two such byte planes that are dedispersed one after the other: S = S_lo + 256*S_hi.)
//   NL = 8: eight 16-bit lanes (word q holds lanes 2q (low half) and 2q+1 (high half)): samples with headroom for
//           packed sums (uint8, decimated or delta-coded), or the uint16 samples themselves (kModeWide)
//   NL = 4: four 32-bit lanes
// A delay of d samples is a shift of d superwords for every lane at once, so any delay is a
// 16-byte aligned access.
constexpr int kSuperwordBytes = 16;
constexpr int kRD = 8;            // trials register-blocked per thread (one "trial group"), NL = 8 and 4
constexpr int kRD16 = 4;          // the same for NL = 16 (twice the accumulator registers per trial)
__host__ __device__ constexpr int trials_per_thread(int NL) { return NL == 16 ? kRD16 : kRD; }

// How the tiled kernel finds the staged superword of (channel, trial):
//   kModeGeneral       per channel and trial: a 32-bit byte offset inside the stage (row of the channel included), one
//                      shared-memory load per trial
//   kModeGeneralReuse  same table; the load is skipped when the offset equals the previous trial's
//   kModeDelta         every delay step inside a trial group is 0 or 1 (fine DM grids): per channel the
//                      offset of the group's first trial plus one "changed" bit per later trial; a changed
//                      bit advances the address by one superword and reloads, otherwise the registers are reused
//   kModeDeltaShare    kModeDelta plus sharing of partial sums (variant DD_KERNEL_SHARED): while
//                      no channel of a quad changes its delay, the quad's sum wa+wb+wc+wd is the same for
//                      consecutive trials and is added as ONE term.  Same table, same bits, fewer executed adds.
//   kModeDeltaPair     exact two-channel sub-bands (variant DD_KERNEL_SUBBAND): neighbouring channels
//                      2v, 2v+1 differ in delay by delta_v or delta_v + 1 for EVERY trial of the range, so the two
//                      pre-summed rows U_p[i] = y_2v[i] + y_2v+1[i + delta_v + p], p = 0, 1 (built once per execute,
//                      interleaved: superword 2i + p) replace both channels: one load and one add per trial and PAIR.
//                      Table per quad of pairs: one "changed" bit per trial step and pair as in kModeDelta, plus a byte
//                      offset per trial and pair that selects the row (U_0 or U_1) and the delay.
//   kModeWide          uint16 samples in the 16-bit lanes of NL = 8 (undecimated uint16 input on coarse DM grids): a lane has no
//                      headroom, so a word w of two lanes is accumulated as E += w (mod 2^32) and O += w >> 16; lane sums are
//                      E - (O << 16) and O.  Table: eight 32-bit byte offsets inside the stage (row included) per (channel,
//                      trial group); the load is skipped when the offset equals the previous trial's.
//   kModeHybrid        per channel CHUNK (pipeline stage): the leading chunks -- the highest channels, whose delay steps
//                      never exceed 1 -- carry the delta table, the remaining ones the offsets table with reuse.  A range whose
//                      lowest channels step by a little more than one sample per trial keeps the delta kernel for most
//                      of its channels instead of losing it altogether.
//   kModeWideHybrid    the same for uint16 lanes (kModeWide adder in both kinds of chunk)
enum TiledMode {
  kModeGeneral = 0, kModeGeneralReuse = 1, kModeDelta = 2, kModeDeltaShare = 3, kModeDeltaPair = 4, kModeWide = 5,
  kModeHybrid = 6, kModeWideHybrid = 7
};
__host__ __device__ constexpr bool is_hybrid(int mode) { return mode == kModeHybrid || mode == kModeWideHybrid; }
__host__ __device__ constexpr bool is_wide(int mode) { return mode == kModeWide || mode == kModeWideHybrid; }
__host__ __device__ constexpr bool is_delta(int mode) {
  return mode == kModeDelta || mode == kModeDeltaShare || mode == kModeDeltaPair;
}

// kModeDelta processes channels in quads A,B,C,D.  The changed bits of a quad share one 32-bit word laid
// out so that each byte feeds one R2P (register -> 7 predicates): bit n%7 of byte n/7, n = (j-1)*4 + q
// for trial step j = 1..kRD-1 of channel q = 0..3.
__host__ __device__ constexpr int delta_bit(int j, int q) { return (((j - 1) * 4 + q) / 7) * 8 + ((j - 1) * 4 + q) % 7; }

// Staged rows start and end on 128-byte lines (8 superwords): upper bound of the staged length beyond T
// for a block whose delays spread over `spread` superwords.
__host__ __device__ constexpr int aligned_span(int spread) { return (spread + 7 + 7) / 8 * 8; }

// Meta bytes per pipeline stage of Cc channels and G trial groups: one 32-bit byte offset inside the stage (row
// included) per (channel, trial) -- or one 16-byte entry per channel quad and trial group in delta mode.
__host__ __device__ constexpr size_t tiled_meta_bytes(int mode, int NL, int Cc, int G) {
  if (mode == 4) return (size_t)(Cc / 8) * (size_t)G * 80;  // kModeDeltaPair: 5 entries per quad of pairs (8 rows)
  if (is_delta(mode)) return (size_t)(Cc / 4) * (size_t)G * 16;
  return (size_t)Cc * (size_t)G * (size_t)trials_per_thread(NL) * 4;  // one 32-bit byte offset per (channel, trial)
}

struct RangePlan {
  // definition
  double dm_lo = 0, dm_step = 0;
  int ndm = 0, decim = 1;
  int64_t ns = 0, maxd = 0, nout = 0, pitch = 0, offset = 0;
  int64_t row0 = 0;    // index of this range's first trial among the rows of one beam (sum of ndm of earlier ranges)
  int64_t in_off = 0;  // first input sample this range reads (0 unless the plan keeps only the tail: dd_plan_create_tail)
  std::vector<int32_t> delays;  // host copy [ndm][nchans]
  // tiled kernel shape
  int NL = 8;        // lanes per superword
  int RD = 8;        // trials per thread = trials_per_thread(NL)
  int planes = 1;    // 2: uint16 input as low-byte and high-byte planes (NL = 16)
  int64_t plane_bytes = 0;  // bytes of one packed plane in the workspace
  int flush = 0;     // channels between flushes of the 16-bit lanes (0: never, 32-bit lanes)
  int mode = 0;      // TiledMode
  int nd = 0;        // hybrid modes: leading channel chunks with the delta table (0 otherwise)
  int G = 0;         // trial groups per CTA (kRD trials each)
  int T = 0;         // superwords per CTA (multiple of 32)
  int Dcta = 0;      // trials per CTA = G*kRD
  int Cc = 0;        // channels per pipeline stage
  int stages = 0;
  int tiled_ok = 0;  // 0: the tile does not fit shared memory, this range runs the direct kernel
  int nblocks = 0;   // trial blocks = ceil(ndm/Dcta)
  int Smax = 0;      // largest delay spread inside one trial block (superwords)
  int Cpad = 0;      // nchans rounded up to a multiple of Cc (zero rows)
  int64_t H = 0;     // lane segment length (superwords), multiple of 16
  int64_t Wp = 0;    // row pitch of the packed array (superwords), multiple of 4
  int64_t ntau = 0;  // time tiles = ceil(H/T)
  int64_t ws_offset = 0;  // byte offset of this range's packed array in the workspace
  int64_t ws_bytes = 0;
  size_t smem_bytes = 0;
  // tables of the tiled kernel: host copies (built by dd_plan.cu build_tables) and their device twins
  std::vector<uint32_t> h_meta;
  std::vector<int32_t> h_dmin, h_span;
  std::vector<int32_t> h_chan;  // [nblocks][Cpad] channel whose packed row is staged in row s of the block's chunk sequence
  uint4* d_meta = nullptr;      // general: [nblocks][Cpad][G] RD 32-bit byte offsets inside the stage;
                                // delta: [nblocks][chunk][G][Cc/4] {changed bits, offA|offB<<16, offC|offD<<16, any-changed bits};
                                // hybrid: a block's delta chunks first, then its offsets chunks (dd_plan.cu build_tables)
  int32_t* d_dmin = nullptr;    // [nblocks][Cpad] first delay of the block (superwords)
  int32_t* d_span = nullptr;    // [nblocks][Cpad] delay spread of the block (superwords)
  int32_t* d_chan = nullptr;    // [nblocks][Cpad] h_chan
  int32_t* d_delays = nullptr;  // [ndm][nchans], only for the direct kernel (lazy)
  // two-channel sub-bands (kModeDeltaPair), built by dd_plan_set_kernel(DD_KERNEL_SUBBAND): rows are pairs
  int pair_ok = 0;        // 1: this range runs in pair mode under DD_KERNEL_SUBBAND
  int Cc2 = 0;            // pairs per pipeline stage (= Cc / 2; a stage holds Cc rows: U_0 and U_1 of each pair)
  int Smax2 = 0;          // largest staged span of a pair row (superwords)
  int stages2 = 0;
  int64_t ws2_offset = 0, ws2_bytes = 0;  // pair array [nbeams][Cpad][Wp] superwords in the workspace: rows 2v, 2v+1 = U_0, U_1 of pair v
  std::vector<uint32_t> h_meta2;          // [nblocks][Cpad/8][G][5 entries of 4 words]: {changed bits, any bits, 0, 0}, then 8 16-bit offsets per pair
  std::vector<int32_t> h_dmin2, h_span2;  // [nblocks][Cpad]: start / span of the staged row (both rows of a pair: those of channel 2v)
  std::vector<int32_t> h_delta;           // [Cpad/2] delta_v
  std::vector<int32_t> h_chan2;           // [nblocks][Cpad] row of the pair array staged in each row of the block's chunk sequence
  uint4* d_meta2 = nullptr;
  int32_t *d_dmin2 = nullptr, *d_span2 = nullptr, *d_delta = nullptr, *d_chan2 = nullptr;
  int64_t adds_pair = 0;  // adds executed per beam in pair mode (pre-sums included)
};

}  // namespace dd

struct dd_plan {
  // config
  double f_top = 0, cw = 0, tsamp = 0;  // internal order: channel 0 = highest frequency, cw < 0
  int nchans = 0, nbeams = 0, in_bits = 8;
  int layout = 0;      // DD_LAYOUT_* of the caller's input
  int ascending = 0;   // caller's channel c is internal channel nchans-1-c
  int64_t nsamps = 0;
  int64_t tail_new = 0;  // > 0: every range produces only its last tail_new/decim (+ < 16) samples
  std::vector<dd::RangePlan> ranges;
  int64_t beam_stride = 0, out_elems = 0;
  int64_t dm_samples = 0, adds = 0;
  int64_t rows_per_beam = 0;  // sum of ndm over the ranges
  // dd_plan_set_row_stats: [nbeams*rows_per_beam][2] = sum x, sum x^2 of every DM-time row, accumulated by the
  // epilogue of the dedispersion kernels (caller-owned device memory; nullptr = off)
  unsigned long long* row_stats = nullptr;
  int device = 0;
  int variant = DD_KERNEL_AUTO;
  int sps_warp_kernel = 1;  // single-pulse search: the barrier-free kernel where it applies (experiment switch)
  // workspace
  int64_t ws_bytes = 0;      // packed copies of every range
  int64_t ws_pair_bytes = 0; // + the pair arrays of DD_KERNEL_SUBBAND (0 until that variant is selected)
  void* ws = nullptr;
  int64_t ws_have = 0;       // bytes behind ws
  bool ws_owned = false;
  // per-kernel timing hook (dd_plan_set_profiling): events[slot][2*launch + {0,1}]
  int prof_slots = 0;
  mutable long long prof_calls = 0;
  std::vector<cudaEvent_t> prof_events;
  mutable std::vector<int> prof_kind, prof_range, prof_count;  // per slot*max_launches
  // host path: staging buffers, a copy stream and events so that the device-to-host copy of finished trial
  // blocks overlaps the dedispersion of the following ones
  // Two slots of staging buffers, so that back-to-back calls (dd_execute_host_async) overlap the upload of step i+1
  // and the tail of the download of step i with the kernels in between.
  void* h_in_dev[2] = {nullptr, nullptr};
  float* h_out_dev[2] = {nullptr, nullptr};
  cudaStream_t copy_stream = nullptr;  // device-to-host pieces
  cudaStream_t h2d_stream = nullptr;   // host-to-device input
  cudaStream_t host_stream = nullptr;  // the caller's stream of the last host call (dd_host_wait synchronises it)
  cudaEvent_t ev_in_ready[2] = {nullptr, nullptr};  // input of the slot has arrived
  cudaEvent_t ev_in_free[2] = {nullptr, nullptr};   // the kernels that read the slot's input are done
  cudaEvent_t ev_out_free[2] = {nullptr, nullptr};  // the slot's output has been copied back
  long long host_calls = 0;            // slot of a call = host_calls % 2
  int host_pieces = 4;                 // launches per range of the host path (dd_plan_set_host_pieces)
  std::vector<cudaEvent_t> host_events;
};

namespace dd {

// records "<what>: <cuda error string>" for dd_last_cuda_error() (thread-local) and returns DD_ERR_CUDA (dd_plan.cu)
int cuda_fail(cudaError_t e, const char* what);

// launchers (dd_kernels.cu); all enqueue on `stream` and return the CUDA error of the launch
cudaError_t launch_pack(const dd_plan* p, const RangePlan& r, const void* in_dev, cudaStream_t stream);
// all byte planes of the trial blocks blk0 .. blk0+nblk-1 (nblk <= 0: to the end of the range)
cudaError_t launch_tiled(const dd_plan* p, const RangePlan& r, float* out_dev, cudaStream_t stream, int blk0 = 0,
                         int nblk = 0);
cudaError_t launch_direct(const dd_plan* p, const RangePlan& r, const void* in_dev, float* out_dev,
                          cudaStream_t stream);
// kModeDeltaPair: pre-sum the packed rows of a range into its pair rows (reads P, writes P2)
cudaError_t launch_pairs(const dd_plan* p, const RangePlan& r, cudaStream_t stream);
inline bool use_pairs(const dd_plan* p, const RangePlan& r) { return p->variant == DD_KERNEL_SUBBAND && r.pair_ok; }
cudaError_t configure_kernels(const dd_plan* p);  // opt in to the dynamic shared memory sizes
size_t tiled_smem_bytes(const RangePlan& r);

}  // namespace dd
