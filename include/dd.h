/*
 * dd.h -- C ABI of libdd: brute-force incoherent dedispersion on one NVIDIA B200 (sm_100a).
 *
 * The operation (PAPER.md = /root/reference/PAPER.md, arxiv/paper_2605_03531):
 *   - cold-plasma dispersion delay, PAPER.md:256-263 (Eq. 1.1):
 *         dt = 4.14881 ms * DM * (nu1^-2 - nu2^-2)   [nu in GHz, DM in pc cm^-3]
 *     turned into integer sample delays per channel c and trial j of range r
 *         d_r(c,j) = round( K * DM_{r,j} * (f_c^-2 - f_top^-2) / (tsamp * decim_r) ),
 *         K = 4.148808e3 s MHz^2 cm^3/pc, f in MHz, DM_{r,j} = dm_lo_r + j*dm_step_r,
 *     evaluated in IEEE double, rounded half away from zero (BASELINE.json north_star;
 *     DESIGN.md readings A1, A4, A6);
 *   - brute-force dedispersion, the O(m x N) direct sum per trial of PAPER.md:421 (section 3.2),
 *     over a plan of many trial DMs, PAPER.md:317 (section 2.1):
 *         y_r[b][c][t'] = sum_{i<decim_r} in[b][c][decim_r*t' + i]            (time decimation, a SUM)
 *         S_r[b][j][t'] = sum_{c<nchans} y_r[b][c][t' + d_r(c,j)]              t' = 0 .. nout_r-1
 *         out           = fl32(S)                                              (one rounding, RNE)
 *     with ns_r = nsamps / decim_r (tail dropped), maxd_r = d_r(nchans-1, ndm_r-1),
 *     nout_r = ns_r - maxd_r (valid samples only; no padding, no wrap-around);
 *   - DM = 0 is the plain channel sum ("0 DM time series").
 *
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback.  All functions return
 * 0 on success or a negative dd_status code; nothing throws or aborts across this boundary.
 * "dev" pointers are CUDA device pointers on the device that was current at dd_plan_create;
 * "host" pointers are ordinary host memory (pinned memory makes the *_host call asynchronous).
 */
#ifndef DD_H_
#define DD_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DD_VERSION 200 /* major*100 + minor */

typedef enum dd_status {
  DD_OK = 0,
  DD_ERR_INVALID = -1,   /* null pointer; nchans<1; chan_width==0; lowest channel <= 0 MHz; unknown layout; tsamp<=0; nsamps<1; nbeams<1;
                            in_bits not 8/16; nranges<1; decim not in {1,2,4,8}; ndm<1; dm_lo<0; dm_step<0;
                            bad range index; unknown kernel variant */
  DD_ERR_TOO_SHORT = -2, /* some range has nout_r < 1 (largest delay >= decimated length) */
  DD_ERR_OVERFLOW = -3,  /* nchans * (2^in_bits - 1) * decim >= 2^32: exact integer sums impossible */
  DD_ERR_ALIGN = -4,     /* in_dev / out_dev / workspace not 16-byte aligned */
  DD_ERR_CUDA = -5,      /* a CUDA runtime call failed; text via dd_last_cuda_error() */
  DD_ERR_NOMEM = -6,     /* host or device allocation failed; workspace too small */
  DD_ERR_DEVICE = -7     /* the current CUDA device is not the one the plan / stream was created on */
} dd_status;

/* One DM range: trials DM_j = dm_lo + j*dm_step, j = 0..ndm-1, dedispersed on the input summed
 * over `decim` adjacent samples (decim in {1,2,4,8}; 2/4/8 are used for high-DM ranges). */
typedef struct dd_range {
  double dm_lo;    /* pc cm^-3, >= 0 */
  double dm_step;  /* pc cm^-3, >= 0 */
  int32_t ndm;     /* >= 1 */
  int32_t decim;   /* 1, 2, 4 or 8 */
} dd_range_t;

/* The filterbank and the DM plan.  `ranges` is copied by dd_plan_create. */
typedef struct dd_config {
  double f_top_mhz;       /* frequency of channel 0, MHz: the highest channel if chan_width < 0, the lowest if > 0 */
  double chan_width_mhz;  /* f_c = f_top + c*chan_width, non-zero.  Delays are always referenced to the HIGHEST
                             channel (Eq. 1.1); with chan_width > 0 (ascending band) that is channel nchans-1 and
                             the result equals that of the same data with the channel order reversed. */
  int32_t nchans;
  double tsamp_s;         /* sampling time of the input, seconds */
  int64_t nsamps;         /* time samples per channel */
  int32_t nbeams;         /* independent beams sharing the plan, batched in one call */
  int32_t in_bits;        /* 8 (uint8) or 16 (uint16) unsigned samples */
  int32_t nranges;
  const dd_range_t* ranges;
  int32_t in_layout;      /* DD_LAYOUT_*: how `in` is stored */
} dd_config_t;

/* Input layouts.  DD_LAYOUT_CHANNEL_MAJOR [nbeams][nchans][nsamps] (time contiguous) is BASELINE.json's
 * "channels x time samples".  DD_LAYOUT_SPECTRUM_MAJOR [nbeams][nsamps][nchans] (channel contiguous) is how the
 * thesis's shared-memory ring buffers hold a beam: blocks of 800 / 25600 spectra of 4096 channels
 * (2.2); the corner turn is fused into the pack / decimation kernel. */
#define DD_LAYOUT_CHANNEL_MAJOR 0
#define DD_LAYOUT_SPECTRUM_MAJOR 1

typedef struct dd_plan dd_plan_t; /* opaque */

/* Kernel variants selectable for tests and measurements (dd_plan_set_kernel). */
#define DD_KERNEL_AUTO 0   /* the tiled kernel below, tile shape chosen per range */
#define DD_KERNEL_DIRECT 1 /* one thread per (trial, sample), delays from a global table: slow, simple */
#define DD_KERNEL_TILED 2  /* shared-memory staged, register-blocked, packed-lane adder (the product path) */
#define DD_KERNEL_SHARED 3 /* the tiled kernel with partial sums shared between neighbouring trials whose delays
                              coincide over a channel quad (delta-coded ranges; other ranges as DD_KERNEL_TILED):
                              an exact shortcut that executes fewer adds than the brute-force count of
                              PAPER.md:421.  Same bits. */
#define DD_KERNEL_SUBBAND 4 /* exact two-channel sub-bands (the thesis uses redundancy the same way
                              for the FFA).  In a delta-coded range neighbouring channels 2v, 2v+1 differ in
                              delay by delta_v or delta_v + 1 for every trial, so S[j][t] = sum_v U_{p(v,j)}[v][t + d(2v,j)]
                              with the two pre-summed rows U_p[v][i] = y_2v[i] + y_2v+1[i + delta_v + p] (one extra streaming
                              kernel per range and execute).  Half the adds of the brute-force count, same bits.  Ranges
                              where some pair needs a third row run as DD_KERNEL_SHARED.  Needs twice the workspace:
                              dd_plan_set_kernel re-allocates a plan-owned workspace; a caller-owned one must be set again
                              (dd_plan_workspace_bytes reports the new size). */

/*
 * dd_plan_create: host work (delay tables, per-range sizes, tile shapes) plus device allocations and
 * table uploads on the current CUDA device.  Allocates the plan-owned workspace for the packed /
 * decimated copies of the input unless dd_plan_set_workspace is called before the first execute.
 * On success *plan_out owns all of it; release with dd_plan_destroy.  Synchronises the device once.
 */
int dd_plan_create(const dd_config_t* cfg, dd_plan_t** plan_out);

/*
 * dd_plan_create_tail: a plan over cfg->nsamps input samples that produces, for every range, only the outputs
 * whose sums end in the last new_samps input samples: rows of nout_r = new_samps/decim_r + (0..15/decim_r) samples
 * ending at the same last sample as dd_plan_create's rows.  Each range skips the leading input it does not need
 * (in steps of 16 samples).  Used by the stream calls below; layouts and queries as for dd_plan_create.
 * DD_ERR_TOO_SHORT if nsamps < new_samps + maxd_r*decim_r for some range (the window cannot supply the promised
 * new_samps/decim_r outputs); DD_ERR_INVALID if new_samps < 1 or new_samps > nsamps.
 */
int dd_plan_create_tail(const dd_config_t* cfg, int64_t new_samps, dd_plan_t** plan_out);

/*
 * dd_plan_create_host: the host half of dd_plan_create only -- validation, delay tables (Eq. 1.1), per-range
 * sizes, tile shapes and the tables the tiled kernel reads -- without any CUDA call.  The plan answers every
 * query below but cannot execute (dd_execute returns DD_ERR_INVALID).  For inspection and CPU-side tests.
 */
int dd_plan_create_host(const dd_config_t* cfg, dd_plan_t** plan_out);

/*
 * dd_plan_create_tuned: dd_plan_create (host_only = 0) or dd_plan_create_host (host_only != 0) with the automatic
 * choices of the plan builder overridden -- for tests and measurements; the results never change, only the kernel
 * shape.  tuning == NULL means automatic.  (The library reads no environment variables.)
 *   mode        -1 automatic; 0 / 1 / 2 force the table form of the tiled kernel (see dd_plan_tile_info); the delta
 *               form is refused (falls back to 0) for a range with a delay step above 1 between neighbouring trials;
 *               6 asks for the hybrid form wherever at least one leading channel chunk can be delta-coded (automatic:
 *               only when that part is large enough to pay)
 *   byte_lanes  -1 automatic; 1: 8-bit lanes wherever they apply, uint16 input as two byte planes (automatic for uint8;
 *               undecimated uint16 input automatically runs on uint16 lanes instead, table form 5); 0: never use 8-bit or
 *               uint16 lanes (undecimated coarse ranges then run on 16-/32-bit lanes with the table forms 0 / 1)
 *   trial_groups, words_per_cta, chans_per_stage, stages
 *               all 0: automatic; else the CTA shape: trial_groups * words_per_cta in {256, 512} threads,
 *               words_per_cta a multiple of 32, chans_per_stage in {4, 8, .., 32}, 2 <= stages <= 8.  A shape that
 *               fails the checks of the automatic path (shared-memory budget, offset widths) sends the range to the
 *               direct kernel; the ring depth is lowered to what fits.
 * DD_ERR_INVALID for out-of-range mode / byte_lanes.
 */
typedef struct dd_tuning {
  int32_t mode;
  int32_t byte_lanes;
  int32_t trial_groups, words_per_cta, chans_per_stage, stages;
} dd_tuning_t;
int dd_plan_create_tuned(const dd_config_t* cfg, const dd_tuning_t* tuning, int32_t host_only, dd_plan_t** plan_out);

/*
 * dd_execute: enqueue the whole hot path on `cuda_stream` (a cudaStream_t passed as void*; NULL = the
 * legacy default stream): pack/decimate kernels for every range, then the dedispersion kernels, which
 * write fp32 results straight into out_dev.  No host synchronisation, no allocation.
 *   in_dev : [nbeams][nchans][nsamps] (time contiguous) or [nbeams][nsamps][nchans] (in_layout), uint8 or
 *            uint16 (in_bits), 16-byte aligned, read only.
 *   out_dev: dd_plan_out_elems() floats, 16-byte aligned.  Beam b, range r, trial j, sample t' lives at
 *            out_dev[b*beam_stride + offset_r + j*pitch_r + t'],  t' < nout_r; the pitch_r - nout_r pad
 *            floats of each row are left untouched.
 * One execute per plan may be in flight at a time (the workspace is shared).  The caller owns both
 * buffers and the stream.  DD_ERR_DEVICE if the current device is not the plan's.
 */
int dd_execute(const dd_plan_t* plan, const void* in_dev, float* out_dev, void* cuda_stream);

/*
 * dd_execute_host: the same path from HOST buffers, end to end: copies in_host to a plan-owned device
 * buffer, runs the kernels of dd_execute on `cuda_stream` a few trial blocks at a time and copies each finished
 * piece of the DM-time plane back to out_host on a plan-owned copy stream while the next piece is computed
 * (pinned host memory is needed for that overlap), then waits for everything before returning.  Layouts as in dd_execute, except that whole rows are
 * copied back, so the pad floats of out_host are overwritten with unspecified values.  The staging buffers are
 * allocated on first use (DD_ERR_NOMEM if that fails) and freed by dd_plan_destroy.  Refusals (missing workspace or
 * tables, wrong device) come before anything is enqueued; if a CUDA call fails later, both streams are drained before
 * the error is returned, so no copy touches the caller's buffers after the call.
 */
int dd_execute_host(dd_plan_t* plan, const void* in_host, float* out_host, void* cuda_stream);

/*
 * dd_execute_host_async / dd_host_wait: the same end-to-end path for a stream of beams or blocks, one call per step
 * (a search node processes one beam after the other).  dd_execute_host_async enqueues what dd_execute_host
 * does and returns without waiting; dd_host_wait blocks until every call made so far has finished (all results are in
 * their out_host buffers, all in_host buffers have been read).  The plan owns two slots of staging buffers, used
 * alternately, and a second copy stream for the uploads, so that with back-to-back calls the upload of step i+1 and the
 * end of the download of step i run while the kernels of the steps in between compute: per step the time tends to
 * max(kernels, upload, download) instead of their partial sum.  Rules: both host buffers page-locked (else the copies
 * serialise); in_host must stay unchanged and out_host untouched until dd_host_wait returns; the out_host buffers of two
 * consecutive calls must differ (their copies may overlap in time); the same cuda_stream for consecutive calls (a change
 * of stream first waits for everything in flight).  dd_execute_host == dd_execute_host_async + dd_host_wait.  Errors as
 * dd_execute_host; after an error everything in flight has been drained.
 */
int dd_execute_host_async(dd_plan_t* plan, const void* in_host, float* out_host, void* cuda_stream);
int dd_host_wait(dd_plan_t* plan);
/* Launches per range of the host path (1 .. 64, default 4): each finished piece of a range's rows is copied back while the
 * next is computed.  More pieces shorten the copy left over after the last kernel of a synchronous call; fewer pieces
 * cost fewer partial waves of CTAs, which is what matters when calls are queued back to back. */
int dd_plan_set_host_pieces(dd_plan_t* plan, int32_t pieces);

/* dd_plan_destroy: frees host and device memory of the plan.  NULL is a no-op returning DD_OK.  The
 * caller must make sure no execute of this plan is still running. */
int dd_plan_destroy(dd_plan_t* plan);

/* ---- queries: host only, no device work ---------------------------------------------------- */

/* Total floats of the output buffer (all beams, all ranges, pitch padding included). */
int dd_plan_out_elems(const dd_plan_t* plan, int64_t* total_floats);
/* Floats between consecutive beams in the output. */
int dd_plan_beam_stride(const dd_plan_t* plan, int64_t* floats);
/* Per-range sizes (any pointer may be NULL): ns_r, maxd_r, nout_r as defined above; pitch_floats =
 * nout_r rounded up to a multiple of 32; offset_floats = start of the range within one beam. */
int dd_plan_range_info(const dd_plan_t* plan, int32_t r, int64_t* ns_r, int64_t* maxd_r, int64_t* nout_r,
                       int64_t* pitch_floats, int64_t* offset_floats);
/* Test hook: copies the delay table of range r, int32 [ndm_r][nchans], into host_buf.  Channel 0 is the highest
 * frequency (for an ascending band that is the caller's last channel). */
int dd_plan_get_delays(const dd_plan_t* plan, int32_t r, int32_t* host_buf);
/* Sum over beams and ranges of ndm_r * nout_r (the "DM-trial x samples" of one execute) and the
 * brute-force add count, that number times nchans (O(m x N) per trial). */
int dd_plan_work(const dd_plan_t* plan, int64_t* dm_samples, int64_t* adds);
/* Kernel launches one dd_execute enqueues (pack + dedispersion) with the current kernel variant. */
int dd_plan_launches(const dd_plan_t* plan, int32_t* n_launches);
/* Sample additions one dd_execute actually performs with the current kernel variant, all beams (pre-sums of
 * DD_KERNEL_SUBBAND included).  Equals the brute-force count of dd_plan_work for DD_KERNEL_AUTO / TILED / DIRECT. */
int dd_plan_executed_adds(const dd_plan_t* plan, int64_t* adds);
/* DD_KERNEL_SUBBAND, range r (any pointer may be NULL): whether the range runs on two-channel sub-bands, pairs per
 * pipeline stage (each with its two pre-summed rows), superwords per staged row, number of pairs incl. padding. */
int dd_plan_pair_info(const dd_plan_t* plan, int32_t r, int32_t* enabled, int32_t* pairs_per_stage,
                      int32_t* row_superwords, int32_t* npairs);

/* ---- workspace and variants ------------------------------------------------------------------ */

/* Bytes of device scratch dd_execute needs for the packed / decimated input copies. */
int dd_plan_workspace_bytes(const dd_plan_t* plan, int64_t* bytes);
/* Use caller-owned device scratch (16-byte aligned, >= dd_plan_workspace_bytes) instead of the plan's
 * own; frees the plan-owned one.  dev == NULL switches back to a plan-owned allocation. */
int dd_plan_set_workspace(dd_plan_t* plan, void* dev, int64_t bytes);
/* Choose the dedispersion kernel variant (DD_KERNEL_*).  All variants produce identical bits. */
int dd_plan_set_kernel(dd_plan_t* plan, int32_t variant);
/* Tile shape the tiled kernel uses for range r (any pointer may be NULL): trials per CTA, packed time
 * words per CTA, time lanes per packed word (16 = 8-bit lanes, 8 = 16-bit lanes, 4 = 32-bit lanes), channels between
 * flushes of the packed accumulators (0: never), and the table mode: 0 = one shared-memory load per (channel, trial),
 * 1 = load skipped when the delay equals the previous trial's, 2 = delta form (all delay steps inside a
 * group of 8 trials are 0 or 1; one changed bit per trial), 5 = uint16 samples in the 16-bit lanes (undecimated
 * uint16 input; 32-bit byte offsets, load skipped on equal offsets), 6 = hybrid: the leading channel chunks (pipeline
 * stages; the highest channels, whose delay steps never exceed 1) use form 2, the others form 1, 7 = the same on
 * uint16 lanes (forms 2 / 5).  dd_plan_delta_chunks: how many leading chunks of chans_per_stage channels use form 2
 * (all of them for mode 2, none for 0 / 1 / 5). */
int dd_plan_tile_info(const dd_plan_t* plan, int32_t r, int32_t* dm_per_cta, int32_t* words_per_cta,
                      int32_t* lanes, int32_t* flush_chans, int32_t* mode);
int dd_plan_delta_chunks(const dd_plan_t* plan, int32_t r, int32_t* chunks);

/* More of the tile shape of range r (any pointer may be NULL): trial groups per CTA, channels per pipeline
 * stage, ring depth, superwords per staged channel row, channel rows incl. zero padding, trial blocks, and
 * whether the range runs the tiled kernel at all (0: delay steps too large for shared memory -> direct kernel). */
int dd_plan_tile_shape(const dd_plan_t* plan, int32_t r, int32_t* trial_groups, int32_t* chans_per_stage,
                       int32_t* stages, int32_t* row_superwords, int32_t* cpad, int32_t* nblocks, int32_t* tiled);
/* Test hook: the tables of the tiled kernel for range r as they are uploaded.  which = 0: the per-trial table
 * (uint32 words; layout per mode in DESIGN.md "Data layout"), 1: start of the staged row per (trial block,
 * channel) (int32 superwords, multiple of 8), 2: its length beyond the time tile (int32).  After
 * dd_plan_set_kernel(DD_KERNEL_SUBBAND): 3 = the pair-mode table (per trial block, quad of pairs and trial group 20
 * words: changed bits, any bits, 0, 0, then eight 16-bit byte offsets per pair), 4, 5 = start / span per staged row
 * (rows 2v, 2v+1 = the two pre-summed rows of pair v), 6 = delta_v per pair (int32).  7 = the channel whose packed row is
 * staged in each row of a trial block's chunk sequence (int32 [trial blocks][channel rows]; a permutation inside every
 * delta-coded chunk, chosen so that channels whose delays change at the same trials share a quad; tables 0 - 2 are
 * indexed by that row); 8 = the same for the pair mode (row of the pair array staged in each row; tables 3 - 5 are indexed
 * by the staged row, table 6 by the pair).  *bytes = size; the table is copied when host_buf != NULL
 * (DD_ERR_NOMEM if cap_bytes is too small). */
int dd_plan_table(const dd_plan_t* plan, int32_t r, int32_t which, void* host_buf, int64_t cap_bytes, int64_t* bytes);

/* ---- per-kernel timing (measurement hook) ------------------------------------------------------- */

/* Record a CUDA event before and after every kernel launch of the next `max_executes` calls of
 * dd_execute (slot = call index modulo max_executes).  max_executes = 0 switches it off and frees the
 * events.  The events are recorded on the caller's stream; nothing synchronises. */
int dd_plan_set_profiling(dd_plan_t* plan, int32_t max_executes);
/* After the caller has synchronised the stream: device time of each launch of execute slot `slot`, in
 * launch order.  ms[i] = milliseconds, kind[i] = 0 pack/decimate, 1 tiled dedispersion, 2 direct
 * dedispersion, range[i] = range index.  Arrays hold `cap` entries; *n = launches written. */
int dd_plan_kernel_times(const dd_plan_t* plan, int32_t slot, int32_t cap, float* ms, int32_t* kind,
                         int32_t* range, int32_t* n);

/* ---- streaming over blocks of spectra --------------------------------------------- */

/*
 * The thesis's pipeline receives a beam as a sequence of shared-memory blocks (800 or 25600 spectra of 4096
 * channels).  A stream dedisperses such a sequence: cfg->nsamps is the BLOCK length B (a multiple of
 * every range's decim).  The stream keeps the last `hist` >= max_r(maxd_r * decim_r) input samples on the device,
 * puts each new block behind them and runs a tail plan (dd_plan_create_tail, new_samps = B) over that window:
 *   dd_stream_create : builds that plan (query it through dd_stream_plan: out_elems, range_info, ...) and the
 *                      device window buffers, history zeroed.
 *   dd_stream_push   : block_dev = the next B samples of every beam, [nbeams][nchans][B] or [nbeams][B][nchans]
 *                      (cfg->in_layout); out_dev as for dd_execute on the window plan.  Enqueues copy + dd_execute +
 *                      carry on `cuda_stream`.  For range r the LAST B/decim_r samples of every row are new:
 *                      row[nout_r - B/decim_r + i] = S_r[j][p*B/decim_r - maxd_r + i] for push number p, so the new
 *                      pieces of consecutive pushes join exactly (the first maxd_r new samples of push 0 include the
 *                      zero pre-history); the up to 15/decim_r samples before them repeat the previous push.
 * One push per stream may be in flight at a time.
 */
typedef struct dd_stream dd_stream_t; /* opaque */
int dd_stream_create(const dd_config_t* cfg, dd_stream_t** stream_out);
int dd_stream_push(dd_stream_t* s, const void* block_dev, float* out_dev, void* cuda_stream);
const dd_plan_t* dd_stream_plan(const dd_stream_t* s);
int dd_stream_info(const dd_stream_t* s, int64_t* block_samples, int64_t* hist_samples, int64_t* pushes);
int dd_stream_destroy(dd_stream_t* s);

/* ---- single-pulse search on the DM-time plane -------------------------------------- */

/*
 * "The SPS module searches for statistically significant single pulses above a user-specified
 * threshold using time-domain boxcar filtering."  Per row x[0..nout_r) of the plane written by dd_execute:
 *     mean = (sum x)/n, sigma = sqrt((sum x^2)/n - mean^2)                        (sums exact, then IEEE double)
 *     for k < nwidths, w = 2^k:  B[t] = sum_{i<w} x[t+i], t <= n-w
 *         tmax  = first t with the largest B,   snr = sigma > 0 ? (B[tmax] - w*mean)/(sigma*sqrt(w)) : 0
 *         count = number of t with B[t] > w*mean + threshold*sigma*sqrt(w)
 *     (w > n: snr 0, tmax -1, count 0).
 * dd_sps_rows: rows of the outputs = nbeams * (sum of ndm_r); row = beam*(sum ndm) + (trials of earlier ranges) + j.
 * dd_sps_execute: plane_dev = the output buffer of dd_execute for this plan; snr_dev / tmax_dev / count_dev hold
 *     rows*nwidths elements ([row][k]); 1 <= nwidths <= 12; threshold finite.  Enqueues one kernel per range on
 *     `cuda_stream`.  DD_ERR_OVERFLOW if (nchans*(2^in_bits-1)*decim)^2 * nout_r >= 2^63 for some range (sum x^2
 *     would not be exact; uint8 SPOTLIGHT-shaped data is far below).
 *
 * The candidate list ("The list of candidates thus generated is filtered ..."): every (row, k, t) with
 * B[t] > w*mean + threshold*sigma*sqrt(w), with snr = (float)((B[t] - w*mean)/(sigma*sqrt(w))), ordered by row, then k,
 * then t.  dd_sps_candidates: after dd_sps_execute on the same plane with the same nwidths and threshold, count_dev as
 *     written by it.  Writes offsets_dev[rows*nwidths + 1] (int64) = exclusive scan of the counts -- the candidates of
 *     (row, k) are entries offsets[row*nwidths + k] .. offsets[row*nwidths + k + 1] of the list, the last element is the
 *     total -- and the first max_cands candidates to cand_dev.  Two small kernels plus one CTA per row that leaves at
 *     once when the row has no candidate; rows with candidates redo their boxcars.
 *
 * Row statistics from the dedispersion epilogue: dd_plan_set_row_stats(plan, stats_dev) with stats_dev = rows*2
 *     uint64 (caller-owned device memory, 8-byte aligned; NULL switches it off; uint8 input only).  From then on
 *     dd_execute zeroes stats_dev and its dedispersion kernels add sum x and sum x^2 of every row they write (exact
 *     integers), and dd_sps_execute / dd_sps_candidates take S1, S2 from there instead of reading the plane a first
 *     time: the plane is then read ONCE.  The plane handed to them must be the one the last dd_execute of this plan
 *     wrote.  (dd_execute_host does not accumulate statistics.)
 */
typedef struct dd_sps_cand {
  int32_t row;         /* as in dd_sps_rows */
  int32_t width_log2;  /* k: boxcar width 2^k */
  int32_t t;           /* first sample of the window */
  float snr;
} dd_sps_cand_t;
int dd_sps_rows(const dd_plan_t* plan, int64_t* rows);
int dd_sps_execute(const dd_plan_t* plan, const float* plane_dev, int32_t nwidths, double threshold, float* snr_dev,
                   int32_t* tmax_dev, int32_t* count_dev, void* cuda_stream);
int dd_sps_candidates(const dd_plan_t* plan, const float* plane_dev, int32_t nwidths, double threshold,
                      const int32_t* count_dev, int64_t* offsets_dev, dd_sps_cand_t* cand_dev, int64_t max_cands,
                      void* cuda_stream);
int dd_plan_set_row_stats(dd_plan_t* plan, uint64_t* stats_dev);

/* ---- pulsar-side post-processing of dedispersed series ------------------------------ */

/*
 * The thesis's pulsar pipeline continues from the dedispersed series with downsampling, running-
 * median de-reddening and re-sampling that removes the frequency derivatives f1, f2
 * (Eqs 3.1-3.6).  These calls apply one such step to `nrows` independent series stored as rows
 * of floats: row r at in_dev + r*in_pitch, the first n floats valid -- e.g. the rows of one range of the DM-time
 * plane (in_dev = out_dev of dd_execute + offset_r, nrows = ndm_r, in_pitch = pitch_r, n = nout_r).  Device
 * pointers, 4-byte aligned; out rows at out_dev + r*out_pitch; all work is enqueued on `cuda_stream`, nothing
 * synchronises.  Readings where the thesis is silent: DESIGN.md C1-C7.
 *
 * dd_post_downsample  (C1)  out[k] = sum_{i<factor} in[k*factor + i], k < n/factor (a SUM, as the input decimation;
 *     tail dropped), accumulated in double in index order and rounded once.  out_pitch >= n/factor.
 *
 * dd_post_dered       (C2)  window odd, 1 <= window <= min(n, DD_POST_MAX_WINDOW), h = (window-1)/2:
 *         median[t] = the (h+1)-th smallest of in[s .. s+window),  s = min(max(t-h, 0), n-window)
 *     (centred on t; held at the first / last full window near the ends -- no padding), out[t] = in[t] - median[t].
 *     Exact order statistics of the floats (finite values; any sign).  median_dev or out_dev may be NULL (not
 *     wanted), not both; both have pitch out_pitch >= n.
 *
 * dd_resample_*       (C3-C7)  Eq 3.3 laid end to end: bin edges in input samples u_0 = 0, u_{k+1} = u_k + w_k,
 *         t = u_k*tsamp,  w_k = (1 + (f'*t)/F0) + (f''*(t*t))/(2*F0)          (IEEE double, this order)
 *     with (F0, f', f'') = (f0, -f1, -f2) if f1 <= 0, else the series is reversed and (Eqs 3.5, 3.6)
 *     F0 = (f0 + f1*T) + (f2*(T*T))/2, f' = f1 + f2*T, f'' = -f2, T = n*tsamp; M = number of complete bins
 *     (u_{k+1} <= n); w_k < 1/2 is refused (DD_ERR_INVALID).
 *         out[k] = fl32( sum_i in[i] * |[u_k,u_{k+1}) n [i,i+1)| )   left to right in double, no fused multiply-add;
 *     the reversed case reads the row backwards and writes it backwards.
 *     dd_resample_create builds and uploads the edges for series of n samples (current device);
 *     dd_resample_create_host builds them only (queries, no execute); dd_resample_info: M and the reversed flag;
 *     dd_resample_get_edges copies the M+1 edges (test hook); dd_resample_execute: out_pitch >= M.
 */
#define DD_POST_MAX_WINDOW 8191
int dd_post_downsample(const float* in_dev, int64_t nrows, int64_t in_pitch, int64_t n, int32_t factor, float* out_dev,
                       int64_t out_pitch, void* cuda_stream);
int dd_post_dered(const float* in_dev, int64_t nrows, int64_t in_pitch, int64_t n, int32_t window, float* median_dev,
                  float* out_dev, int64_t out_pitch, void* cuda_stream);
typedef struct dd_resample dd_resample_t; /* opaque */
int dd_resample_create(double f0_hz, double f1_hz_s, double f2_hz_s2, double tsamp_s, int64_t n, dd_resample_t** out);
int dd_resample_create_host(double f0_hz, double f1_hz_s, double f2_hz_s2, double tsamp_s, int64_t n, dd_resample_t** out);
int dd_resample_info(const dd_resample_t* r, int64_t* out_len, int32_t* reversed);
int dd_resample_get_edges(const dd_resample_t* r, double* host_buf);
int dd_resample_execute(const dd_resample_t* r, const float* in_dev, int64_t nrows, int64_t in_pitch, float* out_dev,
                        int64_t out_pitch, void* cuda_stream);
int dd_resample_destroy(dd_resample_t* r);

/* ---- errors ---------------------------------------------------------------------------------- */
const char* dd_strerror(int code);       /* static string for a dd_status */
const char* dd_last_cuda_error(void);    /* text of the last CUDA failure seen by this thread ("" if none) */
int dd_version(void);                    /* DD_VERSION */

#ifdef __cplusplus
}
#endif
#endif /* DD_H_ */
