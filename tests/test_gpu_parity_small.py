"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, bit-exact.

Sizes: small enough for the oracle to finish in seconds, large enough to span several time tiles,
trial blocks and channel stages of the tiled kernel, with ragged tails in every dimension.
"""
import numpy as np
import pytest

from paper_2605_03531_b200 import workloads as W

from _util import check_full, gpu_run, oracle_full

pytestmark = pytest.mark.gpu

DIRECT, TILED = 1, 2


def _rng_filterbank(nbeams, nchans, nsamps, bits, seed):
    rng = np.random.default_rng(seed)
    return rng.integers(0, 2 ** bits, size=(nbeams, nchans, nsamps), dtype=np.uint8 if bits == 8 else np.uint16)


@pytest.mark.parametrize("variant", [DIRECT, TILED])
def test_cfg1_tiny_full(variant):
    w = W.CONFIGS[1]
    x = W.generate(w)
    plan, flat = gpu_run(w, x, variant)
    check_full(w, x, plan, flat)
    # the injected pulse is recovered at DM 50 (PAPER.md:387-393 injection test)
    out = plan.view_range(flat, 0)
    j, t = np.unravel_index(np.argmax(out), out.shape)
    assert abs(j - 50) <= 1 and 1024 <= t <= 1028


@pytest.mark.parametrize("variant", [DIRECT, TILED])
def test_cfg3_shaped_multirange_decimation(variant):
    """config-3 shape scaled down: 3 ranges with x1/x2/x4 decimation, zeroed channels, uint8."""
    w = W.scaled(W.CONFIGS[3], nchans=272, nsamps=2 ** 15 + 3,
                 ranges=[W.DMRange(0.0, 0.1, 203, 1), W.DMRange(200.0, 0.2, 150, 2), W.DMRange(600.0, 0.5, 141, 4)])
    x = W.generate(w)
    plan, flat = gpu_run(w, x, variant)
    check_full(w, x, plan, flat)
    if variant == TILED:
        assert plan.tile_info(0)["lanes"] == 8 and plan.tile_info(0)["mode"] == 2


@pytest.mark.parametrize("variant", [DIRECT, TILED])
def test_cfg2_shaped_large_delay_steps(variant):
    """config-2 shape scaled: delays change by several samples per trial (no reuse)."""
    w = W.scaled(W.CONFIGS[2], nchans=200, nsamps=2 ** 15, ranges=[W.DMRange(0.0, 0.5, 301, 1)])
    x = W.generate(w)
    plan, flat = gpu_run(w, x, variant)
    check_full(w, x, plan, flat)


@pytest.mark.parametrize("variant", [DIRECT, TILED])
def test_cfg4_shaped_uint16(variant):
    """uint16 input, x1 and x8 ranges: sums exceed 2^24, result must be fl32(exact sum): 0 ulp."""
    w = W.scaled(W.CONFIGS[4], nchans=520, nsamps=2 ** 16,
                 ranges=[W.DMRange(0.0, 0.25, 130, 1), W.DMRange(1000.0, 1.0, 77, 8)])
    x = W.generate(w)
    assert x.dtype == np.uint16
    want = oracle_full(w, x)
    assert want[0][0].max() > 2 ** 24        # the inexact regime is exercised
    plan, flat = gpu_run(w, x, variant)
    check_full(w, x, plan, flat, want)
    if variant == TILED:   # x1 range: uint16 lanes (table form 5); x8 range: 32-bit lanes
        assert plan.tile_info(0)["lanes"] == 8 and plan.tile_info(0)["mode"] == 5 and plan.tile_info(1)["lanes"] == 4


def test_uint16_extreme_values_exact_rounding():
    """All-65535 rows with a few odd values: sums near 2^32/8, every rounding case hit."""
    rng = np.random.default_rng(4)
    x = np.full((1, 300, 4096), 65535, dtype=np.uint16)
    x[0, ::7, :] -= rng.integers(0, 3, size=x[0, ::7, :].shape, dtype=np.uint16)
    w = W.Workload("u16_extreme", 500.0, -200.0 / 300, 300, 1.31072e-3, 4096, 1, 16,
                   (W.DMRange(0.0, 3.0, 9, 1), W.DMRange(30.0, 5.0, 5, 8)), 1, 0, 0)
    for variant in (DIRECT, TILED):
        plan, flat = gpu_run(w, x, variant)
        check_full(w, x, plan, flat)


@pytest.mark.parametrize("variant", [DIRECT, TILED])
def test_cfg5_shaped_multibeam(variant):
    w = W.scaled(W.CONFIGS[5], nchans=144, nsamps=2 ** 14, nbeams=3, ranges=[W.DMRange(0.0, 0.5, 90, 1)])
    x = W.generate(w)
    assert not np.array_equal(x[0], x[1])
    plan, flat = gpu_run(w, x, variant)
    check_full(w, x, plan, flat)


@pytest.mark.parametrize("decim", [1, 2, 4, 8])
@pytest.mark.parametrize("bits", [8, 16])
def test_all_decimations_saturated_input(decim, bits):
    """Saturated samples (255 / 65535 everywhere but a few): the packed 16-bit lanes reach their bound
    exactly at the flush interval; any missing flush or lane carry shows up."""
    nch, ns = 530, 20000 + decim - 1
    x = np.full((1, nch, ns), 2 ** bits - 1, dtype=np.uint8 if bits == 8 else np.uint16)
    x[0, 3, 100:200] = 0
    w = W.Workload("sat", 750.0, -200.0 / nch, nch, 1.31072e-3, ns, 1, bits, (W.DMRange(0.0, 1.0, 21, decim),), 1, 0, 0)
    plan, flat = gpu_run(w, x, TILED)
    check_full(w, x, plan, flat)
    out = plan.view_range(flat, 0)
    assert out.max() == np.float32(nch * decim * (2 ** bits - 1))


@pytest.mark.parametrize("nchans,nsamps,ndm,step", [
    (1, 700, 5, 10.0),       # single channel: identity (P8)
    (2, 64, 1, 0.0),         # one trial, DM 0
    (3, 5000, 7, 2.0),       # odd channel count: zero-padded channel rows
    (33, 3000, 37, 0.7),     # trial count not a multiple of the register block or the CTA block
    (64, 1211, 9, 3.0),
])
def test_edge_shapes(nchans, nsamps, ndm, step):
    x = _rng_filterbank(1, nchans, nsamps, 8, 100 + nchans)
    w = W.Workload("edge", 500.0, -200.0 / nchans, nchans, 1.024e-3, nsamps, 1, 8, (W.DMRange(0.0, step, ndm, 1),), 1, 0, 0)
    for variant in (DIRECT, TILED):
        plan, flat = gpu_run(w, x, variant)
        check_full(w, x, plan, flat)


def test_minimum_valid_span_nout_1():
    """nout = 1: the largest delay leaves a single valid sample."""
    nch = 16
    import oracle
    tab = oracle.delay_table(500.0, -200.0 / nch, nch, 1.024e-3, 1, 0.0, 1.0, 11)
    ns = int(tab.max()) + 1
    x = _rng_filterbank(1, nch, ns, 8, 5)
    w = W.Workload("nout1", 500.0, -200.0 / nch, nch, 1.024e-3, ns, 1, 8, (W.DMRange(0.0, 1.0, 11, 1),), 1, 0, 0)
    for variant in (DIRECT, TILED):
        plan, flat = gpu_run(w, x, variant)
        assert plan.range_info(0)["nout"] == 1
        check_full(w, x, plan, flat)


def test_too_short_and_overflow_are_rejected():
    from paper_2605_03531_b200 import binding as B
    with pytest.raises(B.DDError) as e:
        B.Plan(500.0, -200.0 / 16, 16, 1.024e-3, 100, [(0.0, 1.0, 11, 1)])
    assert e.value.code == B.DD_ERR_TOO_SHORT
    with pytest.raises(B.DDError) as e:
        B.Plan(500.0, -0.001, 65535, 1.024e-3, 100000, [(0.0, 0.0, 1, 8)], in_bits=16)
    assert e.value.code == B.DD_ERR_OVERFLOW


def test_delay_table_matches_oracle_all_configs():
    """dd_plan_get_delays == oracle table for the five BASELINE configs (plan builder parity)."""
    import oracle
    from paper_2605_03531_b200 import binding as B
    for k, w in W.CONFIGS.items():
        if k == 5:
            w = W.scaled(w, nbeams=1)
        plan = B.Plan.from_workload(w)
        for r, rg in enumerate(w.ranges):
            want = oracle.delay_table(w.f_top_mhz, w.chan_width_mhz, w.nchans, w.tsamp_s, rg.decim, rg.dm_lo, rg.dm_step, rg.ndm)
            got = plan.get_delays(r)
            assert np.array_equal(got.astype(np.int64), want), (k, r)
        plan.destroy()


def test_host_path_and_caller_workspace():
    import torch
    w = W.scaled(W.CONFIGS[3], nchans=96, nsamps=2 ** 14,
                 ranges=[W.DMRange(0.0, 0.1, 40, 1), W.DMRange(200.0, 0.2, 24, 2)])
    x = W.generate(w)
    want = oracle_full(w, x)
    plan, flat = gpu_run(w, x, TILED, host_path=True)
    check_full(w, x, plan, flat, want, check_pad=False)   # the host path copies whole rows back
    ws = torch.empty(plan.workspace_bytes(), dtype=torch.uint8, device="cuda")
    plan.set_workspace(ws)
    xin = torch.from_numpy(x).cuda()
    out = torch.full((plan.out_elems(),), -1.0, dtype=torch.float32, device="cuda")
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        plan.execute(xin, out, s)
    s.synchronize()
    check_full(w, x, plan, out.cpu().numpy(), want)
    assert plan.launches() == 4


# ---- kernel v2: table modes, tile shapes, two-level packed accumulators ---------------------------------

@pytest.mark.parametrize("mode", [0, 1, 2])
def test_table_modes_agree_on_fine_dm_grid(mode):
    """A fine DM grid (every delay step 0 or 1) run through each table form of the tiled kernel:
    0 = one load per trial, 1 = load skipped on equal offsets, 2 = delta bits + uniform skip branch."""
    # byte_lanes 0: keep the undecimated range on 16-bit lanes (else: 8-bit lanes, next test)
    w = W.scaled(W.CONFIGS[3], nchans=260, nsamps=2 ** 14 + 5,
                 ranges=[W.DMRange(0.0, 0.1, 150, 1), W.DMRange(600.0, 0.5, 75, 4)])
    x = W.generate(w)
    plan, flat = gpu_run(w, x, TILED, tuning=dict(mode=mode, byte_lanes=0))
    assert plan.tile_info(0)["mode"] == mode
    check_full(w, x, plan, flat)


@pytest.mark.parametrize("bits,decim,step,tuning,mode,lanes", [
    (8, 4, 0.9, None, 6, 8),              # x4 uint8: the lowest channels step by 1.09 samples per trial -> delta chunks + offsets chunks
    (8, 1, 0.23, dict(mode=6), 6, 8),     # x1 uint8, 1.11 at the bottom (automatic: 8-bit lanes): hybrid on request
    (16, 1, 0.23, dict(mode=6), 7, 8),    # x1 uint16 (automatic: uint16 lanes, offsets table): hybrid on the same lanes
    (16, 4, 0.9, None, 6, 4),             # x4 uint16: 32-bit lanes
])
def test_hybrid_table_modes(bits, decim, step, tuning, mode, lanes):
    """Ranges that are delta-codable except for their lowest channels (dd_internal.h kModeHybrid / kModeWideHybrid):
    every output element against the oracle, with saturated rows on both sides of the chunk boundary; then the same
    plan with the offsets table forced (mode 1), identical bits."""
    nch, ns = 300, 2 ** 15 + 37
    rng = np.random.default_rng(31 * bits + decim)
    x = rng.integers(0, 2 ** bits, size=(2, nch, ns), dtype=np.uint8 if bits == 8 else np.uint16)
    x[0, 40:60, :] = 2 ** bits - 1
    x[1, 250:, 1000:20000] = 2 ** bits - 1
    w = W.Workload("hybrid", 750.0, -200.0 / nch, nch, 1.31072e-3, ns, 2, bits, (W.DMRange(100.0, step, 150, decim),), 1, 0, 0)
    plan, flat = gpu_run(w, x, TILED, tuning=tuning)
    info = plan.tile_info(0)
    assert (info["mode"], info["lanes"]) == (mode, lanes), info
    nd, shape = plan.delta_chunks(0), plan.tile_shape(0)
    assert 0 < nd < shape["cpad"] // shape["chans_per_stage"]
    check_full(w, x, plan, flat)
    plan2, flat2 = gpu_run(w, x, TILED, tuning=dict(mode=1, byte_lanes=0))
    assert plan2.tile_info(0)["mode"] == 1
    assert np.array_equal(flat.view(np.uint32)[flat != -1.0], flat2.view(np.uint32)[flat2 != -1.0])


def test_hybrid_forced_on_a_coarse_grid_with_few_delta_chunks():
    """dd_tuning_t::mode = 6 on a config-2-shaped range: only the first chunks qualify; several trial blocks and tiles."""
    w = W.scaled(W.CONFIGS[2], nchans=200, nsamps=2 ** 15, ranges=[W.DMRange(0.0, 0.5, 301, 1)])
    x = W.generate(w)
    plan, flat = gpu_run(w, x, TILED, tuning=dict(mode=6, byte_lanes=0))
    assert plan.tile_info(0)["mode"] == 6 and plan.delta_chunks(0) >= 1
    check_full(w, x, plan, flat)


def test_delta_mode_is_refused_for_coarse_dm_grid():
    """Delay steps above 1 cannot be delta coded: the plan falls back to the offsets table."""
    w = W.scaled(W.CONFIGS[2], nchans=64, nsamps=2 ** 14, ranges=[W.DMRange(0.0, 2.0, 40, 1)])
    x = W.generate(w)
    plan, flat = gpu_run(w, x, TILED, tuning=dict(mode=2))
    assert plan.tile_info(0)["mode"] == 0
    check_full(w, x, plan, flat)


@pytest.mark.parametrize("tile", ["16,32,32,3", "16,32,4,6", "8,64,16,4", "4,128,8,3", "2,256,8,2", "1,512,4,2",
                                  "8,32,16,4", "4,64,8,5", "1,256,8,2"])
def test_tile_shapes(tile):
    """Every CTA shape (trial groups x superwords, channels per stage, ring depth) gives the same bits."""
    g, t, cc, st = (int(v) for v in tile.split(","))
    w = W.scaled(W.CONFIGS[3], nchans=100, nsamps=2 ** 15 + 77,
                 ranges=[W.DMRange(0.0, 0.1, 77, 1), W.DMRange(50.0, 1.5, 19, 2)])   # delta + offsets tables
    x = W.generate(w)
    plan, flat = gpu_run(w, x, TILED, tuning=dict(trial_groups=g, words_per_cta=t, chans_per_stage=cc, stages=st))
    assert plan.tile_shape(0)["tiled"] == 1 and plan.tile_shape(0)["chans_per_stage"] == cc
    assert plan.tile_info(0)["dm_per_cta"] == 8 * g and plan.tile_info(0)["words_per_cta"] == t
    check_full(w, x, plan, flat)


def test_packed_lane_residual_plus_saturated_interval():
    """Two-level accumulators: lanes keep their low byte at a flush, so the next interval starts from up to
    255.  First 256 channels sum to 255 (mod 256 = 255), the next 256 are saturated: 255 + 256*255 = 65535
    is the exact lane bound."""
    nch, ns = 768, 6000
    x = np.zeros((1, nch, ns), dtype=np.uint8)
    x[0, 0, :] = 255
    x[0, 256:512, :] = 255
    x[0, 512:, :] = 7
    x[0, 300, 1000:1100] = 3
    w = W.Workload("resid", 750.0, -200.0 / nch, nch, 1.31072e-3, ns, 1, 8, (W.DMRange(0.0, 0.2, 19, 1),), 1, 0, 0)
    plan, flat = gpu_run(w, x, TILED)
    assert plan.tile_info(0)["lanes"] == 8 and plan.tile_info(0)["flush_chans"] == 256
    check_full(w, x, plan, flat)


def test_many_flushes_and_wide_fallback():
    """uint8 x8 decimation: lanes hold at most 32 saturated channels between flushes.  3840 channels = 120
    flushes of the upper bytes (the 16-bit lane bound allows 256); 3872 channels go to 32-bit lanes."""
    for nch, lanes in ((3840, 8), (3872, 4)):
        ns = 8 * 700
        x = np.full((1, nch, ns), 255, dtype=np.uint8)
        x[0, 5::97, :] = 254
        w = W.Workload("flushes", 750.0, -200.0 / nch, nch, 1.31072e-3, ns, 1, 8, (W.DMRange(0.0, 10.0, 9, 8),), 1, 0, 0)
        plan, flat = gpu_run(w, x, TILED)
        assert plan.tile_info(0)["lanes"] == lanes
        check_full(w, x, plan, flat)


@pytest.mark.parametrize("bits", [8, 16])
def test_byte_lanes_coarse_dm_grid(bits):
    """Undecimated range with delay steps of several samples: 8-bit lanes (uint16: low and high byte planes,
    S = S_lo + 256 S_hi, one rounding).  Saturated rows next to random ones reach the lane bounds; 600 channels
    cross two flushes."""
    nch, ns = 600, 2 ** 15 + 3
    rng = np.random.default_rng(77 + bits)
    x = rng.integers(0, 2 ** bits, size=(2, nch, ns), dtype=np.uint8 if bits == 8 else np.uint16)
    x[0, 100:420, :] = 2 ** bits - 1
    x[1, ::3, 500:9000] = 2 ** bits - 1
    w = W.Workload("bytes", 750.0, -200.0 / nch, nch, 655.36e-6, ns, 2, bits, (W.DMRange(0.0, 3.0, 70, 1),), 1, 0, 0)
    plan, flat = gpu_run(w, x, TILED, tuning=dict(byte_lanes=1))
    assert plan.tile_info(0)["lanes"] == 16 and plan.tile_info(0)["mode"] == 0
    assert plan.launches() == 1 + bits // 8
    check_full(w, x, plan, flat)
    plan2, flat2 = gpu_run(w, x, TILED, tuning=dict(byte_lanes=0))
    assert plan2.tile_info(0)["lanes"] == (8 if bits == 8 else 4)
    assert np.array_equal(flat.view(np.uint32)[flat != -1.0], flat2.view(np.uint32)[flat2 != -1.0])
    # automatic choice: byte lanes for uint8; uint16 samples in 16-bit lanes (E / O accumulators, table form 5)
    plan3, flat3 = gpu_run(w, x, TILED)
    info = plan3.tile_info(0)
    assert (info["lanes"], info["mode"]) == ((16, 0) if bits == 8 else (8, 5))
    assert plan3.launches() == 2
    assert np.array_equal(flat.view(np.uint32)[flat != -1.0], flat3.view(np.uint32)[flat3 != -1.0])


@pytest.mark.parametrize("bits", [8, 16])
def test_host_path_pieces_and_beams(bits):
    """dd_execute_host dedisperses a few trial blocks per launch and copies each finished piece back on its own
    stream: several pieces per range, two beams, delta / byte-plane / 32-bit-lane ranges."""
    import torch
    nch, ns = 96, 2 ** 14
    rng = np.random.default_rng(900 + bits)
    x = rng.integers(0, 2 ** bits, size=(2, nch, ns), dtype=np.uint8 if bits == 8 else np.uint16)
    w = W.Workload("hostpieces", 750.0, -200.0 / nch, nch, 1.31072e-3, ns, 2, bits,
                   (W.DMRange(0.0, 0.1, 700, 1), W.DMRange(70.0, 2.5, 300, 1), W.DMRange(820.0, 5.0, 41, 4)), 1, 0, 0)
    want = oracle_full(w, x)
    from paper_2605_03531_b200 import binding as B
    plan = B.Plan.from_workload(w)
    hin = torch.from_numpy(x.view(np.int16) if bits == 16 else x).pin_memory()
    hout = torch.full((plan.out_elems(),), -1.0, dtype=torch.float32).pin_memory()
    for _ in range(2):   # twice: the events and the staging buffers are reused
        hout.fill_(-1.0)
        plan.execute_host(hin, hout, torch.cuda.current_stream())
        check_full(w, x, plan, hout.numpy(), want, check_pad=False)


@pytest.mark.parametrize("variant", [TILED, DIRECT])
def test_host_path_async_back_to_back_steps(variant):
    """dd_execute_host_async: five steps with different inputs queued back to back (two staging slots used
    alternately, uploads on their own stream), one dd_host_wait, every step's plane equal to the oracle's; then the
    synchronous call on the same plan, and a change of stream in between."""
    import torch
    from paper_2605_03531_b200 import binding as B
    nch, ns, steps = 80, 2 ** 13 + 40, 5
    w = W.Workload("hostasync", 750.0, -200.0 / nch, nch, 1.31072e-3, ns, 2, 8,
                   (W.DMRange(0.0, 0.1, 300, 1), W.DMRange(30.0, 2.5, 100, 1), W.DMRange(280.0, 5.0, 33, 4)), 1, 0, 0)
    rng = np.random.default_rng(4242)
    xs = [rng.integers(0, 256, size=(2, nch, ns), dtype=np.uint8) for _ in range(steps)]
    plan = B.Plan.from_workload(w)
    plan.set_kernel(variant)
    hins = [torch.from_numpy(x).pin_memory() for x in xs]
    houts = [torch.full((plan.out_elems(),), -1.0, dtype=torch.float32).pin_memory() for _ in range(steps)]
    side = torch.cuda.Stream()
    for s in range(steps):
        plan.execute_host_async(hins[s], houts[s], torch.cuda.current_stream())
    plan.host_wait()
    for s in range(steps):
        check_full(w, xs[s], plan, houts[s].numpy(), check_pad=False)
    # another stream (everything in flight is drained first), then the synchronous form
    houts[0].fill_(-1.0), houts[1].fill_(-1.0)
    plan.execute_host_async(hins[3], houts[0], side)
    plan.execute_host(hins[1], houts[1], side)
    check_full(w, xs[3], plan, houts[0].numpy(), check_pad=False)
    check_full(w, xs[1], plan, houts[1].numpy(), check_pad=False)
    plan.host_wait()   # nothing in flight: returns at once


def test_shared_partial_sums_variant():
    """DD_KERNEL_SHARED: the sum of a channel quad is reused across neighbouring trials
    while none of its delays changes.  Fewer executed adds, identical bits (delta ranges; others unchanged)."""
    SHARED = 3
    w = W.scaled(W.CONFIGS[3], nchans=272, nsamps=2 ** 15 + 3,
                 ranges=[W.DMRange(0.0, 0.1, 203, 1), W.DMRange(200.0, 0.2, 150, 2), W.DMRange(600.0, 3.0, 41, 4)])
    x = W.generate(w)
    plan, flat = gpu_run(w, x, SHARED)
    assert [plan.tile_info(r)["mode"] for r in range(3)] == [2, 2, 6]   # (the coarse x4 range: hybrid, not shared)
    check_full(w, x, plan, flat)
    # saturated input: the quad sum 4*1020 still fits its 16-bit lane
    xs = np.full_like(x, 255)
    xs[0, 7, 50:90] = 0
    plan, flat = gpu_run(w, xs, SHARED)
    check_full(w, xs, plan, flat)


# ---- NEXT-1: spectrum-major input, ascending bands ------------------------------------

@pytest.mark.parametrize("variant", [DIRECT, TILED])
@pytest.mark.parametrize("layout,ascending", [(1, False), (0, True), (1, True)])
def test_input_layouts_uint8(variant, layout, ascending):
    """[beam][time][channel] input (the thesis's ring-buffer order) and bands listed from the lowest
    channel upwards give the bits of the channel-major, descending description of the same data."""
    w = W.scaled(W.CONFIGS[3], nchans=150, nsamps=2 ** 14 + 9, nbeams=2,
                 ranges=[W.DMRange(0.0, 0.1, 90, 1), W.DMRange(50.0, 2.0, 33, 1), W.DMRange(200.0, 0.2, 70, 2),
                         W.DMRange(600.0, 0.5, 40, 4)])
    x = W.generate(w)
    plan, flat = gpu_run(w, x, variant, in_layout=layout, ascending=ascending)
    check_full(w, x, plan, flat)


@pytest.mark.parametrize("layout,ascending", [(1, False), (1, True), (0, True)])
def test_input_layouts_uint16(layout, ascending):
    w = W.scaled(W.CONFIGS[4], nchans=200, nsamps=2 ** 15,
                 ranges=[W.DMRange(0.0, 0.25, 60, 1), W.DMRange(1000.0, 1.0, 37, 8)])
    x = W.generate(w)
    for variant in (DIRECT, TILED):
        plan, flat = gpu_run(w, x, variant, in_layout=layout, ascending=ascending)
        check_full(w, x, plan, flat)


def test_bad_layout_and_zero_width_are_rejected():
    from paper_2605_03531_b200 import binding as B
    for kw in ({"in_layout": 7}, {}):
        with pytest.raises(B.DDError) as e:
            B.Plan(500.0, 0.0 if not kw else -1.0, 16, 1.024e-3, 4096, [(0.0, 1.0, 3, 1)], **kw)
        assert e.value.code == B.DD_ERR_INVALID
    with pytest.raises(B.DDError) as e:   # ascending band whose lowest channel is not above 0 MHz
        B.Plan(-10.0, 1.0, 16, 1.024e-3, 4096, [(0.0, 1.0, 3, 1)])
    assert e.value.code == B.DD_ERR_INVALID


@pytest.mark.parametrize("layout", [0, 1])
def test_streaming_blocks_join_exactly(layout):
    """dd_stream_*: a long filterbank pushed block by block (PAPER.md:351 ring-buffer blocks) with a carried halo.
    The new samples of consecutive pushes, concatenated, are the oracle's dedispersion of the whole series."""
    import torch
    from paper_2605_03531_b200 import binding as B
    nch, block, npush = 64, 4096, 5
    w = W.Workload("stream", 750.0, -200.0 / nch, nch, 1.31072e-3, block * npush, 2, 8,
                   (W.DMRange(0.0, 0.1, 120, 1), W.DMRange(30.0, 4.0, 50, 1), W.DMRange(200.0, 0.5, 60, 4)), 1, 0, 0)
    x = _rng_filterbank(w.nbeams, nch, w.nsamps, 8, 4242)
    want = oracle_full(w, x)                       # [beam][range] -> [ndm][N/k - maxd]
    st = B.Stream(w.f_top_mhz, w.chan_width_mhz, nch, w.tsamp_s, block,
                  [(r.dm_lo, r.dm_step, r.ndm, r.decim) for r in w.ranges], nbeams=2, in_layout=layout)
    assert st.hist % 64 == 0 and st.block == block
    out = torch.empty(st.plan.out_elems(), dtype=torch.float32, device="cuda")
    pieces = [[[] for _ in w.ranges] for _ in range(w.nbeams)]
    for p in range(npush):
        blk = x[:, :, p * block:(p + 1) * block]
        blk = np.ascontiguousarray(blk.transpose(0, 2, 1) if layout == 1 else blk)
        st.push(torch.from_numpy(blk).cuda(), out, torch.cuda.current_stream())
        torch.cuda.synchronize()
        flat = out.cpu().numpy()
        for b in range(w.nbeams):
            for r, rg in enumerate(w.ranges):
                rows = st.plan.view_range(flat, r, beam=b)
                pieces[b][r].append(rows[:, rows.shape[1] - block // rg.decim:].copy())
    for b in range(w.nbeams):
        for r, rg in enumerate(w.ranges):
            got = np.concatenate(pieces[b][r], axis=1)
            maxd = st.plan.range_info(r)["maxd"]
            ref = want[b][r]
            assert ref.shape[1] == got.shape[1] - maxd
            assert np.array_equal(got[:, maxd:].view(np.uint32), ref.view(np.uint32)), (b, r)
    st.destroy()


def test_row_pitch_regression_gpu():
    """a staged row wider than the last channel's (per-channel rounding) overran the next row of
    the shared-memory stage.  The reported plan, plus a few hundred-trial fine grids of the same band."""
    nch, ns = 128, 4096
    rng = np.random.default_rng(5)
    x = rng.integers(0, 256, size=(1, nch, ns), dtype=np.uint8)
    for lo, step, ndm in [(23.979060551005045, 0.01977691285836024, 16), (3.0, 0.0213, 333), (11.7, 0.0171, 400)]:
        w = W.Workload("rowpitch", 1399.6529111929856, -2.664227517042692, nch, 327.68e-6, ns, 1, 8,
                       (W.DMRange(lo, step, ndm, 1),), 1, 0, 0)
        plan, flat = gpu_run(w, x, TILED)
        assert plan.tile_shape(0)["tiled"] == 1
        check_full(w, x, plan, flat)


SUBBAND = 4
_CW = -200.0 / 4096   # SPOTLIGHT's channel width: neighbouring channels differ by less than a sample in delay


@pytest.mark.parametrize("nchans", [272, 271, 64])
def test_subband_pairs_variant(nchans):
    """DD_KERNEL_SUBBAND: two-channel sub-band rows pre-summed once per execute, one load and
    one add per trial and PAIR -- half the brute-force adds, identical bits.  Odd channel counts pair the last channel
    with a zero row; a coarse range in the same plan keeps its own kernel."""
    w = W.Workload("pairs", 600.0, _CW, nchans, 1.31072e-3, 2 ** 15 + 3, 1, 8,
                   (W.DMRange(0.0, 0.1, 203, 1), W.DMRange(200.0, 0.2, 150, 2), W.DMRange(600.0, 3.0, 41, 4),
                    W.DMRange(900.0, 0.9, 90, 1), W.DMRange(100.0, 300.0, 12, 2)), 353103, 128, 12)
    x = W.generate(w)
    plan, flat = gpu_run(w, x, SUBBAND)
    en = [plan.pair_info(r)["enabled"] for r in range(5)]
    assert en == [1, 1, 1, 1, 0]
    assert plan.executed_adds() < 0.56 * plan.work()[1]
    assert plan.launches() == 5 + 5 + 4
    check_full(w, x, plan, flat)


def test_subband_saturated_input_and_flushes():
    """Pair rows hold up to 2 * 255 * decim per 16-bit lane and the packed accumulators are flushed every flush/2 pair
    rows: saturated input over 1024 channels crosses several flushes at the exact lane bound."""
    nch, ns = 1024, 2 ** 14
    x = np.full((1, nch, ns), 255, dtype=np.uint8)
    x[0, 7::13, :] = 254
    x[0, :, 5000:5003] = 0
    for decim, step in ((1, 0.3), (4, 1.2), (8, 2.4)):
        w = W.Workload("pairsat", 750.0, _CW, nch, 1.31072e-3, ns, 1, 8, (W.DMRange(0.0, step, 90, decim),), 1, 0, 0)
        plan, flat = gpu_run(w, x, SUBBAND)
        assert plan.pair_info(0)["enabled"] == 1
        check_full(w, x, plan, flat)


def test_subband_host_path_and_two_beams():
    nch, ns = 128, 2 ** 14
    rng = np.random.default_rng(4242)
    x = rng.integers(0, 256, size=(2, nch, ns), dtype=np.uint8)
    w = W.Workload("pairhost", 700.0, _CW, nch, 1.31072e-3, ns, 2, 8,
                   (W.DMRange(0.0, 1.0, 300, 1), W.DMRange(300.0, 2.0, 100, 2)), 1, 0, 0)
    plan, flat = gpu_run(w, x, SUBBAND, host_path=True)
    assert plan.pair_info(0)["enabled"] == 1 and plan.pair_info(1)["enabled"] == 1
    check_full(w, x, plan, flat, check_pad=False)


def test_random_plans_every_element():
    """Seeded random small plans -- fine, borderline (hybrid) and coarse DM grids, all decimations, both input widths,
    one or two beams, both input layouts and band orders, two ranges each -- through the automatic kernel choice, every
    output element against the oracle.
    Covers the table forms and lane widths in combinations no hand-written case names."""
    rng = np.random.default_rng(20261105)
    seen = set()
    for i in range(28):
        nch = int(rng.integers(20, 180))
        f_top = float(rng.uniform(400.0, 1500.0))
        cw = -float(rng.uniform(0.2, 0.5)) * f_top / nch
        tsamp = float(rng.choice([327.68e-6, 655.36e-6, 1.31072e-3]))
        bits = 16 if i % 3 == 2 else 8
        nbeams = 1 + (i % 2)
        f_lo = f_top + (nch - 1) * cw
        ranges, maxd_in = [], 0
        for k in range(2):
            decim = int(rng.choice([1, 2, 4, 8]))
            sweep_per_dm = 4.148808e3 * (f_lo ** -2 - f_top ** -2) / (tsamp * decim)
            kind = (i + k) % 3
            step = float((rng.uniform(0.2, 0.95), rng.uniform(0.95, 1.5), rng.uniform(1.5, 5.0))[kind]) / sweep_per_dm
            ndm = int(rng.integers(40, 260)) if kind < 2 else int(rng.integers(10, 90))
            lo = float(rng.uniform(0.0, 30.0)) * step
            ranges.append(W.DMRange(lo, step, ndm, decim))
            maxd_in = max(maxd_in, (int(sweep_per_dm * (lo + ndm * step)) + 2) * decim)
        ns = maxd_in + int(rng.integers(700, 5000))
        w = W.Workload("rand%d" % i, f_top, cw, nch, tsamp, ns, nbeams, bits, tuple(ranges), 1, 0, 0)
        x = rng.integers(0, 2 ** bits, size=(nbeams, nch, ns), dtype=np.uint8 if bits == 8 else np.uint16)
        x[0, nch // 3, : ns // 2] = 2 ** bits - 1
        plan, flat = gpu_run(w, x, TILED, in_layout=(i // 4) % 2, ascending=bool((i // 8) % 2))   # all four input conventions
        check_full(w, x, plan, flat)
        seen |= {(plan.tile_info(r)["lanes"], plan.tile_info(r)["mode"]) for r in range(2)}
    assert {(8, 2), (16, 0), (8, 5), (8, 6)} <= seen, seen   # delta, 8-bit lanes, uint16 lanes and hybrid all occurred
