"""CPU-only checks of the plan builder (step a1 and the host logic of the tiled kernel): no GPU needed.

dd_plan_create_host builds everything dd_plan_create builds except the device copies.  The delay tables are
compared with the oracle's (Eq. 1.1); the tables the tiled kernel reads (offsets / delta bits,
row starts and lengths) are decoded here, independently of the kernel, and must reproduce the delay table for
every (trial block, channel, trial) of all five BASELINE configs, padding rows and padding trials included.
"""
import numpy as np
import pytest

import oracle
from paper_2605_03531_b200 import binding as B
from paper_2605_03531_b200 import workloads as W


def _host_plan(w, **kw):
    return B.Plan.from_workload(W.scaled(w, nbeams=1) if w.nbeams > 1 else w, host_only=True, **kw)


def _padded_delays(plan, r, shape, rd):
    """[nblocks*Dcta][Cpad]: trials past the end repeat the last one, channel rows past nchans have delay 0."""
    d = plan.get_delays(r).astype(np.int64)
    ndm, nch = d.shape
    dcta = shape["trial_groups"] * rd
    rows = np.minimum(np.arange(shape["nblocks"] * dcta), ndm - 1)
    out = np.zeros((rows.size, shape["cpad"]), dtype=np.int64)
    out[:, :nch] = d[rows]
    return out


def _decode(plan, r):
    """Delays implied by the kernel tables: [nblocks][Dcta][Cpad] (absolute, superwords).  A trial block holds the
    table slices of its channel chunks one after the other: the first `delta_chunks` in the delta form (one 4-word
    entry per trial group and channel quad), the others as one 32-bit byte offset per (channel, trial)."""
    info, shape = plan.tile_info(r), plan.tile_shape(r)
    rd = 4 if info["lanes"] == 16 else 8
    g, cc, cpad, rowp, nb = (shape[k] for k in ("trial_groups", "chans_per_stage", "cpad", "row_superwords", "nblocks"))
    nchunks, nd = cpad // cc, plan.delta_chunks(r)
    assert nd == (nchunks if info["mode"] == 2 else nd) and (nd == 0 or info["mode"] in (2, 6, 7))
    assert 0 < nd < nchunks if info["mode"] in (6, 7) else True
    meta = plan.table(r, 0).astype(np.int64)
    dmin = plan.table(r, 1).astype(np.int64).reshape(nb, cpad)
    span = plan.table(r, 2).astype(np.int64).reshape(nb, cpad)
    wd, wg = cc // 4 * g * 4, cc * g * rd
    assert meta.size == nb * (nd * wd + (nchunks - nd) * wg)
    meta = meta.reshape(nb, nd * wd + (nchunks - nd) * wg)
    rowoff = (np.arange(cpad) % cc) * rowp                                    # superwords, row of the channel in its stage
    rel = np.zeros((nb, g, rd, cpad), dtype=np.int64)
    cd = nd * cc                                                              # channels under the delta form
    if nd:
        e = meta[:, :nd * wd].reshape(nb, nd, g, cc // 4, 4).transpose(0, 1, 3, 2, 4).reshape(nb, cd // 4, g, 4)  # [chunk][group][quad]
        anyb = np.zeros((nb, cd // 4, g), dtype=np.int64)
        for q in range(4):
            field = (e[..., 1 + q // 2] >> (16 * (q % 2))) & 0xFFFF           # [nb][quad][g] byte offset in the stage
            assert (field % 16 == 0).all()
            first = field // 16 - rowoff[q:cd:4][None, :, None]
            cur = first.copy()
            rel[:, :, 0, q:cd:4] = first.transpose(0, 2, 1)
            for j in range(1, rd):
                n = (j - 1) * 4 + q
                bit = (e[..., 0] >> ((n // 7) * 8 + n % 7)) & 1
                anyb |= bit << j
                cur = cur + bit
                rel[:, :, j, q:cd:4] = cur.transpose(0, 2, 1)
        assert np.array_equal(anyb, e[..., 3]), "any-changed bits are the OR of the quad's changed bits"
        assert (e[..., 0] & 0x80808080 == 0).all()                            # bit 7 of each byte is unused
    if nd < nchunks:                                                          # 32-bit byte offsets, row included
        e = meta[:, nd * wd:].reshape(nb, cpad - cd, g, rd)
        assert (e % 16 == 0).all()
        rel[:, :, :, cd:] = (e // 16 - rowoff[None, cd:, None, None]).transpose(0, 2, 3, 1)
    assert (rel >= 0).all() and (rel <= span[:, None, None, :]).all(), "every load stays inside the staged row"
    assert (dmin % 8 == 0).all() and (span % 8 == 0).all(), "staged rows start and end on 128-byte lines"
    assert (span + info["words_per_cta"] <= rowp).all()
    absd = rel + dmin[:, None, None, :]                                      # [nb][g][rd][row of the chunk sequence]
    # which channel each row holds (dd_plan_table 7): a permutation inside every chunk, the identity outside the delta form
    chan = plan.table(r, 7).astype(np.int64).reshape(nb, cpad)
    assert np.array_equal(np.sort(chan.reshape(nb, nchunks, cc), axis=2),
                          np.broadcast_to(np.arange(cpad).reshape(nchunks, cc), (nb, nchunks, cc)))
    assert np.array_equal(chan[:, cd:], np.broadcast_to(np.arange(cd, cpad), (nb, cpad - cd)))
    bych = np.empty_like(absd)
    np.put_along_axis(bych, np.broadcast_to(chan[:, None, None, :], absd.shape), absd, axis=3)
    return bych.reshape(nb * g * rd, cpad), rd, shape


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_kernel_tables_reproduce_the_delay_table(cfg):
    w = W.CONFIGS[cfg]
    plan = _host_plan(w)
    for r, rg in enumerate(w.ranges):
        want = oracle.delay_table(w.f_top_mhz, w.chan_width_mhz, w.nchans, w.tsamp_s, rg.decim, rg.dm_lo, rg.dm_step, rg.ndm)
        assert np.array_equal(plan.get_delays(r).astype(np.int64), want), (cfg, r)   # a1 against the oracle
        assert plan.tile_shape(r)["tiled"] == 1
        got, rd, shape = _decode(plan, r)
        assert np.array_equal(got, _padded_delays(plan, r, shape, rd)), (cfg, r)
        # shared memory of the launch: ring + barriers + prefetch pad fits the 227 KB opt-in limit
        mode = plan.tile_info(r)["mode"]
        rd = 4 if plan.tile_info(r)["lanes"] == 16 else 8
        meta_stage = shape["chans_per_stage"] // 4 * shape["trial_groups"] * 16 if mode == 2 else \
            shape["chans_per_stage"] * shape["trial_groups"] * rd * 4
        stage = -(-(shape["chans_per_stage"] * shape["row_superwords"] * 16 + meta_stage) // 128) * 128
        assert 128 + shape["stages"] * stage + 512 <= 227 * 1024 and shape["stages"] >= 2
    plan.destroy()


def test_lane_widths_and_modes_of_the_five_configs():
    """Which adder each range gets: delta-coded 16-bit lanes for the fine DM grids of
    config 3, 8-bit lanes for undecimated coarse grids of uint8 data, uint16 lanes for undecimated uint16 data, 32-bit
    lanes for decimated uint16."""
    want = {1: [(16, 0)], 2: [(16, 0)], 3: [(8, 2), (8, 2), (8, 2)], 4: [(8, 5), (4, 6)], 5: [(16, 0)]}
    for cfg, exp in want.items():
        plan = _host_plan(W.CONFIGS[cfg])
        for r, (lanes, mode) in enumerate(exp):
            info = plan.tile_info(r)
            assert info["lanes"] == lanes and (mode is None or info["mode"] == mode), (cfg, r, info)
            if lanes == 8 and info["mode"] in (5, 7):
                assert info["flush_chans"] == 0   # E (mod 2^32) and O never overflow: no flush
            elif lanes == 8:   # 255 + flush*maxval <= 65535, at most 256 flushes
                maxval = 255 * plan.ranges[r][3]
                assert 255 + info["flush_chans"] * maxval <= 65535
                assert -(-plan.tile_shape(r)["cpad"] // info["flush_chans"]) <= 256
        assert plan.launches() == 2 * len(exp)   # one pack and one dedispersion launch per range
        plan.destroy()


def test_hybrid_tables_where_only_the_lowest_channels_step_by_more_than_one():
    """The mode cliff: a DM step a little too coarse for the lowest channels.  A decimated range keeps the
    delta table for the chunks of channels above them (kModeHybrid) instead of dropping to the offsets table
    altogether; undecimated data stays on 8-bit (uint8) or uint16 lanes unless the hybrid form is asked for
    (dd_tuning_t::mode = 6: packed 16-bit lanes for uint8, uint16 lanes for uint16); a forced table form switches it off."""
    w3 = W.CONFIGS[3]
    cases = [  # (bits, (dm_lo, step, ndm, decim), tuning, expected mode, lanes)
        (8, (600.0, 0.9, 600, 4), None, 6, 8),              # x4: lowest-channel step 1.09 samples per trial
        (8, (0.0, 0.23, 600, 1), None, 0, 16),              # x1 uint8, step 1.11 at the bottom: byte lanes
        (8, (0.0, 0.23, 600, 1), dict(mode=6), 6, 8),       # ... hybrid on request
        (16, (0.0, 0.23, 600, 1), None, 5, 8),              # x1 uint16: uint16 lanes
        (16, (0.0, 0.23, 600, 1), dict(mode=6), 7, 8),      # ... hybrid on request, same lanes
        (16, (600.0, 0.9, 600, 4), None, 6, 4),             # x4 uint16: 32-bit lanes, hybrid
    ]
    for bits, rg, tuning, mode, lanes in cases:
        p = B.Plan(w3.f_top_mhz, -200.0 / 1032, 1024 + 8, w3.tsamp_s, 2 ** 16, [rg], in_bits=bits, host_only=True,
                   tuning=tuning)
        info = p.tile_info(0)
        assert (info["mode"], info["lanes"]) == (mode, lanes), (bits, rg, info)
        got, rd, shape = _decode(p, 0)
        assert np.array_equal(got, _padded_delays(p, 0, shape, rd))
        if mode in (6, 7):
            nd, cc = p.delta_chunks(0), shape["chans_per_stage"]
            d = p.get_delays(0).astype(np.int64)
            steps = np.diff(d, axis=0)
            steps[7::8] = 0                                  # the first trial of a group always loads
            first_bad = int(np.argmax(steps.max(axis=0) > 1))
            assert nd == first_bad // cc and 0 < nd < shape["cpad"] // cc
            forced = B.Plan(w3.f_top_mhz, -200.0 / 1032, 1024 + 8, w3.tsamp_s, 2 ** 16, [rg], in_bits=bits,
                            host_only=True, tuning=dict(mode=1, byte_lanes=0))
            assert forced.tile_info(0)["mode"] == 1 and forced.delta_chunks(0) == 0
            forced.destroy()
        p.destroy()


def test_ascending_band_has_the_descending_delay_table():
    w = W.scaled(W.CONFIGS[3], nchans=4096, nsamps=2 ** 16)
    a, d = _host_plan(w, ascending=True), _host_plan(w)
    for r in range(len(w.ranges)):
        assert np.array_equal(a.get_delays(r), d.get_delays(r))
        assert np.array_equal(a.table(r, 0), d.table(r, 0))
    assert [a.range_info(r) for r in range(3)] == [d.range_info(r) for r in range(3)]


def test_host_only_plans_cannot_execute_and_edge_shapes_build():
    lib = B._load()
    for nch, ndm, step, decim, bits in [(1, 5, 10.0, 1, 8), (3, 7, 2.0, 2, 8), (33, 37, 0.7, 1, 8), (64, 9, 3.0, 8, 16),
                                        (30000, 3, 0.01, 1, 8), (40000, 3, 0.01, 1, 8)]:
        p = B.Plan(700.0, -300.0 / nch, nch, 1e-3, 20000, [(0.0, step, ndm, decim)], in_bits=bits, host_only=True)
        got, rd, shape = _decode(p, 0)
        assert np.array_equal(got, _padded_delays(p, 0, shape, rd))
        assert lib.dd_execute(p._h, 16, 16, None) == B.DD_ERR_INVALID      # no device half
        info = p.tile_info(0)
        if info["mode"] == 2 or decim > 1:          # delta-coded or decimated: 16-bit lanes while they can hold the sums
            assert info["lanes"] == (8 if bits == 8 and nch <= 30720 else 4)
        elif bits == 16:                            # undecimated uint16, coarse steps: the samples in 16-bit lanes
            assert info["lanes"] == 8 and info["mode"] == 5
        else:                                       # undecimated uint8, coarse steps: byte lanes
            assert info["lanes"] == (16 if nch <= 30720 else 4)
        p.destroy()


def _row_invariant(plan, r):
    """Every staged row (time tile + span of the block's delays) fits the row pitch of the shared-memory stage."""
    info, shape = plan.tile_info(r), plan.tile_shape(r)
    if not shape["tiled"]:
        return True
    span = plan.table(r, 2).astype(np.int64)
    return bool((span + info["words_per_cta"] <= shape["row_superwords"]).all())


def test_row_pitch_covers_every_channels_span_regression():
    """the row pitch was sized from the LAST channel's delay spread only; delays are rounded per
    channel, so another channel's staged row could be 8 superwords longer and its bulk copy overran the next row.
    The reported case: span 16 where the last channel gave 8."""
    p = B.Plan(1399.6529111929856, -2.664227517042692, 128, 327.68e-6, 4096,
               [(23.979060551005045, 0.01977691285836024, 16, 1)], host_only=True)
    assert p.tile_shape(0)["tiled"] == 1 and _row_invariant(p, 0)
    got, rd, shape = _decode(p, 0)
    assert np.array_equal(got, _padded_delays(p, 0, shape, rd))
    p.destroy()


def test_row_pitch_property_random_plans():
    """Host-only property test over random small plans: multi-block fine grids (delta form), grids whose lowest channels
    step by a little more than one sample (hybrid forms) and coarse grids (offsets forms, 8-bit and uint16 lanes), both
    input widths.  Every staged row fits its pitch, and the kernel tables, decoded independently of the kernel, give back
    the plan's delay table for every (trial block, row, trial) -- channel dealing included."""
    rng = np.random.default_rng(20261104)
    checked = 0
    modes = {}
    for i in range(400):
        nch = int(rng.integers(4, 200))
        f_top = float(rng.uniform(300.0, 1500.0))
        cw = -float(rng.uniform(0.2, 0.6)) * f_top / nch
        tsamp = float(rng.choice([81.92e-6, 327.68e-6, 655.36e-6, 1.31072e-3]))
        decim = int(rng.choice([1, 2, 4, 8]))
        bits = 16 if i % 5 == 4 else 8
        kind = i % 4            # 0, 2: fine; 1: coarse; 3: borderline
        ndm = int(rng.integers(1, 80)) if kind == 1 else int(rng.integers(200, 1000))
        # fine: steps of at most ~1 sample at the lowest channel (delta form); coarse: a few samples per trial
        f_lo = f_top + (nch - 1) * cw
        sweep_per_dm = 4.148808e3 * (f_lo ** -2 - f_top ** -2) / (tsamp * decim)
        step = float(rng.uniform(1.0, 6.0) if kind == 1 else rng.uniform(0.9, 1.6) if kind == 3 else rng.uniform(0.2, 0.999)) / sweep_per_dm
        lo = float(rng.uniform(0.0, 50.0)) * step
        maxd = int(sweep_per_dm * (lo + ndm * step)) + 2
        try:
            p = B.Plan(f_top, cw, nch, tsamp, (maxd + 600) * decim, [(lo, step, ndm, decim)], in_bits=bits, host_only=True)
        except B.DDError:
            continue
        assert _row_invariant(p, 0), (i, f_top, cw, nch, tsamp, decim, lo, step, ndm)
        if p.tile_shape(0)["tiled"]:
            got, rd, shape = _decode(p, 0)
            assert np.array_equal(got, _padded_delays(p, 0, shape, rd)), (i, f_top, cw, nch, tsamp, decim, lo, step, ndm, bits)
        m = p.tile_info(0)["mode"]
        modes[m] = modes.get(m, 0) + 1
        checked += 1
        p.destroy()
    assert checked > 300 and modes.get(2, 0) > 100 and modes.get(6, 0) > 10 and modes.get(0, 0) > 10 and modes.get(5, 0) > 3, modes


def test_tuned_plan_goes_through_the_same_checks():
    """dd_plan_create_tuned: forced modes / shapes are validated like the automatic choice (no environment variables)."""
    w = W.scaled(W.CONFIGS[3], nchans=100, nsamps=2 ** 15, ranges=[W.DMRange(0.0, 0.1, 77, 1)])
    p = B.Plan.from_workload(w, host_only=True, tuning=dict(trial_groups=8, words_per_cta=64, chans_per_stage=16, stages=4))
    assert p.tile_info(0)["dm_per_cta"] == 64 and p.tile_shape(0)["tiled"] == 1 and _row_invariant(p, 0)
    p.destroy()
    # a shape the kernels are not built for is refused: the range falls back to the direct kernel, never a bad launch
    p = B.Plan.from_workload(w, host_only=True, tuning=dict(trial_groups=3, words_per_cta=100, chans_per_stage=5, stages=2))
    assert p.tile_shape(0)["tiled"] == 0
    p.destroy()
    # delta rows above 64 KB per stage cannot be addressed with 16-bit byte offsets: refused as well
    p = B.Plan.from_workload(w, host_only=True, tuning=dict(mode=2, trial_groups=1, words_per_cta=512, chans_per_stage=32, stages=2))
    assert p.tile_shape(0)["tiled"] == 0
    p.destroy()
    with pytest.raises(B.DDError):
        B.Plan.from_workload(w, host_only=True, tuning=dict(mode=7))
    import os
    os.environ["DD_MODE"] = "0"      # the library reads no environment variables
    try:
        p = B.Plan.from_workload(w, host_only=True)
        assert p.tile_info(0)["mode"] == 2
        p.destroy()
    finally:
        del os.environ["DD_MODE"]


def _decode_pairs(plan, r):
    """DD_KERNEL_SUBBAND tables -> delays of both channels of every pair: [nblocks*Dcta][Cpad]."""
    info, shape, pi = plan.tile_info(r), plan.tile_shape(r), plan.pair_info(r)
    g, cpad, nb, cc = shape["trial_groups"], shape["cpad"], shape["nblocks"], shape["chans_per_stage"]
    nvc, rowsw = pi["npairs"], pi["row_superwords"]
    assert nvc == cpad // 2 and pi["pairs_per_stage"] * 2 == cc
    e = plan.table(r, 3).reshape(nb, nvc // 4, g, 20).astype(np.int64)
    dmin = plan.table(r, 4).astype(np.int64).reshape(nb, cpad)
    span = plan.table(r, 5).astype(np.int64).reshape(nb, cpad)
    delta = plan.table(r, 6).astype(np.int64)
    assert (dmin % 8 == 0).all() and (span % 8 == 0).all() and (span + info["words_per_cta"] <= rowsw).all()
    assert np.array_equal(dmin[:, 0::2], dmin[:, 1::2]) and np.array_equal(span[:, 0::2], span[:, 1::2])
    # which pair sits in which double row (dd_plan_table 8): a permutation of the pairs inside every chunk
    chan2 = plan.table(r, 8).astype(np.int64).reshape(nb, cpad)
    assert np.array_equal(chan2[:, 1::2], chan2[:, 0::2] + 1) and (chan2[:, 0::2] % 2 == 0).all()
    src = chan2[:, 0::2] // 2                                                        # [nb][slot pair] -> pair
    assert np.array_equal(np.sort(src.reshape(nb, nvc // (cc // 2), cc // 2), axis=2),
                          np.broadcast_to(np.arange(nvc).reshape(nvc // (cc // 2), cc // 2), (nb, nvc // (cc // 2), cc // 2)))
    out = np.zeros((nb, g, 8, cpad), dtype=np.int64)
    anyb = np.zeros((nb, nvc // 4, g), dtype=np.int64)
    assert (e[..., 2:4] == 0).all()
    for q in range(4):
        v = np.arange(q, nvc, 4)                                                    # the slot pairs in position q of their quad
        sv = src[:, v]                                                               # [nb][quad]: the pairs staged there
        prev = None
        for j in range(8):
            off = (e[..., 4 + 4 * q + j // 2] >> (16 * (j % 2))) & 0xFFFF             # [nb][quad][g] byte offset in the stage
            assert (off % 16 == 0).all()
            sw = off // 16
            row, rel = sw // rowsw, sw % rowsw                                       # row inside the stage, superword inside the row
            pbit = row - ((2 * v) % cc)[None, :, None]                               # which pre-summed row: U_0 or U_1
            assert ((pbit == 0) | (pbit == 1)).all()
            assert (rel <= span[:, 2 * v][:, :, None]).all(), "loads stay inside the staged row"
            D = rel + dmin[:, 2 * v][:, :, None]
            if j > 0:
                n = (j - 1) * 4 + q
                chg = (e[..., 0] >> ((n // 7) * 8 + n % 7)) & 1
                assert np.array_equal(chg, (off != prev).astype(np.int64)), "changed bit <=> the offset differs from the previous trial's"
                anyb |= chg << j
            prev = off
            idx = np.broadcast_to(sv[:, None, :], (nb, g, v.size))
            np.put_along_axis(out[:, :, j, :], 2 * idx, D.transpose(0, 2, 1), axis=2)
            np.put_along_axis(out[:, :, j, :], 2 * idx + 1, (D + delta[sv][:, :, None] + pbit).transpose(0, 2, 1), axis=2)
    assert np.array_equal(anyb, e[..., 1]), "any bits are the OR of the quad's changed bits"
    return out.reshape(nb * g * 8, cpad)


@pytest.mark.parametrize("cfg,nchans", [(3, 4096), (3, 4095), (3, 1001), (1, 128)])
def test_pair_tables_reproduce_the_delay_table(cfg, nchans):
    """DD_KERNEL_SUBBAND (NEXT-3): the pair-row tables, decoded independently of the kernel, give back the oracle's
    delay of BOTH channels of every pair for every trial; padded rows follow their partner."""
    w = W.CONFIGS[cfg]
    if nchans != w.nchans:
        w = W.scaled(w, nchans=nchans, nsamps=2 ** 16)
    plan = _host_plan(w)
    plan.set_kernel(B.DD_KERNEL_SUBBAND)
    for r, rg in enumerate(w.ranges):
        pi = plan.pair_info(r)
        if plan.tile_info(r)["mode"] != 2:
            assert pi["enabled"] == 0                       # coarse grids are not delta coded: no pair mode
            continue
        want = oracle.delay_table(w.f_top_mhz, w.chan_width_mhz, w.nchans, w.tsamp_s, rg.decim, rg.dm_lo, rg.dm_step, rg.ndm)
        npair = w.nchans // 2
        diff = want[:, 1:2 * npair:2] - want[:, 0:2 * npair:2]
        valid = bool(((diff.max(axis=0) - diff.min(axis=0)) <= 1).all())   # two neighbouring values per pair over ALL trials
        assert pi["enabled"] == int(valid), (cfg, r)
        if cfg == 3 and nchans >= 4095:
            assert valid                                      # the SPOTLIGHT-shaped beam qualifies in all three ranges
        if not valid:
            continue
        shape = plan.tile_shape(r)
        got = _decode_pairs(plan, r)
        rows = np.minimum(np.arange(got.shape[0]), rg.ndm - 1)
        assert np.array_equal(got[:, : w.nchans], want[rows]), (cfg, r)
        if w.nchans % 2:                                     # the pad partner of the last channel copies its delay
            assert np.array_equal(got[:, w.nchans], want[rows][:, -1])
        rows = shape["chans_per_stage"]
        stage = -(-(rows * pi["row_superwords"] * 16 + rows // 8 * shape["trial_groups"] * 80) // 128) * 128
        assert rows * pi["row_superwords"] * 16 <= 65536 and 128 + 2 * stage + 512 <= 227 * 1024
    brute = plan.work()[1]
    assert plan.executed_adds() < 0.52 * brute if cfg == 3 and nchans == 4096 else plan.executed_adds() <= brute
    plan.set_kernel(B.DD_KERNEL_TILED)
    assert plan.executed_adds() == brute
    plan.destroy()


def test_workspace_is_the_largest_packed_copy_not_their_sum():
    """The ranges are packed and dedispersed one after the other into one scratch (dd_execute), so the workspace is the
    largest packed copy: [nbeams][Cpad][Wp] superwords of 16 bytes, Wp = time tiles x tile + largest delay + 8, rounded
    to 8.  Config 3: 2.2 GB, not the 4.0 GB of three copies side by side; the sub-band variant adds one pair array."""
    w = W.CONFIGS[3]
    plan = _host_plan(w)
    sizes = []
    for r in range(len(w.ranges)):
        info, shape, ri = plan.tile_info(r), plan.tile_shape(r), plan.range_info(r)
        lanes, t = info["lanes"], info["words_per_cta"]
        h = -(-(-(-ri["nout"] // lanes)) // 16) * 16                    # lane segment, multiple of 16 superwords
        ntau = -(-h // t)
        wp = -(-(ntau * t + ri["maxd"] + 8) // 8) * 8
        sizes.append(-(-(shape["cpad"] * wp * 16) // 256) * 256)
    assert plan.workspace_bytes() == max(sizes) and plan.workspace_bytes() < 0.6 * sum(sizes)
    assert 2.0e9 < plan.workspace_bytes() < 2.4e9
    plan.set_kernel(B.DD_KERNEL_SUBBAND)
    assert plan.workspace_bytes() == 2 * max(sizes)                     # + the pair rows of the largest range
    plan.destroy()
