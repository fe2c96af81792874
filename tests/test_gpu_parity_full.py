"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (tiled kernel,
tile shape chosen by the plan), element by element against the oracle (last pin row).

  * config 2: EVERY output element (1001 trials x 126243 samples).
  * configs 3, 4, 5: trials chosen so that every CTA trial block of every range (plan.tile_info "dm_per_cta") is hit
    several times and, over a block's picks, every position of the per-thread register group (8 trials, or 4 on
    byte lanes) and several trial groups of the CTA are covered -- a stride-`_STRIDE` sweep whose phase rotates
    from block to block, plus the first and last trial of each range -- each over its FULL valid span, compared
    bit for bit.  Config 5 on 8 of its 32 beams, first and last included.  DD_TEST_FULL_STRIDE=1 in the
    environment of the test run compares every element of every config (config 3: ~4 minutes of oracle time on
    16 cores).
  * config 4 (uint16; sums above 2^24 are rounded once): the ulp distance of every compared element is
    histogrammed and printed; the stated tolerance is <= 1 ulp (BASELINE.json), the assertion is max = 0.
  * extras that hold at any size, for EVERY trial of every checked beam: the row sum over time,
        sum_t S[j][t] = sum_c ( Y[c][d(c,j) + nout] - Y[c][d(c,j)] ),   Y = prefix sum of y over time,
    in exact integer arithmetic from the oracle's decimated input and delay table against the float64 sum of the
    GPU row (exact for uint8; 1e-7 relative for uint16); DM = 0 equals the plain channel sum; row
    padding untouched; (uint8) the single-pulse search over the whole plane agrees with the oracle's search on the
    oracle's rows for the compared trials.
"""
import os

import numpy as np
import pytest

import oracle
from paper_2605_03531_b200 import workloads as W

gpu = pytest.mark.gpu

_STRIDE = max(1, int(os.environ.get("DD_TEST_FULL_STRIDE", "8")))   # test density only; the library reads no environment
_CHUNK = 48                                                          # trials per oracle call (bounds host memory)


def pick_trials(ndm, dcta, rd, stride):
    """Trials to compare: inside block b the sweep starts at phase (3*b) mod stride, so consecutive blocks hit
    different register positions (j mod rd) and trial groups; first and last trial always included."""
    if stride <= 1:
        return np.arange(ndm, dtype=np.int32)
    sel = {0, ndm - 1}
    nblocks = -(-ndm // dcta)
    for b in range(nblocks):
        j0, j1 = b * dcta, min(ndm, (b + 1) * dcta)
        picks = list(range(j0 + (3 * b) % stride, j1, stride))
        if not picks:                       # a short last block: still take one trial of it
            picks = [j0 + (b % (j1 - j0))]
        sel.update(picks)
    return np.array(sorted(sel), dtype=np.int32)


def test_pick_trials_covers_every_block_and_register_position():
    for ndm, dcta, rd in [(2000, 128, 8), (2801, 128, 8), (4000, 32, 4), (2001, 64, 8), (2001, 32, 4), (101, 16, 4)]:
        sel = pick_trials(ndm, dcta, rd, 8)
        blocks = sel // dcta
        assert set(blocks.tolist()) == set(range(-(-ndm // dcta)))
        assert set((sel % rd).tolist()) == set(range(rd))                       # every register position ...
        full = [b for b in set(blocks.tolist()) if (b + 1) * dcta <= ndm]
        if dcta >= 8 * rd:                                                      # ... and several trial groups per block
            assert all(len(set(((sel[blocks == b] % dcta) // rd).tolist())) >= 4 for b in full)


def _run_full(key, beams_to_check, stride):
    import torch
    from paper_2605_03531_b200 import binding as B

    w = W.CONFIGS[key]
    x = W.generate(w)
    plan = B.Plan.from_workload(w)
    xin = torch.from_numpy(x.view(np.int16) if x.dtype == np.uint16 else x).cuda()
    out = torch.full((plan.out_elems(),), -1.0, dtype=torch.float32, device="cuda")
    plan.execute(xin, out, torch.cuda.current_stream())
    torch.cuda.synchronize()
    del xin
    exact = w.in_bits == 8
    sps_k, sps_thr, sps = 8, 6.0, None
    if exact:   # NEXT-2: single-pulse search over the whole plane, checked on the compared trials below
        nrows = plan.sps_rows()
        sps = [torch.empty((nrows, sps_k), dtype=dt, device="cuda") for dt in (torch.float32, torch.int32, torch.int32)]
        plan.sps_execute(out, sps_k, sps_thr, *sps, torch.cuda.current_stream())
        torch.cuda.synchronize()
        sps = [a.cpu().numpy() for a in sps]
    rows_per_beam = sum(rg.ndm for rg in w.ranges)
    ulp_hist = np.zeros(4, dtype=np.int64)          # ulp distance 0, 1, 2, >= 3
    compared = 0
    for beam in beams_to_check:
        for r, rg in enumerate(w.ranges):
            tab = oracle.delay_table(w.f_top_mhz, w.chan_width_mhz, w.nchans, w.tsamp_s, rg.decim, rg.dm_lo, rg.dm_step, rg.ndm)
            ns_r, maxd, nout = oracle.range_sizes(w.nsamps, rg.decim, tab)
            info, tile = plan.range_info(r), plan.tile_info(r)
            assert (info["ns"], info["maxd"], info["nout"]) == (ns_r, maxd, nout)
            assert plan.tile_shape(r)["tiled"] == 1                      # the configuration bench.py times
            y = oracle.decimate(x[beam], rg.decim)
            view = plan.view_range(out, r, beam)                          # torch view [ndm][nout] on the GPU
            # (1) the chosen trials, full span, bit for bit
            rd = 4 if tile["lanes"] == 16 else 8
            sel_all = pick_trials(rg.ndm, tile["dm_per_cta"], rd, stride)
            for i0 in range(0, len(sel_all), _CHUNK):
                sel = sel_all[i0:i0 + _CHUNK]
                want = oracle.dedisperse(y, tab, sel=sel, t0=0, nt=nout)
                got = view[torch.from_numpy(sel.astype(np.int64)).cuda()].cpu().numpy()
                gi, wi = got.view(np.int32).astype(np.int64), want.view(np.int32).astype(np.int64)   # non-negative floats:
                dist = np.abs(gi - wi)                                                              # ulp distance
                ulp_hist += np.bincount(np.minimum(dist, 3).ravel(), minlength=4)
                compared += dist.size
                if dist.max() != 0:
                    jj, tt = np.unravel_index(int(np.argmax(dist)), dist.shape)
                    raise AssertionError("config %d beam %d range %d trial %d sample %d: got %r want %r (%d ulp); ulp histogram %s"
                                         % (key, beam, r, sel[jj], tt, got[jj, tt], want[jj, tt], dist.max(), ulp_hist.tolist()))
                if sps is not None:   # the oracle's search on the oracle's rows vs the GPU's search on the GPU's plane
                    ref = oracle.sps(want, nout, sps_k, sps_thr)
                    idx = beam * rows_per_beam + sum(q.ndm for q in w.ranges[:r]) + sel
                    assert np.array_equal(sps[0][idx].view(np.uint32), ref["snr"].view(np.uint32)), (key, beam, r)
                    assert np.array_equal(sps[1][idx], ref["tmax"]) and np.array_equal(sps[2][idx], ref["count"]), (key, beam, r)
                del want, got, gi, wi, dist
            # (2) every trial: row sums from prefix sums (exact integers)
            Y = np.zeros((w.nchans, ns_r + 1), dtype=np.uint64)
            np.cumsum(y, axis=1, dtype=np.uint64, out=Y[:, 1:])
            rows = np.arange(w.nchans)
            want_sum = np.empty(rg.ndm, dtype=np.float64)
            for j in range(rg.ndm):
                d = tab[j]
                want_sum[j] = float((Y[rows, d + nout] - Y[rows, d]).sum())
            got_sum = view.sum(dim=1, dtype=torch.float64).cpu().numpy()
            if exact:
                assert np.array_equal(got_sum, want_sum), (key, beam, r, int(np.argmax(got_sum != want_sum)))
            else:
                assert np.allclose(got_sum, want_sum, rtol=1e-7, atol=0), (key, beam, r)
            # (3) DM = 0
            if r == 0 and rg.dm_lo == 0.0:
                plain = y.sum(axis=0, dtype=np.uint64)[:nout]
                assert np.array_equal(view[0].cpu().numpy(), plain.astype(np.float64).astype(np.float32))
            # row padding untouched
            flat = out[beam * plan.beam_stride() + info["offset"]: beam * plan.beam_stride() + info["offset"] + info["ndm"] * info["pitch"]]
            pad = flat.reshape(info["ndm"], info["pitch"])[:, info["nout"]:]
            assert bool((pad == -1.0).all())
            del y, Y
    plan.destroy()
    print("\nconfig %d: %d output elements compared with the oracle (stride %d over trials, full span); ulp distance histogram "
          "[0, 1, 2, >=3] = %s" % (key, compared, stride, ulp_hist.tolist()))
    assert ulp_hist[1:].sum() == 0
    return compared


@gpu
def test_full_cfg2_1024ch_every_element():
    n = _run_full(2, [0], 1)
    assert n == 1001 * 126243


@gpu
def test_full_cfg3_spotlight_4096ch():
    _run_full(3, [0], _STRIDE)


@gpu
def test_full_cfg4_uint16_ulp_histogram():
    _run_full(4, [0], _STRIDE)


@gpu
def test_full_cfg5_32beams():
    _run_full(5, [0, 4, 9, 13, 18, 22, 27, 31], max(_STRIDE, 1) * (1 if _STRIDE == 1 else 2))


@gpu
def test_full_cfg3_subband_variant_equals_default_everywhere():
    """NEXT-3 at full size: the two-channel sub-band variant (half the brute-force adds) writes the same bits as the
    default kernel for EVERY element of the config-3 plane (the default is compared with the oracle above)."""
    import torch
    from paper_2605_03531_b200 import binding as B

    w = W.CONFIGS[3]
    x = torch.from_numpy(W.generate(w)).cuda()
    plan = B.Plan.from_workload(w)
    a = torch.full((plan.out_elems(),), -1.0, dtype=torch.float32, device="cuda")
    plan.execute(x, a, torch.cuda.current_stream())
    plan.set_kernel(B.DD_KERNEL_SUBBAND)
    assert all(plan.pair_info(r)["enabled"] == 1 for r in range(3))
    assert plan.executed_adds() < 0.51 * plan.work()[1]
    b = torch.full((plan.out_elems(),), -1.0, dtype=torch.float32, device="cuda")
    plan.execute(x, b, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert bool(torch.equal(a.view(torch.int32), b.view(torch.int32)))
    plan.destroy()
