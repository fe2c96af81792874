"""GPU parity of the boxcar single-pulse search (dd_sps_execute) against oracle/oracle_sps.c.
The oracle's input is the ORACLE's own DM-time plane, never the GPU's; both must agree bit for bit (float snr
included: the few double operations per row are done in the same order with round-to-nearest on both sides)."""
import numpy as np
import pytest

import oracle
from paper_2605_03531_b200 import workloads as W

from _util import gpu_run, oracle_full

pytestmark = pytest.mark.gpu


def _sps_both(w, x, K, thr):
    import torch
    plan, flat = gpu_run(w, x, 2)
    rows = plan.sps_rows()
    plane = torch.from_numpy(flat).cuda()
    snr = torch.full((rows, K), -7.0, dtype=torch.float32, device="cuda")
    tmax = torch.full((rows, K), -7, dtype=torch.int32, device="cuda")
    cnt = torch.full((rows, K), -7, dtype=torch.int32, device="cuda")
    plan.sps_execute(plane, K, thr, snr, tmax, cnt, torch.cuda.current_stream())
    torch.cuda.synchronize()
    got = {"snr": snr.cpu().numpy(), "tmax": tmax.cpu().numpy(), "count": cnt.cpu().numpy()}
    want_planes = oracle_full(w, x)
    ref = {"snr": [], "tmax": [], "count": []}
    for b in range(w.nbeams):
        for r in range(len(w.ranges)):
            res = oracle.sps(np.ascontiguousarray(want_planes[b][r]), want_planes[b][r].shape[1], K, thr)
            for k in ref:
                ref[k].append(res[k])
    ref = {k: np.concatenate(v, axis=0) for k, v in ref.items()}
    return plan, got, ref


@pytest.mark.parametrize("K,thr", [(1, 3.0), (6, 5.0), (12, 2.5)])
def test_sps_matches_oracle_multirange(K, thr):
    w = W.scaled(W.CONFIGS[3], nchans=96, nsamps=2 ** 14 + 37, nbeams=2,
                 ranges=[W.DMRange(0.0, 0.1, 37, 1), W.DMRange(40.0, 3.0, 21, 1), W.DMRange(600.0, 0.5, 19, 4)])
    x = W.generate(w)
    x[0, :, 6000:6012] = np.minimum(x[0, :, 6000:6012].astype(np.int32) + 9, 255).astype(np.uint8)   # a DM-0 pulse
    plan, got, ref = _sps_both(w, x, K, thr)
    assert got["tmax"].shape == (2 * (37 + 21 + 19), K)
    for k in ("tmax", "count"):
        assert np.array_equal(got[k], ref[k]), k
    assert np.array_equal(got["snr"].view(np.uint32), ref["snr"].view(np.uint32))
    # the injected pulse is found at DM 0 by a filter of about its width
    assert ref["snr"][0].max() > 6 and abs(int(ref["tmax"][0, np.argmax(ref["snr"][0])]) - 6000) <= 16


def test_sps_short_rows_constant_rows_and_wide_filters():
    """Rows shorter than the widest filters and than one tile; a constant plane (sigma = 0)."""
    nch = 8
    w = W.Workload("spsedge", 500.0, -200.0 / nch, nch, 1.024e-3, 700, 1, 8, (W.DMRange(0.0, 1.0, 5, 1), W.DMRange(0.0, 1.0, 3, 4)), 1, 0, 0)
    x = np.full((1, nch, 700), 100, dtype=np.uint8)
    plan, got, ref = _sps_both(w, x, 12, 1.0)
    for k in ("tmax", "count"):
        assert np.array_equal(got[k], ref[k]), k
    assert (got["snr"] == 0).all() and (got["tmax"][:, -1] == -1).all()
    x = np.random.default_rng(3).integers(0, 256, size=(1, nch, 700), dtype=np.uint8)
    plan, got, ref = _sps_both(w, x, 12, -50.0)
    for k in ("tmax", "count"):
        assert np.array_equal(got[k], ref[k]), k
    assert np.array_equal(got["snr"].view(np.uint32), ref["snr"].view(np.uint32))


def test_sps_rejects_inexact_sums_and_bad_arguments():
    import torch
    from paper_2605_03531_b200 import binding as B
    plan = B.Plan(500.0, -200.0 / 4096, 4096, 1.31072e-3, 2 ** 18, [(0.0, 1.0, 2, 1)], in_bits=16)   # (4096*65535)^2 * n > 2^63
    buf = torch.zeros(16, device="cuda")
    with pytest.raises(B.DDError) as e:
        plan.sps_execute(buf, 4, 5.0, buf, buf, buf)
    assert e.value.code == B.DD_ERR_OVERFLOW
    plan8 = B.Plan(500.0, -200.0 / 16, 16, 1e-3, 4096, [(0.0, 1.0, 2, 1)])
    for K, thr in ((0, 1.0), (13, 1.0), (4, float("nan")), (4, float("inf"))):
        with pytest.raises(B.DDError) as e:
            plan8.sps_execute(buf, K, thr, buf, buf, buf)
        assert e.value.code == B.DD_ERR_INVALID


def test_sps_all_zero_rows_and_long_rows():
    """An all-zero filterbank (every boxcar 0: the first window is the tied best) and rows spanning many tiles
    with a late, narrow peak."""
    nch = 4
    w = W.Workload("spszero", 500.0, -200.0 / nch, nch, 1.024e-3, 40000, 1, 8, (W.DMRange(0.0, 1.0, 3, 1),), 1, 0, 0)
    x = np.zeros((1, nch, 40000), dtype=np.uint8)
    plan, got, ref = _sps_both(w, x, 10, 2.0)
    for k in ("tmax", "count"):
        assert np.array_equal(got[k], ref[k]), k
    assert (got["tmax"] == 0).all() and (got["snr"] == 0).all()
    x[0, :, 39000:39003] = 200
    x[0, 0, 100] = 1
    plan, got, ref = _sps_both(w, x, 10, 2.0)
    for k in ("tmax", "count"):
        assert np.array_equal(got[k], ref[k]), k
    assert np.array_equal(got["snr"].view(np.uint32), ref["snr"].view(np.uint32))


# ---- the candidate list (dd_sps_candidates) and the row statistics of the dedispersion epilogue -------------------------
def _candidates_gpu(plan, plane, K, thr, cnt, max_cands):
    import torch
    rows = plan.sps_rows()
    offsets = torch.full((rows * K + 1,), -1, dtype=torch.int64, device="cuda")
    cand = torch.full((max(1, max_cands), 4), -1, dtype=torch.int32, device="cuda")
    plan.sps_candidates(plane, K, thr, cnt, offsets, cand, max_cands, torch.cuda.current_stream())
    torch.cuda.synchronize()
    return offsets.cpu().numpy(), cand.cpu().numpy()


def _oracle_candidates(want_planes, w, K, thr):
    """The oracle's list over the oracle's planes, rows renumbered as in dd_sps_rows (beam-major, ranges in order)."""
    out, row0 = [], 0
    for b in range(w.nbeams):
        for r in range(len(w.ranges)):
            pl = np.ascontiguousarray(want_planes[b][r])
            cand, total = oracle.sps_candidates(pl, pl.shape[1], K, thr, cap=1 << 22)
            assert total == len(cand)
            c = cand.copy()
            c["row"] += row0
            out.append(c)
            row0 += pl.shape[0]
    return np.concatenate(out)


@pytest.mark.parametrize("K,thr,stats", [(6, 4.0, False), (6, 4.0, True), (12, 3.0, False), (3, -1.0, True)])
def test_candidate_list_matches_oracle(K, thr, stats):
    """Every (row, k, t, snr) above the threshold, in the order row, k, t -- bit for bit, with the row statistics
    either recomputed by the search (two reads of the plane) or taken from the dedispersion epilogue (one read)."""
    import torch
    from paper_2605_03531_b200 import binding as B
    w = W.scaled(W.CONFIGS[3], nchans=64, nsamps=2 ** 13 + 123, nbeams=2,
                 ranges=[W.DMRange(0.0, 0.2, 21, 1), W.DMRange(40.0, 3.0, 9, 2), W.DMRange(600.0, 2.0, 7, 4)])
    x = W.generate(w)
    x[0, :, 3000:3006] = np.minimum(x[0, :, 3000:3006].astype(np.int32) + 25, 255).astype(np.uint8)
    x[1, :, 7000:7100] = np.minimum(x[1, :, 7000:7100].astype(np.int32) + 6, 255).astype(np.uint8)
    plan = B.Plan.from_workload(w)
    rows = plan.sps_rows()
    out = torch.zeros(plan.out_elems(), dtype=torch.float32, device="cuda")
    st = None
    if stats:
        st = torch.full((rows, 2), -1, dtype=torch.int64, device="cuda")
        plan.set_row_stats(st)
    plan.execute(torch.from_numpy(x).cuda(), out, torch.cuda.current_stream())
    snr = torch.empty((rows, K), dtype=torch.float32, device="cuda")
    tmax = torch.empty((rows, K), dtype=torch.int32, device="cuda")
    cnt = torch.empty((rows, K), dtype=torch.int32, device="cuda")
    plan.sps_execute(out, K, thr, snr, tmax, cnt, torch.cuda.current_stream())
    want_planes = oracle_full(w, x)
    want = _oracle_candidates(want_planes, w, K, thr)
    assert len(want) > 50
    offsets, cand = _candidates_gpu(plan, out, K, thr, cnt, len(want) + 10)
    counts = cnt.cpu().numpy().ravel()
    assert offsets[0] == 0 and offsets[-1] == len(want) and np.array_equal(np.diff(offsets), counts)
    got = cand[: len(want)]
    assert np.array_equal(got[:, 0], want["row"]) and np.array_equal(got[:, 1], want["k"]) and np.array_equal(got[:, 2], want["t"])
    assert np.array_equal(got[:, 3].view(np.uint32), want["snr"].view(np.uint32))
    assert (cand[len(want):] == -1).all()                              # nothing written past the list
    if stats:   # the epilogue's sums are the exact row sums
        sth = st.cpu().numpy()
        row = 0
        for b in range(w.nbeams):
            for r in range(len(w.ranges)):
                pl = want_planes[b][r].astype(np.float64)
                assert np.array_equal(sth[row: row + pl.shape[0], 0], pl.sum(axis=1).astype(np.int64))
                assert np.array_equal(sth[row: row + pl.shape[0], 1], (pl * pl).sum(axis=1).astype(np.int64))
                row += pl.shape[0]
        # and the search gives the same results with and without them
        plan.set_row_stats(None)
        snr2, tmax2, cnt2 = torch.empty_like(snr), torch.empty_like(tmax), torch.empty_like(cnt)
        plan.sps_execute(out, K, thr, snr2, tmax2, cnt2, torch.cuda.current_stream())
        torch.cuda.synchronize()
        assert torch.equal(snr.view(torch.int32), snr2.view(torch.int32)) and torch.equal(tmax, tmax2) and torch.equal(cnt, cnt2)
    # a capacity below the total: the first entries, and the total still reported
    offsets2, few = _candidates_gpu(plan, out, K, thr, cnt, 17)
    assert offsets2[-1] == len(want) and np.array_equal(few[:17], cand[:17])
    plan.destroy()


def test_row_stats_with_the_direct_kernel_and_subband_variant():
    import torch
    from paper_2605_03531_b200 import binding as B
    w = W.Workload("stats", 600.0, -200.0 / 4096, 96, 1.31072e-3, 2 ** 13, 1, 8,
                   (W.DMRange(0.0, 0.3, 40, 1), W.DMRange(300.0, 0.9, 24, 2)), 5, 128, 12)
    x = W.generate(w)
    want_planes = oracle_full(w, x)
    for variant in (B.DD_KERNEL_DIRECT, B.DD_KERNEL_TILED, B.DD_KERNEL_SUBBAND):
        plan = B.Plan.from_workload(w)
        plan.set_kernel(variant)
        st = torch.full((plan.sps_rows(), 2), -1, dtype=torch.int64, device="cuda")
        plan.set_row_stats(st)
        out = torch.zeros(plan.out_elems(), dtype=torch.float32, device="cuda")
        for _ in range(2):                                             # twice: the sums are zeroed by every execute
            plan.execute(torch.from_numpy(x).cuda(), out, torch.cuda.current_stream())
        torch.cuda.synchronize()
        sth, row = st.cpu().numpy(), 0
        for r in range(2):
            pl = want_planes[0][r].astype(np.float64)
            assert np.array_equal(sth[row: row + pl.shape[0], 0], pl.sum(axis=1).astype(np.int64)), variant
            assert np.array_equal(sth[row: row + pl.shape[0], 1], (pl * pl).sum(axis=1).astype(np.int64)), variant
            row += pl.shape[0]
        plan.destroy()
    p16 = B.Plan(500.0, -1.0, 16, 1e-3, 4096, [(0.0, 1.0, 2, 1)], in_bits=16)
    with pytest.raises(B.DDError):
        p16.set_row_stats(st)


# ---- last on purpose: written after GPU access had closed, so a failure here hides no other test ----
def _check_all(got, ref):
    for k in ("tmax", "count"):
        assert np.array_equal(got[k], ref[k]), k
    assert np.array_equal(got["snr"].view(np.uint32), ref["snr"].view(np.uint32))


@pytest.mark.parametrize("K", [1, 4, 8, 9])
def test_sps_barrier_free_kernel_edge_cases(K):
    """Up to 9 widths and 32-bit sums run in dd_sps_warp_kernel (every warp filters tiles of its own; records per warp and
    tile; all ranges in one launch): rows shorter than one warp tile and than the widest filter, constant and all-zero rows
    (every window ties: the first one wins, across warps and tiles), equal maxima far apart, a late narrow peak in a long
    row, a threshold below everything (every window counted), two beams, and more ranges than one launch takes."""
    nch = 8
    # short rows, constant plane (sigma = 0), then random data with a threshold that counts every window
    w = W.Workload("spsw_short", 500.0, -200.0 / nch, nch, 1.024e-3, 700, 2, 8,
                   (W.DMRange(0.0, 1.0, 5, 1), W.DMRange(0.0, 1.0, 3, 4)), 1, 0, 0)
    x = np.full((2, nch, 700), 100, dtype=np.uint8)
    plan, got, ref = _sps_both(w, x, K, 1.0)
    _check_all(got, ref)
    assert (got["snr"] == 0).all()
    x = np.random.default_rng(30 + K).integers(0, 256, size=(2, nch, 700), dtype=np.uint8)
    plan, got, ref = _sps_both(w, x, K, -50.0)
    _check_all(got, ref)
    # long rows (40 warp tiles): all zero; then equal maxima in different tiles and warps plus a late narrow peak
    nch = 4
    w = W.Workload("spsw_long", 500.0, -200.0 / nch, nch, 1.024e-3, 41000, 1, 8, (W.DMRange(0.0, 1.0, 3, 1),), 1, 0, 0)
    x = np.zeros((1, nch, 41000), dtype=np.uint8)
    plan, got, ref = _sps_both(w, x, K, 2.0)
    _check_all(got, ref)
    assert (got["tmax"] == 0).all() and (got["snr"] == 0).all()
    for t0 in (5000, 1030, 20500, 33333):            # the same pulse four times: the earliest position is reported
        x[0, :, t0:t0 + 3] = 90
    plan, got, ref = _sps_both(w, x, K, 2.0)
    _check_all(got, ref)
    x[0, :, 40960:40962] = 250                        # a stronger one a few samples before the end of the row (its tail loop)
    x[0, 0, 100] = 1
    plan, got, ref = _sps_both(w, x, K, 2.0)
    _check_all(got, ref)
    # eleven ranges of different row lengths (two launches of the merged kernel), noise with pulses
    rgs = tuple(W.DMRange(10.0 * i, 1.0 + 0.3 * i, 3 + i % 4, (1, 2, 4, 8)[i % 4]) for i in range(11))
    w = W.Workload("spsw_many", 700.0, -300.0 / 16, 16, 1.024e-3, 9000, 1, 8, rgs, 1, 0, 0)
    x = np.random.default_rng(77).integers(100, 140, size=(1, 16, 9000), dtype=np.uint8)
    x[0, :, 4000:4006] += 60
    plan, got, ref = _sps_both(w, x, K, 4.0)
    _check_all(got, ref)
