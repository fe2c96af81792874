"""Pins of the single-pulse-search oracle (oracle/oracle_sps.c, PAPER.md:317-325:
"statistically significant single pulses above a user-specified threshold using time-domain boxcar filtering").
Closed forms, limits and a brute force that do not go through the oracle's own code.  No GPU needed."""
import math

import numpy as np
import pytest

import oracle


def _row(vals):
    return np.asarray(vals, dtype=np.float32)[None, :]


def test_constant_row_has_no_significance():
    """x = v everywhere: sigma = 0 -> snr 0, the first window is the (tied) best, nothing above the mean."""
    res = oracle.sps(_row([37] * 500), 500, 6, 3.0)
    assert res["mean"][0] == 37.0 and res["sigma"][0] == 0.0
    assert (res["snr"] == 0).all() and (res["tmax"] == 0).all() and (res["count"] == 0).all()


def test_single_impulse_closed_form():
    """One sample of height h at t0 on a zero row of n samples: mean = h/n, var = h^2/n - h^2/n^2; every width
    peaks at the first window that contains t0 with B = h."""
    n, h, t0, K = 4096, 200.0, 1234, 8
    x = np.zeros(n, dtype=np.float32)
    x[t0] = h
    res = oracle.sps(x[None, :], n, K, 5.0)
    mean, sigma = h / n, math.sqrt(h * h / n - (h / n) ** 2)
    assert res["mean"][0] == mean and abs(res["sigma"][0] - sigma) < 1e-12
    for k in range(K):
        w = 2 ** k
        assert res["tmax"][0, k] == t0 - w + 1
        want = (h - w * mean) / (sigma * math.sqrt(w))
        assert abs(res["snr"][0, k] - want) <= 1e-6 * want
        # windows containing the impulse: w of them, each with B = h; above threshold iff snr > 5
        assert res["count"][0, k] == (w if want > 5.0 else 0)
    assert np.argmax(res["snr"][0]) == 0          # an unresolved impulse is best matched by width 1


def test_boxcar_pulse_is_best_matched_by_its_own_width():
    """A boxcar of width 8 (PAPER.md:387-393 injects such pulses): the width-8 filter has the largest snr,
    snr_w / snr_8 = sqrt(w/8) for w < 8 and sqrt(8/w) for w > 8 up to the mean term."""
    n, h, t0 = 1 << 14, 30.0, 5000
    x = np.zeros(n, dtype=np.float32)
    x[t0:t0 + 8] = h
    res = oracle.sps(x[None, :], n, 7, 4.0)
    snr = res["snr"][0]
    assert np.argmax(snr) == 3 and res["tmax"][0, 3] == t0
    for k in range(7):
        w = 2 ** k
        ratio = math.sqrt(w / 8) if w <= 8 else math.sqrt(8 / w)
        assert abs(snr[k] / snr[3] - ratio) < 2e-3
        assert res["tmax"][0, k] == (t0 if w <= 8 else t0 + 8 - w)   # first window with the largest overlap


def test_ramp_mean_and_variance():
    """x[t] = t: mean (n-1)/2, population variance (n^2-1)/12; the best window of every width is the last."""
    n, K = 1000, 5
    res = oracle.sps(_row(np.arange(n)), n, K, 0.0)
    assert res["mean"][0] == (n - 1) / 2 and abs(res["sigma"][0] - math.sqrt((n * n - 1) / 12)) < 1e-9
    for k in range(K):
        w = 2 ** k
        assert res["tmax"][0, k] == n - w
        # B[t] = w*t + w(w-1)/2 > w*mean  <=>  t > mean - (w-1)/2
        assert res["count"][0, k] == n - w + 1 - (math.floor((n - 1) / 2 - (w - 1) / 2) + 1)


def test_threshold_limits_and_wide_filters():
    rng = np.random.default_rng(1)
    n = 300
    x = rng.integers(0, 1000, n).astype(np.float32)
    lo = oracle.sps(x[None, :], n, 10, -1e9)
    hi = oracle.sps(x[None, :], n, 10, 1e9)
    for k in range(10):
        w = 2 ** k
        if w <= n:
            assert lo["count"][0, k] == n - w + 1 and hi["count"][0, k] == 0
        else:                                   # filter wider than the row: no window
            assert lo["count"][0, k] == 0 and lo["tmax"][0, k] == -1 and lo["snr"][0, k] == 0


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_brute_force_on_random_rows(seed):
    """Pure-Python double loop, Python floats (IEEE double) in the oracle's stated operation order."""
    rng = np.random.default_rng(seed)
    n, K, thr = 97, 6, 1.5
    rows = rng.integers(0, 5000, size=(3, 128)).astype(np.float32)
    rows[1, 40:44] += 20000
    res = oracle.sps(rows, n, K, thr)
    for r in range(3):
        x = [int(v) for v in rows[r, :n]]
        mean = sum(x) / n
        var = sum(v * v for v in x) / n - mean * mean
        sigma = math.sqrt(max(var, 0.0))
        for k in range(K):
            w = 2 ** k
            sums = [sum(x[t:t + w]) for t in range(n - w + 1)]
            best = max(sums)
            den = sigma * math.sqrt(w)
            assert res["tmax"][r, k] == sums.index(best)
            assert res["snr"][r, k] == np.float32((best - w * mean) / den)
            assert res["count"][r, k] == sum(1 for b in sums if b > w * mean + thr * den)


def test_offset_invariance_of_position_and_near_invariance_of_snr():
    """Adding a constant to the row moves the mean, not the peaks."""
    rng = np.random.default_rng(9)
    n = 2000
    x = rng.integers(0, 300, n).astype(np.float32)
    x[700:716] += 400
    a = oracle.sps(x[None, :], n, 8, 3.0)
    b = oracle.sps((x + 1000)[None, :], n, 8, 3.0)
    assert np.array_equal(a["tmax"], b["tmax"]) and np.array_equal(a["count"], b["count"])
    assert np.allclose(a["snr"], b["snr"], rtol=1e-5)


# ---- the candidate list ("The list of candidates thus generated is filtered ...") ---------------------
def test_candidate_list_single_impulse_closed_form():
    """One impulse of height h at t0 over a constant level c: for width w the windows that contain it are
    t0-w+1 .. t0, each with B = w*c + h and snr = (B - w*mean)/(sigma*sqrt(w)); they are the only candidates and come
    in the order (row, width index, t)."""
    n, c, h, t0, K, thr = 2000, 50.0, 400.0, 700, 6, 4.0
    x = np.full(n, c, dtype=np.float32)
    x[t0] += h
    mean = (n * c + h) / n
    sigma = math.sqrt((((n - 1) * c * c + (c + h) ** 2) / n) - mean * mean)
    cand, total = oracle.sps_candidates(x[None, :], n, K, thr)
    want = []
    for k in range(K):
        w = 2 ** k
        snr = (w * c + h - w * mean) / (sigma * math.sqrt(w))
        if snr > thr:
            want += [(0, k, t, snr) for t in range(t0 - w + 1, t0 + 1)]
    assert total == len(want) == len(cand) and total > 0
    assert [(int(a["row"]), int(a["k"]), int(a["t"])) for a in cand] == [(r, k, t) for r, k, t, _ in want]
    assert np.allclose(cand["snr"], [s for *_, s in want], rtol=1e-6, atol=0)


def test_candidate_list_agrees_with_counts_order_and_brute_force():
    rng = np.random.default_rng(99)
    rows = rng.integers(900, 1100, size=(5, 700)).astype(np.float32)
    rows[1, 100:108] += 300.0
    rows[3, 650:700] += 120.0
    rows[4, :] = 1000.0                      # sigma = 0: nothing can exceed the mean
    K, thr = 7, 3.5
    res = oracle.sps(rows, 700, K, thr)
    cand, total = oracle.sps_candidates(rows, 700, K, thr)
    assert total == len(cand) == int(res["count"].sum()) and total > 20
    key = cand["row"].astype(np.int64) * 10 ** 9 + cand["k"].astype(np.int64) * 10 ** 6 + cand["t"]
    assert (np.diff(key) > 0).all()          # strictly increasing in (row, k, t)
    for r in range(5):                       # count per (row, k) == list length per (row, k)
        for k in range(K):
            assert int(((cand["row"] == r) & (cand["k"] == k)).sum()) == res["count"][r, k]
    # brute force in Python doubles: same membership, snr compared as float32 bits
    for r in (1, 3):
        x = [float(v) for v in rows[r]]
        n = len(x)
        mean = sum(x) / n
        var = sum(v * v for v in x) / n - mean * mean
        sigma = math.sqrt(max(var, 0.0))
        mine = []
        for k in range(K):
            w = 2 ** k
            den = sigma * math.sqrt(w)
            for t in range(n - w + 1):
                b = sum(x[t:t + w])
                if b > w * mean + thr * den:
                    mine.append((k, t, np.float32((b - w * mean) / den)))
        got = cand[cand["row"] == r]
        assert [(int(a["k"]), int(a["t"])) for a in got] == [(k, t) for k, t, _ in mine]
        assert np.array_equal(got["snr"].view(np.uint32), np.array([s for *_, s in mine], dtype=np.float32).view(np.uint32))
    # the best candidate of a (row, k) is the snr / tmax the search reports
    for r, k in ((1, 3), (3, 5)):
        sel = cand[(cand["row"] == r) & (cand["k"] == k)]
        assert sel["snr"].max() == res["snr"][r, k] and int(sel["t"][np.argmax(sel["snr"])]) == res["tmax"][r, k]
    # a capacity below the total truncates the list but still reports the total
    few, total2 = oracle.sps_candidates(rows, 700, K, thr, cap=10)
    assert total2 == total and len(few) == 10 and np.array_equal(few, cand[:10])
