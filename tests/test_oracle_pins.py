"""Pins for the CPU oracle (oracle/oracle_dedisp.c) against what the paper and the mathematics fix.

No GPU, no CUDA path.  Each test names the pin of SURVEY.md section 8(c) it implements and the
oracle step a mistake there would break:
  P1 hand-worked Eq. 1.1 values (tests/golden/delay_hand_values.txt)  -> constant, units, f^-2, /tsamp*decim, rounding
  P2 structure of the delay table                                      -> indexing [trial][chan], sign, monotonicity
  P3 DM=0 row = plain channel sum                        -> the sum itself
  P4 impulse along the sweep peaks at nchans*height at its DM           -> sign of the shift (t + d), trial/channel indexing
  P5 linearity                                                          -> no hidden normalisation
  P6 constant input -> nchans*decim*v                                   -> "sum, not mean"; nout
  P7 time-shift covariance                                              -> edges/valid span
  P8 single channel identity                                            -> delay of channel 0 is 0
  P9 decimation reduction                                               -> O6 feeds O7 with tsamp*decim
  P10 pure-Python brute force with hand-derived delays                  -> everything, end to end
  P11 exactness bounds of the five configs                              -> bit-exact parity bar is justified
  P12 zeroed channels = dedispersion over the remaining subset          -> channel loop covers all rows
"""
import os

import numpy as np
import pytest

import oracle
from paper_2605_03531_b200 import workloads as W


def _read_golden(path):
    rows = []
    with open(path) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if line:
                f_top, f_c, tsamp, decim, dm, d = line.split()
                rows.append((float(f_top), float(f_c), float(tsamp), int(decim), float(dm), int(d)))
    return rows


# ---------------------------------------------------------------- P1
def test_p1_hand_worked_delays(golden_dir):
    rows = _read_golden(os.path.join(golden_dir, "delay_hand_values.txt"))
    assert len(rows) >= 20
    for f_top, f_c, tsamp, decim, dm, want in rows:
        if f_c == f_top:
            # channel 0 of any band
            tab = oracle.delay_table(f_top, -1.0, 4, tsamp, decim, dm, 0.0, 1)
            assert tab[0, 0] == want
            continue
        # two-channel band whose second channel is f_c; dm placed at trial index 3 of a 4-trial range
        step = dm / 3.0
        tab = oracle.delay_table(f_top, f_c - f_top, 2, tsamp, decim, 0.0, step, 4)
        assert tab.shape == (4, 2)
        assert tab[3, 1] == want, (f_top, f_c, tsamp, decim, dm, int(tab[3, 1]), want)
        assert tab[3, 0] == 0
        # the same value through dm_lo instead of the step
        tab2 = oracle.delay_table(f_top, f_c - f_top, 2, tsamp, decim, dm, 1.0, 1)
        assert tab2[0, 1] == want


def test_p1_survey_cross_values():
    """Values listed in SURVEY.md section 8(c) P1 for the BASELINE configs (derived there in numpy;
    kept as a cross-check that sizes of the five configs match the scope table)."""
    want_maxd = {1: [2835], 2: [4829], 3: [966, 1450, 2417], 4: [22492, 8436], 5: [4833]}
    want_nout = {1: [5357], 2: [126243], 3: [261178, 129622, 63119], 4: [239652, 24332], 5: [60703]}
    for k, w in W.CONFIGS.items():
        for r, rg in enumerate(w.ranges):
            last = oracle.delay_table(w.f_top_mhz, w.chan_width_mhz, w.nchans, w.tsamp_s, rg.decim,
                                      rg.dm_lo + (rg.ndm - 1) * rg.dm_step, 0.0, 1)
            ns_r, maxd, nout = oracle.range_sizes(w.nsamps, rg.decim, last)
            assert maxd == want_maxd[k][r]
            assert nout == want_nout[k][r]
    c1 = W.CONFIGS[1]
    tab = oracle.delay_table(c1.f_top_mhz, c1.chan_width_mhz, c1.nchans, c1.tsamp_s, 1, 0.0, 1.0, 101)
    assert tab[50, 127] == 1417 and tab[100, 127] == 2835 and tab[50, 64] == 456 and tab[100, 1] == 10


# ---------------------------------------------------------------- P2
@pytest.mark.parametrize("decim", [1, 2, 4, 8])
def test_p2_delay_table_structure(decim):
    nch, ndm = 64, 40
    tab = oracle.delay_table(750.0, -200.0 / nch, nch, 1.31072e-3, decim, 0.0, 2.5, ndm)
    assert tab.dtype == np.int64 and tab.shape == (ndm, nch)
    assert (tab[:, 0] == 0).all()              # reference channel
    assert (tab[0, :] == 0).all()              # DM = 0
    assert (np.diff(tab, axis=1) >= 0).all()   # lower frequency -> later
    assert (np.diff(tab, axis=0) >= 0).all()   # larger DM -> later
    assert tab[-1, -1] > 0
    # decimation by k divides the unrounded delay by k: |k*d_k - d_1| <= k/2 + 1/2
    tab1 = oracle.delay_table(750.0, -200.0 / nch, nch, 1.31072e-3, 1, 0.0, 2.5, ndm)
    assert (np.abs(decim * tab - tab1) <= decim / 2 + 0.5).all()
    # freqs
    f = oracle.channel_freqs(750.0, -200.0 / nch, nch)
    assert f[0] == 750.0 and abs(f[-1] - (750.0 - 200.0 * (nch - 1) / nch)) < 1e-9


def test_p2_delay_scales_linearly_with_dm_and_inverse_tsamp():
    a = oracle.delay_table(600.0, -300.0, 2, 1e-4, 1, 0.0, 10.0, 11)[:, 1].astype(float)
    # unrounded x is linear in DM: second differences of the rounded table are at most 2
    assert np.abs(np.diff(a, 2)).max() <= 2
    b = oracle.delay_table(600.0, -300.0, 2, 2e-4, 1, 0.0, 10.0, 11)[:, 1].astype(float)
    assert np.abs(a - 2 * b).max() <= 1.5


def test_invalid_arguments_rejected():
    with pytest.raises(ValueError):
        oracle.delay_table(500.0, +1.0, 4, 1e-3, 1, 0.0, 1.0, 2)   # ascending band rejected (reading A3)
    with pytest.raises(ValueError):
        oracle.delay_table(500.0, -1.0, 4, 1e-3, 3, 0.0, 1.0, 2)   # decim must be 1,2,4,8
    with pytest.raises(ValueError):
        oracle.delay_table(500.0, -1.0, 4, 0.0, 1, 0.0, 1.0, 2)
    y = np.ones((2, 16), dtype=np.uint32)
    d = np.array([[0, 10]], dtype=np.int64)
    with pytest.raises(ValueError):
        oracle.dedisperse(y, d, t0=0, nt=7)                         # 7 + 10 > 16: outside the valid span
    assert oracle.dedisperse(y, d, t0=0, nt=6).shape == (1, 6)


# ---------------------------------------------------------------- helpers
def _small(seed=7, nch=24, ns=1500, bits=8):
    rng = np.random.default_rng(seed)
    x = rng.integers(0, 2 ** bits, size=(nch, ns), dtype=np.uint8 if bits == 8 else np.uint16)
    tab = oracle.delay_table(500.0, -200.0 / nch, nch, 1.024e-3, 1, 0.0, 1.5, 20)
    return x, tab


# ---------------------------------------------------------------- P3
def test_p3_dm0_is_plain_channel_sum():
    x, tab = _small()
    out = oracle.dedisperse(oracle.decimate(x, 1), tab)
    nout = x.shape[1] - int(tab.max())
    assert out.shape == (20, nout)
    want = x.astype(np.uint64).sum(axis=0)[:nout]
    assert (out[0].astype(np.uint64) == want).all()
    assert not (out[5].astype(np.uint64) == want).all()


# ---------------------------------------------------------------- P4
@pytest.mark.parametrize("jstar", [3, 11, 19])
def test_p4_impulse_peaks_at_its_dm(jstar):
    nch, ns, h, t0 = 32, 1500, 7, 123
    tab = oracle.delay_table(500.0, -200.0 / nch, nch, 1.024e-3, 1, 0.0, 2.0, 20)
    x = np.zeros((nch, ns), dtype=np.uint8)
    for c in range(nch):
        x[c, t0 + tab[jstar, c]] = h
    out = oracle.dedisperse(oracle.decimate(x, 1), tab)
    assert out[jstar, t0] == nch * h
    j, t = np.unravel_index(np.argmax(out), out.shape)
    assert (j, t) == (jstar, t0)
    assert (out == nch * h).sum() == 1          # unique maximum: the bow-tie of PAPER.md:363
    assert out.max() == nch * h and out.sum() <= nch * h * out.shape[0]


# ---------------------------------------------------------------- P5
def test_p5_linearity():
    rng = np.random.default_rng(3)
    nch, ns = 16, 1000
    tab = oracle.delay_table(500.0, -200.0 / nch, nch, 1.024e-3, 1, 0.0, 3.0, 9)
    x = rng.integers(0, 40, size=(nch, ns), dtype=np.uint8)
    y = rng.integers(0, 40, size=(nch, ns), dtype=np.uint8)
    dx = oracle.dedisperse(oracle.decimate(x, 1), tab).astype(np.int64)
    dy = oracle.dedisperse(oracle.decimate(y, 1), tab).astype(np.int64)
    dz = oracle.dedisperse(oracle.decimate((2 * x + 3 * y).astype(np.uint8), 1), tab).astype(np.int64)
    assert (dz == 2 * dx + 3 * dy).all()


# ---------------------------------------------------------------- P6
@pytest.mark.parametrize("decim,bits", [(1, 8), (2, 8), (4, 8), (8, 8), (1, 16), (8, 16)])
def test_p6_constant_input(decim, bits):
    nch, ns, v = 20, 803, (200 if bits == 8 else 60000)
    x = np.full((nch, ns), v, dtype=np.uint8 if bits == 8 else np.uint16)
    tab = oracle.delay_table(500.0, -10.0, nch, 1.024e-3, decim, 0.0, 4.0, 6)
    y = oracle.decimate(x, decim)
    assert y.shape == (nch, ns // decim) and (y == decim * v).all()
    ns_r, maxd, nout = oracle.range_sizes(ns, decim, tab)
    out = oracle.dedisperse(y, tab)
    assert out.shape == (6, nout) and nout == ns // decim - int(tab[-1, -1])
    assert (out == np.float32(nch * decim * v)).all()


# ---------------------------------------------------------------- P7
def test_p7_time_shift_covariance():
    x, tab = _small(seed=11)
    s = 17
    xs = np.zeros_like(x)
    xs[:, s:] = x[:, :-s]
    a = oracle.dedisperse(oracle.decimate(x, 1), tab)
    b = oracle.dedisperse(oracle.decimate(xs, 1), tab)
    assert (b[:, s:] == a[:, :-s]).all()


# ---------------------------------------------------------------- P8
def test_p8_single_channel_is_identity():
    rng = np.random.default_rng(5)
    x = rng.integers(0, 256, size=(1, 300), dtype=np.uint8)
    tab = oracle.delay_table(500.0, -1.0, 1, 1e-3, 1, 0.0, 10.0, 5)
    assert (tab == 0).all()
    out = oracle.dedisperse(oracle.decimate(x, 1), tab)
    assert out.shape == (5, 300)
    assert (out == x.astype(np.float32)).all()


# ---------------------------------------------------------------- P9
@pytest.mark.parametrize("decim", [2, 4, 8])
def test_p9_decimation_reduction(decim):
    rng = np.random.default_rng(9)
    nch, ns = 12, 1003                      # 1003 mod k != 0: the tail is dropped
    x = rng.integers(0, 256, size=(nch, ns), dtype=np.uint8)
    y = oracle.decimate(x, decim)
    want = x[:, :(ns // decim) * decim].astype(np.uint32).reshape(nch, ns // decim, decim).sum(axis=2)
    assert (y == want).all()
    # a xk range == the x1 path on the pre-summed series sampled at tsamp*k
    tab_k = oracle.delay_table(500.0, -15.0, nch, 1.0e-3, decim, 5.0, 2.0, 7)
    tab_1 = oracle.delay_table(500.0, -15.0, nch, 1.0e-3 * decim, 1, 5.0, 2.0, 7)
    assert (tab_k == tab_1).all()
    a = oracle.dedisperse(y, tab_k)
    pre = want.astype(np.uint16)            # a 16-bit filterbank sampled at tsamp*k
    b = oracle.dedisperse(oracle.decimate(pre, 1), tab_1)
    assert a.shape == b.shape and (a == b).all()


# ---------------------------------------------------------------- P10
def test_p10_brute_force_hand_delays():
    """4 channels at 1000/800/600/400 MHz, tsamp 1 ms, DMs 0, 0.5, 1.0.  Delays worked by hand from
    Eq. 1.1 with (1/f_GHz^2 - 1) = 0, 0.5625, 1.7778, 5.25:
        DM 0.5: 0, 1.167 -> 1, 3.688 -> 4, 10.891 -> 11
        DM 1.0: 0, 2.334 -> 2, 7.376 -> 7, 21.781 -> 22"""
    hand = [[0, 0, 0, 0], [0, 1, 4, 11], [0, 2, 7, 22]]
    tab = oracle.delay_table(1000.0, -200.0, 4, 1.0e-3, 1, 0.0, 0.5, 3)
    assert tab.tolist() == hand
    rng = np.random.default_rng(10)
    x = rng.integers(0, 256, size=(4, 32), dtype=np.uint8)
    out = oracle.dedisperse(oracle.decimate(x, 1), tab)
    nout = 32 - 22
    assert out.shape == (3, nout)
    for j in range(3):
        for t in range(nout):
            s = 0
            for c in range(4):
                s += int(x[c][t + hand[j][c]])
            assert out[j][t] == float(s)
    # a selected trial and window give the same numbers
    sub = oracle.dedisperse(oracle.decimate(x, 1), tab, sel=[2, 1], t0=3, nt=5)
    assert (sub[0] == out[2, 3:8]).all() and (sub[1] == out[1, 3:8]).all()


def test_p10_brute_force_decimated_uint16():
    """Same idea through O6: channels at 1000/700/400 MHz, tsamp 0.5 ms, x2 decimation (1 ms per
    decimated sample), DM 1, uint16 data.  Hand delays from Eq. 1.1:
        (1/0.7^2 - 1) = 1.040816 -> 4.148808*1.040816 = 4.31815 ms -> 4.318 samples -> 4
        (1/0.4^2 - 1) = 5.25     -> 21.78124 ms -> 21.78 samples -> 22"""
    tab = oracle.delay_table(1000.0, -300.0, 3, 0.5e-3, 2, 0.0, 1.0, 2)
    hand = [[0, 0, 0], [0, 4, 22]]
    assert tab.tolist() == hand
    rng = np.random.default_rng(12)
    x = rng.integers(60000, 65536, size=(3, 101), dtype=np.uint16)
    y = oracle.decimate(x, 2)
    out = oracle.dedisperse(y, tab)
    nout = 50 - 22
    assert out.shape == (2, nout)
    for j in range(2):
        for t in range(nout):
            s = 0
            for c in range(3):
                tt = t + hand[j][c]
                s += int(x[c][2 * tt]) + int(x[c][2 * tt + 1])
            assert out[j][t] == np.float32(s)


def test_float_conversion_rounds_to_nearest_even():
    """Sums above 2^24 are rounded once (uint64 -> double -> float), config-4 regime."""
    nch = 300
    x = np.full((nch, 8), 65535, dtype=np.uint16)
    x[0, :] = 65534                       # S = 300*65535 - 1 = 19660499 > 2^24, odd
    tab = np.zeros((1, nch), dtype=np.int64)
    out = oracle.dedisperse(oracle.decimate(x, 1), tab)
    s = 300 * 65535 - 1
    assert s > 2 ** 24
    assert out[0, 0] == np.float32(s) and float(out[0, 0]) in (float(s - 1), float(s + 1), float(s))
    assert float(np.float32(s)) != float(s)     # really inexact: the rounding is exercised


# ---------------------------------------------------------------- P11
def test_p11_exactness_bounds():
    """u8 configs: every sum < 2^24 so fp32 holds it exactly -> GPU must match bit for bit.
    config 4: sums fit uint32."""
    for k, w in W.CONFIGS.items():
        for rg in w.ranges:
            bound = w.nchans * (2 ** w.in_bits - 1) * rg.decim
            if w.in_bits == 8:
                assert bound < 2 ** 24, (k, bound)
            else:
                assert bound < 2 ** 32, (k, bound)


# ---------------------------------------------------------------- P12
def test_p12_zeroed_channels_equal_subset():
    x, tab = _small(seed=21, nch=30)
    tab = oracle.delay_table(500.0, -200.0 / 30, 30, 1.024e-3, 1, 0.0, 1.5, 20)
    dead = [3, 4, 17, 29]
    xz = x.copy()
    xz[dead, :] = 0
    a = oracle.dedisperse(oracle.decimate(xz, 1), tab)
    keep = [c for c in range(30) if c not in dead]
    nout = a.shape[1]
    b = oracle.dedisperse(oracle.decimate(x[keep], 1), tab[:, keep], t0=0, nt=nout)
    assert (a == b).all()


# ---------------------------------------------------------------- workloads sanity (shared generator)
def test_workload_generator_is_seeded_and_shaped():
    w = W.CONFIGS[1]
    a = W.generate(w)
    b = W.generate(w, threads=1)
    assert a.shape == (1, 128, 8192) and a.dtype == np.uint8 and (a == b).all()
    assert abs(a.mean() - 128) < 0.5 and abs(a.std() - 10) < 0.5
    assert [r.ndm for r in W.CONFIGS[3].ranges] == [2000, 2000, 2801]
    assert [r.ndm for r in W.CONFIGS[4].ranges] == [4000, 2001]
    assert W.CONFIGS[2].total_trials == 1001 and W.CONFIGS[5].total_trials == 2001
    w3 = W.scaled(W.CONFIGS[3], nchans=256, nsamps=4096)
    x3 = W.generate(w3)
    z = W.zeroed_channels(w3, 0)
    assert len(z) == 5 and (x3[0, z] == 0).all()


def test_cfg1_injected_pulse_recovered_at_dm50():
    """End-to-end sanity in the spirit of the thesis's injection test: the config-1
    pulse (DM 50, t0 1024, width 4, height +40) is the global maximum of the oracle's DM-time plane."""
    w = W.CONFIGS[1]
    x = W.generate(w)[0]
    rg = w.ranges[0]
    tab = oracle.delay_table(w.f_top_mhz, w.chan_width_mhz, w.nchans, w.tsamp_s, 1, rg.dm_lo, rg.dm_step, rg.ndm)
    out = oracle.dedisperse(oracle.decimate(x, 1), tab)
    j, t = np.unravel_index(np.argmax(out), out.shape)
    assert abs(j - 50) <= 1 and 1024 <= t <= 1028
