"""NEXT-4 parity: downsampling, running-median de-reddening and re-sampling of dedispersed series (PAPER.md:421,
:425, :441-484) -- the CUDA path through the C ABI against oracle/oracle_post.c, element by element, bit for bit.
CPU part: the re-sampling bin edges of the host plan builder against the oracle's (no GPU needed)."""
import numpy as np
import pytest

import oracle
from paper_2605_03531_b200 import binding as B
from paper_2605_03531_b200 import workloads as W

gpu = pytest.mark.gpu

_RESAMPLE_CASES = [(2.5, 0.0, 0.0, 1e-3, 5000), (2.5, -1.25e-4, 0.0, 1e-3, 60000), (2.5, -1.0e-4, -3.0e-6, 1e-3, 60000),
                   (2.5, 1.25e-4, 0.0, 1e-3, 60000), (3.0, 0.04, 0.002, 1e-3, 5000), (10.0, -0.5, 0.0, 0.01, 2000),
                   (5.0, -0.8, -0.02, 2e-3, 3000), (700.0, -3.0, 0.05, 1.31072e-3, 65536), (4.0, -6.0, 2.0, 0.05, 40)]


def test_resample_edges_match_the_oracle_bit_for_bit():
    """a1-like check without a GPU: dd_resample_create_host builds the edges of Eq 3.3 (reading C3) in the same IEEE
    double operations as the oracle."""
    for f0, f1, f2, ts, n in _RESAMPLE_CASES:
        u, rev = oracle.resample_edges(f0, f1, f2, ts, n)
        r = B.Resample(f0, f1, f2, ts, n, host_only=True)
        assert r.out_len == len(u) - 1 and r.reversed == rev, (f0, f1, f2)
        assert np.array_equal(r.edges().view(np.uint64), u.view(np.uint64)), (f0, f1, f2)
        r.destroy()
    with pytest.raises(B.DDError):          # folds back / bins shorter than half a sample: refused like the oracle
        B.Resample(1.0, 0.0, 50.0, 0.01, 100000, host_only=True)
    with pytest.raises(B.DDError):
        B.Resample(0.0, 0.0, 0.0, 0.01, 100, host_only=True)


def _plane(nrows, n, seed, kind="dmtime"):
    """Rows shaped like DM-time rows: integer-valued floats around nchans*mean with a slow baseline and pulses."""
    rng = np.random.default_rng(seed)
    t = np.arange(n)
    rows = np.empty((nrows, n), dtype=np.float32)
    for r in range(nrows):
        base = 524288.0 + 3000.0 * np.sin(2 * np.pi * t / (700.0 + 90 * r)) + 0.2 * t
        x = np.rint(base + rng.normal(0.0, 770.0, size=n))
        for _ in range(5 if n > 100 else 0):
            p = int(rng.integers(0, n - 40))
            x[p:p + int(rng.integers(1, 30))] += 5000.0
        rows[r] = x
    if kind == "ties":
        rows = np.floor(rows / 512.0).astype(np.float32)          # heavy ties
    if kind == "signed":
        rows = (rows - 524288.0).astype(np.float32) * np.float32(0.37)   # negative and fractional values
    return rows


def _gpu_rows(rows, pitch):
    import torch
    buf = torch.full((rows.shape[0], pitch), -7.0, dtype=torch.float32, device="cuda")
    buf[:, : rows.shape[1]] = torch.from_numpy(rows).cuda()
    return buf


@gpu
@pytest.mark.parametrize("factor", [1, 2, 3, 8, 13, 64])
def test_downsample_bit_exact(factor):
    import torch
    rows = _plane(5, 10007, 1)
    rows[0, :16] = 2.0 ** 24 + np.arange(16) * 2.0                 # sums above 2^24: the single rounding matters
    want = oracle.downsample(rows, factor)
    m = want.shape[1]
    x = _gpu_rows(rows, 10016)
    out = torch.full((5, m + 3), -1.0, dtype=torch.float32, device="cuda")
    B.post_downsample(x, 5, 10016, 10007, factor, out, m + 3, torch.cuda.current_stream())
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.array_equal(got[:, :m].view(np.uint32), want.view(np.uint32))
    assert (got[:, m:] == -1.0).all()


@gpu
@pytest.mark.parametrize("kind", ["dmtime", "ties", "signed"])
@pytest.mark.parametrize("n,window", [(5000, 1), (5000, 3), (4097, 33), (7001, 101), (9000, 1001), (2500, 2499), (300, 299),
                                      (20000, 4095)])
def test_running_median_bit_exact(kind, n, window):
    import torch
    if window > 1500 and kind != "dmtime":
        pytest.skip("large windows once")
    nrows = 3
    rows = _plane(nrows, n, 100 + window, kind)
    med, out = oracle.running_median(rows, window)
    pitch = (n + 31) // 32 * 32
    x = _gpu_rows(rows, pitch)
    gm = torch.full((nrows, pitch), -1.0, dtype=torch.float32, device="cuda")
    go = torch.full((nrows, pitch), -1.0, dtype=torch.float32, device="cuda")
    B.post_dered(x, nrows, pitch, n, window, gm, go, pitch, torch.cuda.current_stream())
    torch.cuda.synchronize()
    gmh, goh = gm.cpu().numpy(), go.cpu().numpy()
    bad = np.argwhere(gmh[:, :n] != med)
    assert bad.size == 0, (bad[:5], gmh[tuple(bad[0])], med[tuple(bad[0])])
    assert np.array_equal(goh[:, :n].view(np.uint32), out.view(np.uint32))
    assert (gmh[:, n:] == -1.0).all() and (goh[:, n:] == -1.0).all()
    # either output may be left out
    go.fill_(-1.0)
    B.post_dered(x, nrows, pitch, n, window, None, go, pitch, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert np.array_equal(go.cpu().numpy()[:, :n].view(np.uint32), out.view(np.uint32))


@gpu
def test_running_median_rejects_bad_windows():
    import torch
    x = torch.zeros((2, 64), dtype=torch.float32, device="cuda")
    o = torch.zeros((2, 64), dtype=torch.float32, device="cuda")
    for w in (0, 2, 65, 8193):
        with pytest.raises(B.DDError) as e:
            B.post_dered(x, 2, 64, 64, w, None, o, 64)
        assert e.value.code == B.DD_ERR_INVALID
    with pytest.raises(B.DDError):
        B.post_dered(x, 2, 64, 64, 3, None, None, 64)


@gpu
@pytest.mark.parametrize("case", _RESAMPLE_CASES)
def test_resample_bit_exact(case):
    import torch
    f0, f1, f2, ts, n = case
    rows = _plane(4, n, 7)
    want = oracle.resample(rows, f0, f1, f2, ts)
    r = B.Resample(f0, f1, f2, ts, n)
    m = r.out_len
    assert m == want.shape[1]
    x = _gpu_rows(rows, n + 5)
    out = torch.full((4, m + 2), -1.0, dtype=torch.float32, device="cuda")
    r.execute(x, 4, n + 5, out, m + 2, torch.cuda.current_stream())
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.array_equal(got[:, :m].view(np.uint32), want.view(np.uint32)), case
    assert (got[:, m:] == -1.0).all()
    r.destroy()


@gpu
def test_post_chain_on_a_dedispersed_plane():
    """The thesis's order: dedisperse -> downsample -> de-redden -> re-sample, on the rows of the
    DM-time plane written by dd_execute, against the oracle chain fed the oracle's plane."""
    import torch
    w = W.scaled(W.CONFIGS[2], nchans=64, nsamps=2 ** 15, ranges=[W.DMRange(0.0, 2.0, 24, 1)])
    x = W.generate(w)
    plan = B.Plan.from_workload(w)
    out = torch.zeros(plan.out_elems(), dtype=torch.float32, device="cuda")
    plan.execute(torch.from_numpy(x).cuda(), out, torch.cuda.current_stream())
    info = plan.range_info(0)
    ndm, nout, pitch = info["ndm"], info["nout"], info["pitch"]
    tab = oracle.delay_table(w.f_top_mhz, w.chan_width_mhz, w.nchans, w.tsamp_s, 1, 0.0, 2.0, 24)
    plane = oracle.dedisperse(oracle.decimate(x[0], 1), tab)
    F, Wn = 4, 257
    d_want = oracle.downsample(plane, F)
    _, r_want = oracle.running_median(d_want, Wn)
    f0, f1, f2, ts = 1.4, -2.0e-4, 0.0, w.tsamp_s * F
    s_want = oracle.resample(r_want, f0, f1, f2, ts)
    nd = nout // F
    d = torch.empty((ndm, nd), dtype=torch.float32, device="cuda")
    B.post_downsample(out[info["offset"]:], ndm, pitch, nout, F, d, nd, torch.cuda.current_stream())
    rr = torch.empty((ndm, nd), dtype=torch.float32, device="cuda")
    B.post_dered(d, ndm, nd, nd, Wn, None, rr, nd, torch.cuda.current_stream())
    rs = B.Resample(f0, f1, f2, ts, nd)
    s = torch.empty((ndm, rs.out_len), dtype=torch.float32, device="cuda")
    rs.execute(rr, ndm, nd, s, rs.out_len, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert np.array_equal(d.cpu().numpy().view(np.uint32), d_want.view(np.uint32))
    assert np.array_equal(rr.cpu().numpy().view(np.uint32), r_want.view(np.uint32))
    assert np.array_equal(s.cpu().numpy().view(np.uint32), s_want.view(np.uint32))
