"""Helpers shared by the parity tests: run a workload through the C ABI (CUDA) and through the oracle."""
from __future__ import annotations

import numpy as np

import oracle
from paper_2605_03531_b200 import workloads as W


def oracle_tables(w: W.Workload):
    """Per range: (delays int64 [ndm][nchans], ns_r, maxd_r, nout_r) from the oracle."""
    out = []
    for rg in w.ranges:
        tab = oracle.delay_table(w.f_top_mhz, w.chan_width_mhz, w.nchans, w.tsamp_s, rg.decim, rg.dm_lo, rg.dm_step, rg.ndm)
        ns_r, maxd, nout = oracle.range_sizes(w.nsamps, rg.decim, tab)
        out.append((tab, ns_r, maxd, nout))
    return out


def oracle_full(w: W.Workload, x: np.ndarray):
    """Oracle DM-time planes: result[beam][range] = float32 [ndm_r][nout_r]."""
    tabs = oracle_tables(w)
    res = []
    for b in range(w.nbeams):
        per = []
        for rg, (tab, ns_r, maxd, nout) in zip(w.ranges, tabs):
            y = oracle.decimate(x[b], rg.decim)
            per.append(oracle.dedisperse(y, tab))
        res.append(per)
    return res


def gpu_run(w: W.Workload, x: np.ndarray, variant: int = 0, host_path: bool = False, in_layout: int = 0,
            ascending: bool = False, tuning=None):
    """CUDA path through the C ABI.  Returns (plan, flat float32 numpy output).  `x` is always given as
    [beam][channel][time] with channel 0 the highest frequency (the oracle's order); for the other input
    conventions of the ABI it is re-laid out here (channel order reversed / spectra contiguous) before the call."""
    import torch
    from paper_2605_03531_b200 import binding as B

    plan = B.Plan.from_workload(w, in_layout=in_layout, ascending=ascending, tuning=tuning)
    if ascending:
        x = x[:, ::-1, :]
    if in_layout == B.DD_LAYOUT_SPECTRUM_MAJOR:
        x = x.transpose(0, 2, 1)
    x = np.ascontiguousarray(x)
    plan.set_kernel(variant)
    n = plan.out_elems()
    if host_path:
        out = np.full(n, -1.0, dtype=np.float32)
        plan.execute_host(np.ascontiguousarray(x), out)
        return plan, out
    xin = torch.from_numpy(x.view(np.int16) if x.dtype == np.uint16 else x).cuda()
    out = torch.full((n,), -1.0, dtype=torch.float32, device="cuda")
    plan.execute(xin, out, torch.cuda.current_stream())
    torch.cuda.synchronize()
    return plan, out.cpu().numpy()


def check_full(w: W.Workload, x: np.ndarray, plan, flat: np.ndarray, want=None, check_pad=True):
    """Bit-exact comparison of every valid output element with the oracle; pad floats untouched."""
    if want is None:
        want = oracle_full(w, x)
    stride = plan.beam_stride()
    for b in range(w.nbeams):
        for r in range(len(w.ranges)):
            info = plan.range_info(r)
            ref = want[b][r]
            assert ref.shape == (info["ndm"], info["nout"]), (ref.shape, info)
            base = b * stride + info["offset"]
            blk = flat[base: base + info["ndm"] * info["pitch"]].reshape(info["ndm"], info["pitch"])
            got = blk[:, : info["nout"]]
            if not np.array_equal(got.view(np.uint32), ref.view(np.uint32)):
                bad = np.argwhere(got != ref)
                j, t = bad[0]
                raise AssertionError("beam %d range %d: %d mismatches, first at trial %d sample %d: got %r want %r"
                                     % (b, r, len(bad), j, t, got[j, t], ref[j, t]))
            if check_pad:
                assert (blk[:, info["nout"]:] == -1.0).all(), "row padding was written"
