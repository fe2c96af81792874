"""ctypes binding to oracle/oracle_dedisp.c (plain C, OpenMP over trials).

TEST INFRASTRUCTURE ONLY -- see oracle/__init__.py.  The arithmetic lives in the C file; this
module only marshals numpy arrays and composes steps O5 (sizes) from the C results.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_dedisp.c")
_LIB = os.path.join(_HERE, "liboracle_dedisp.so")
_SRC_SPS = os.path.join(_HERE, "oracle_sps.c")
_LIB_SPS = os.path.join(_HERE, "liboracle_sps.so")
_SRC_POST = os.path.join(_HERE, "oracle_post.c")
_LIB_POST = os.path.join(_HERE, "liboracle_post.so")
_lib = None
_lib_sps = None
_lib_post = None

_ERRORS = {-1: "invalid argument", -2: "window exceeds the valid span (too short)", -3: "out of memory"}


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (baseline x86-64, -O3, OpenMP).  Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.run(
            ["gcc", "-O3", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"],
            check=True,
        )
        os.replace(tmp, _LIB)
    if force or not os.path.exists(_LIB_SPS) or os.path.getmtime(_LIB_SPS) < os.path.getmtime(_SRC_SPS):
        tmp = _LIB_SPS + ".tmp.%d" % os.getpid()
        subprocess.run(  # no FMA contraction: the operation order of oracle_sps.c is part of its definition
            ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC_SPS, "-lm"],
            check=True,
        )
        os.replace(tmp, _LIB_SPS)
    if force or not os.path.exists(_LIB_POST) or os.path.getmtime(_LIB_POST) < os.path.getmtime(_SRC_POST):
        tmp = _LIB_POST + ".tmp.%d" % os.getpid()
        subprocess.run(  # no FMA contraction: the operation order of oracle_post.c is part of its definition
            ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC_POST, "-lm"],
            check=True,
        )
        os.replace(tmp, _LIB_POST)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i32, i64, f64, vp = ctypes.c_int32, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_channel_freqs.argtypes = [f64, f64, i32, vp]
        lib.oracle_delay_table.argtypes = [f64, f64, i32, f64, i32, f64, f64, i32, vp]
        lib.oracle_decimate.argtypes = [vp, i32, i64, i64, i32, vp]
        lib.oracle_dedisperse.argtypes = [vp, i64, i64, vp, i32, vp, i32, i64, i64, vp]
        for fn in (lib.oracle_channel_freqs, lib.oracle_delay_table, lib.oracle_decimate, lib.oracle_dedisperse):
            fn.restype = ctypes.c_int
        _lib = lib
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise ValueError("oracle %s: %s (code %d)" % (what, _ERRORS.get(rc, "error"), rc))


def _ptr(a: np.ndarray) -> int:
    return a.ctypes.data


def num_threads() -> int:
    """OpenMP threads the oracle will use (OMP_NUM_THREADS or the host core count)."""
    return int(_load().oracle_num_threads())


def channel_freqs(f_top_mhz: float, chan_width_mhz: float, nchans: int) -> np.ndarray:
    """O2: f_c = f_top + c*width."""
    f = np.empty(nchans, dtype=np.float64)
    _check(_load().oracle_channel_freqs(f_top_mhz, chan_width_mhz, nchans, _ptr(f)), "channel_freqs")
    return f


def delay_table(f_top_mhz, chan_width_mhz, nchans, tsamp_s, decim, dm_lo, dm_step, ndm) -> np.ndarray:
    """O3+O4 (Eq. 1.1): int64 delays [ndm][nchans] in samples of tsamp*decim."""
    d = np.empty((ndm, nchans), dtype=np.int64)
    rc = _load().oracle_delay_table(f_top_mhz, chan_width_mhz, nchans, tsamp_s, decim, dm_lo, dm_step, ndm, _ptr(d))
    _check(rc, "delay_table")
    return d


def range_sizes(nsamps: int, decim: int, delays: np.ndarray):
    """O5: ns_r = nsamps // decim, maxd_r = largest delay of the range, nout_r = ns_r - maxd_r."""
    ns_r = int(nsamps) // int(decim)
    maxd = int(delays.max())
    return ns_r, maxd, ns_r - maxd


def decimate(x: np.ndarray, decim: int) -> np.ndarray:
    """O6: y[c][t'] = sum_{i<decim} x[c][decim*t'+i] as uint32; x is [nchans][nsamps] uint8/uint16."""
    if x.ndim != 2 or x.dtype not in (np.uint8, np.uint16):
        raise ValueError("oracle decimate: x must be a 2-D uint8/uint16 array")
    x = np.ascontiguousarray(x)
    nchans, nsamps = x.shape
    y = np.empty((nchans, nsamps // decim), dtype=np.uint32)
    _check(_load().oracle_decimate(_ptr(x), 8 * x.dtype.itemsize, nchans, nsamps, decim, _ptr(y)), "decimate")
    return y


def dedisperse(y: np.ndarray, delays: np.ndarray, sel=None, t0: int = 0, nt: int | None = None) -> np.ndarray:
    """O7: S[j][t'] = sum_c y[c][t'+d(c,j)] for trials `sel` and t' in [t0, t0+nt).

    y: uint32 [nchans][ns_r] (output of decimate); delays: int64 [ndm][nchans].
    nt defaults to the range's valid span nout_r - t0.  Returns float32 [len(sel)][nt].
    """
    if y.ndim != 2 or y.dtype != np.uint32:
        raise ValueError("oracle dedisperse: y must be a 2-D uint32 array")
    y = np.ascontiguousarray(y)
    delays = np.ascontiguousarray(delays, dtype=np.int64)
    nchans, ns_r = y.shape
    ndm = delays.shape[0]
    if delays.shape[1] != nchans:
        raise ValueError("oracle dedisperse: delay table does not match nchans")
    if sel is None:
        sel_arr = np.arange(ndm, dtype=np.int32)
    else:
        sel_arr = np.ascontiguousarray(sel, dtype=np.int32)
    if nt is None:
        nt = ns_r - int(delays.max()) - t0
    out = np.empty((len(sel_arr), nt), dtype=np.float32)
    rc = _load().oracle_dedisperse(_ptr(y), nchans, ns_r, _ptr(delays), ndm, _ptr(sel_arr), len(sel_arr), t0, nt, _ptr(out))
    _check(rc, "dedisperse")
    return out


def sps(rows: np.ndarray, n: int, nwidths: int, threshold: float):
    """Boxcar single-pulse search on rows of the DM-time plane (oracle_sps.c).

    rows: float32 [nrows][pitch], the first n samples of each row valid.  Returns dict of
    snr float32 [nrows][K], tmax int32, count int32, mean float64 [nrows], sigma float64 [nrows].
    """
    global _lib_sps
    if _lib_sps is None:
        build()
        lib = ctypes.CDLL(_LIB_SPS)
        vp, i64 = ctypes.c_void_p, ctypes.c_int64
        lib.oracle_sps.argtypes = [vp, i64, i64, i64, ctypes.c_int, ctypes.c_double, vp, vp, vp, vp, vp]
        lib.oracle_sps.restype = ctypes.c_int
        _lib_sps = lib
    if rows.ndim != 2 or rows.dtype != np.float32:
        raise ValueError("oracle sps: rows must be a 2-D float32 array")
    rows = np.ascontiguousarray(rows)
    nrows, pitch = rows.shape
    snr = np.empty((nrows, nwidths), dtype=np.float32)
    tmax = np.empty((nrows, nwidths), dtype=np.int32)
    count = np.empty((nrows, nwidths), dtype=np.int32)
    mean = np.empty(nrows, dtype=np.float64)
    sigma = np.empty(nrows, dtype=np.float64)
    rc = _lib_sps.oracle_sps(_ptr(rows), nrows, pitch, n, nwidths, float(threshold), _ptr(snr), _ptr(tmax), _ptr(count),
                             _ptr(mean), _ptr(sigma))
    _check(rc, "sps")
    return {"snr": snr, "tmax": tmax, "count": count, "mean": mean, "sigma": sigma}


def sps_candidates(rows: np.ndarray, n: int, nwidths: int, threshold: float, cap: int = 1 << 20):
    """The candidate list of the boxcar search (oracle_sps.c): structured array of (row, k, t, snr)
    ordered by row, k, t, and the total count (which may exceed `cap`)."""
    sps(rows[:1], n, 1, 0.0)  # loads the library
    lib = _lib_sps
    vp, i64 = ctypes.c_void_p, ctypes.c_int64
    lib.oracle_sps_candidates.argtypes = [vp, i64, i64, i64, ctypes.c_int, ctypes.c_double, vp, vp, vp, vp, i64, vp]
    lib.oracle_sps_candidates.restype = ctypes.c_int
    rows = np.ascontiguousarray(rows)
    nrows, pitch = rows.shape
    cr, ck, ct = (np.empty(cap, dtype=np.int32) for _ in range(3))
    cs = np.empty(cap, dtype=np.float32)
    total = ctypes.c_int64()
    rc = lib.oracle_sps_candidates(_ptr(rows), nrows, pitch, n, nwidths, float(threshold), _ptr(cr), _ptr(ck), _ptr(ct),
                                   _ptr(cs), cap, ctypes.byref(total))
    _check(rc, "sps_candidates")
    m = min(cap, total.value)
    out = np.empty(m, dtype=[("row", np.int32), ("k", np.int32), ("t", np.int32), ("snr", np.float32)])
    out["row"], out["k"], out["t"], out["snr"] = cr[:m], ck[:m], ct[:m], cs[:m]
    return out, total.value


# ---- pulsar-side post-processing of dedispersed series (oracle_post.c) ----------------
def _post():
    global _lib_post
    if _lib_post is None:
        build()
        lib = ctypes.CDLL(_LIB_POST)
        vp, i64, i32, f64 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double
        lib.oracle_downsample.argtypes = [vp, i64, i64, i64, i32, vp, i64]
        lib.oracle_running_median.argtypes = [vp, i64, i64, i64, i32, vp, vp, i64]
        lib.oracle_resample_edges.argtypes = [f64, f64, f64, f64, i64, vp, i64, vp, vp]
        lib.oracle_resample.argtypes = [vp, i64, i64, i64, f64, f64, f64, f64, vp, i64]
        for fn in (lib.oracle_downsample, lib.oracle_running_median, lib.oracle_resample_edges, lib.oracle_resample):
            fn.restype = ctypes.c_int
        _lib_post = lib
    return _lib_post


def _rows(x: np.ndarray) -> np.ndarray:
    if x.ndim != 2 or x.dtype != np.float32:
        raise ValueError("oracle post: rows must be a 2-D float32 array")
    return np.ascontiguousarray(x)


def downsample(rows: np.ndarray, factor: int) -> np.ndarray:
    """C1: y[k] = sum_{i<F} x[k*F+i], k < n//F; float32 [nrows][n//F]."""
    rows = _rows(rows)
    nrows, n = rows.shape
    out = np.empty((nrows, n // factor), dtype=np.float32)
    _check(_post().oracle_downsample(_ptr(rows), nrows, n, n, factor, _ptr(out), max(1, n // factor)), "downsample")
    return out


def running_median(rows: np.ndarray, window: int):
    """C2: (median, x - median) with the centred odd window held at the first / last full window
    near the ends; both float32 [nrows][n]."""
    rows = _rows(rows)
    nrows, n = rows.shape
    med = np.empty((nrows, n), dtype=np.float32)
    out = np.empty((nrows, n), dtype=np.float32)
    _check(_post().oracle_running_median(_ptr(rows), nrows, n, n, window, _ptr(med), _ptr(out), n), "running_median")
    return med, out


def resample_edges(f0: float, f1: float, f2: float, tsamp: float, n: int):
    """C3-C4 (Eq. 3.3): (edges float64 [M+1] in input-sample units, reversed flag)."""
    m = ctypes.c_int64()
    rev = ctypes.c_int32()
    _check(_post().oracle_resample_edges(f0, f1, f2, tsamp, n, None, 0, ctypes.byref(m), ctypes.byref(rev)), "resample_edges")
    u = np.empty(m.value + 1, dtype=np.float64)
    _check(_post().oracle_resample_edges(f0, f1, f2, tsamp, n, _ptr(u), m.value + 1, ctypes.byref(m), ctypes.byref(rev)),
           "resample_edges")
    return u, bool(rev.value)


def resample(rows: np.ndarray, f0: float, f1: float, f2: float, tsamp: float) -> np.ndarray:
    """C5-C7 (Eqs 3.1-3.6): fractional-overlap re-sampling of every row; float32 [nrows][M]."""
    rows = _rows(rows)
    nrows, n = rows.shape
    u, _ = resample_edges(f0, f1, f2, tsamp, n)
    m = len(u) - 1
    out = np.empty((nrows, max(1, m)), dtype=np.float32)
    _check(_post().oracle_resample(_ptr(rows), nrows, n, n, f0, f1, f2, tsamp, _ptr(out), max(1, m)), "resample")
    return out[:, :m]
