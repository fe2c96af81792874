"""Thin ctypes binding to libdd.so -- same names as include/dd.h, argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; there is no CPU fallback.
If the library is missing or cannot be loaded this module raises at import of the symbol, loudly.
Device memory and streams come from PyTorch (`tensor.data_ptr()`, `torch.cuda.current_stream()`).
"""
from __future__ import annotations

import ctypes
import os
from typing import List, Optional, Sequence, Tuple

from .build import LIB, build

DD_OK = 0
DD_ERR_INVALID, DD_ERR_TOO_SHORT, DD_ERR_OVERFLOW, DD_ERR_ALIGN, DD_ERR_CUDA, DD_ERR_NOMEM, DD_ERR_DEVICE = -1, -2, -3, -4, -5, -6, -7
DD_KERNEL_AUTO, DD_KERNEL_DIRECT, DD_KERNEL_TILED, DD_KERNEL_SHARED, DD_KERNEL_SUBBAND = 0, 1, 2, 3, 4
DD_LAYOUT_CHANNEL_MAJOR, DD_LAYOUT_SPECTRUM_MAJOR = 0, 1

# every symbol include/dd.h declares
SYMBOLS = [
    "dd_plan_create", "dd_execute", "dd_execute_host", "dd_execute_host_async", "dd_host_wait", "dd_plan_set_host_pieces", "dd_plan_destroy", "dd_plan_out_elems",
    "dd_plan_beam_stride", "dd_plan_range_info", "dd_plan_get_delays", "dd_plan_work", "dd_plan_launches",
    "dd_plan_executed_adds", "dd_plan_pair_info",
    "dd_plan_workspace_bytes", "dd_plan_set_workspace", "dd_plan_set_kernel", "dd_plan_tile_info", "dd_plan_delta_chunks",
    "dd_plan_create_host", "dd_plan_create_tail", "dd_plan_create_tuned", "dd_plan_tile_shape", "dd_plan_table",
    "dd_sps_rows", "dd_sps_execute", "dd_sps_candidates", "dd_plan_set_row_stats", "dd_stream_create", "dd_stream_push", "dd_stream_plan", "dd_stream_info", "dd_stream_destroy",
    "dd_plan_set_profiling", "dd_plan_kernel_times", "dd_strerror", "dd_last_cuda_error", "dd_version",
    "dd_post_downsample", "dd_post_dered", "dd_resample_create", "dd_resample_create_host", "dd_resample_info",
    "dd_resample_get_edges", "dd_resample_execute", "dd_resample_destroy",
]
DD_POST_MAX_WINDOW = 8191


class dd_range_t(ctypes.Structure):
    _fields_ = [("dm_lo", ctypes.c_double), ("dm_step", ctypes.c_double), ("ndm", ctypes.c_int32), ("decim", ctypes.c_int32)]


class dd_config_t(ctypes.Structure):
    _fields_ = [
        ("f_top_mhz", ctypes.c_double), ("chan_width_mhz", ctypes.c_double), ("nchans", ctypes.c_int32),
        ("tsamp_s", ctypes.c_double), ("nsamps", ctypes.c_int64), ("nbeams", ctypes.c_int32),
        ("in_bits", ctypes.c_int32), ("nranges", ctypes.c_int32), ("ranges", ctypes.POINTER(dd_range_t)),
        ("in_layout", ctypes.c_int32),
    ]


class dd_tuning_t(ctypes.Structure):
    _fields_ = [("mode", ctypes.c_int32), ("byte_lanes", ctypes.c_int32), ("trial_groups", ctypes.c_int32),
                ("words_per_cta", ctypes.c_int32), ("chans_per_stage", ctypes.c_int32), ("stages", ctypes.c_int32)]


class DDError(RuntimeError):
    def __init__(self, code: int, what: str):
        self.code = code
        lib = _load()
        msg = lib.dd_strerror(code).decode()
        if code == DD_ERR_CUDA:
            msg += " -- " + lib.dd_last_cuda_error().decode()
        super().__init__("%s failed: %s (code %d)" % (what, msg, code))


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()  # returns at once when libdd.so is newer than every source; rebuilds after any edit of csrc/ or dd.h
        lib = ctypes.CDLL(LIB)  # raises OSError if the CUDA extension is missing: no fallback
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        P = ctypes.POINTER
        lib.dd_plan_create.argtypes = [P(dd_config_t), P(vp)]
        lib.dd_execute.argtypes = [vp, vp, vp, vp]
        lib.dd_execute_host.argtypes = [vp, vp, vp, vp]
        lib.dd_execute_host_async.argtypes = [vp, vp, vp, vp]
        lib.dd_host_wait.argtypes = [vp]
        lib.dd_plan_set_host_pieces.argtypes = [vp, i32]
        lib.dd_plan_destroy.argtypes = [vp]
        lib.dd_plan_out_elems.argtypes = [vp, P(i64)]
        lib.dd_plan_beam_stride.argtypes = [vp, P(i64)]
        lib.dd_plan_range_info.argtypes = [vp, i32, P(i64), P(i64), P(i64), P(i64), P(i64)]
        lib.dd_plan_get_delays.argtypes = [vp, i32, vp]
        lib.dd_plan_work.argtypes = [vp, P(i64), P(i64)]
        lib.dd_plan_launches.argtypes = [vp, P(i32)]
        lib.dd_plan_executed_adds.argtypes = [vp, P(i64)]
        lib.dd_plan_pair_info.argtypes = [vp, i32, P(i32), P(i32), P(i32), P(i32)]
        lib.dd_plan_workspace_bytes.argtypes = [vp, P(i64)]
        lib.dd_plan_set_workspace.argtypes = [vp, vp, i64]
        lib.dd_plan_set_kernel.argtypes = [vp, i32]
        lib.dd_plan_tile_info.argtypes = [vp, i32, P(i32), P(i32), P(i32), P(i32), P(i32)]
        lib.dd_plan_delta_chunks.argtypes = [vp, i32, P(i32)]
        lib.dd_plan_create_host.argtypes = [P(dd_config_t), P(vp)]
        lib.dd_plan_create_tail.argtypes = [P(dd_config_t), ctypes.c_int64, P(vp)]
        lib.dd_plan_create_tuned.argtypes = [P(dd_config_t), P(dd_tuning_t), i32, P(vp)]
        lib.dd_sps_rows.argtypes = [vp, P(ctypes.c_int64)]
        lib.dd_sps_execute.argtypes = [vp, vp, i32, ctypes.c_double, vp, vp, vp, vp]
        lib.dd_sps_candidates.argtypes = [vp, vp, i32, ctypes.c_double, vp, vp, vp, i64, vp]
        lib.dd_plan_set_row_stats.argtypes = [vp, vp]
        lib.dd_stream_create.argtypes = [P(dd_config_t), P(vp)]
        lib.dd_stream_push.argtypes = [vp, vp, vp, vp]
        lib.dd_stream_plan.argtypes = [vp]
        lib.dd_stream_plan.restype = vp
        lib.dd_stream_info.argtypes = [vp, P(ctypes.c_int64), P(ctypes.c_int64), P(ctypes.c_int64)]
        lib.dd_stream_destroy.argtypes = [vp]
        lib.dd_plan_tile_shape.argtypes = [vp, i32] + [P(i32)] * 7
        lib.dd_plan_table.argtypes = [vp, i32, i32, vp, ctypes.c_int64, P(ctypes.c_int64)]
        lib.dd_plan_set_profiling.argtypes = [vp, i32]
        lib.dd_plan_kernel_times.argtypes = [vp, i32, i32, P(ctypes.c_float), P(i32), P(i32), P(i32)]
        f64 = ctypes.c_double
        lib.dd_post_downsample.argtypes = [vp, i64, i64, i64, i32, vp, i64, vp]
        lib.dd_post_dered.argtypes = [vp, i64, i64, i64, i32, vp, vp, i64, vp]
        lib.dd_resample_create.argtypes = [f64, f64, f64, f64, i64, P(vp)]
        lib.dd_resample_create_host.argtypes = [f64, f64, f64, f64, i64, P(vp)]
        lib.dd_resample_info.argtypes = [vp, P(i64), P(i32)]
        lib.dd_resample_get_edges.argtypes = [vp, vp]
        lib.dd_resample_execute.argtypes = [vp, vp, i64, i64, vp, i64, vp]
        lib.dd_resample_destroy.argtypes = [vp]
        lib.dd_strerror.argtypes = [ctypes.c_int]
        lib.dd_strerror.restype = ctypes.c_char_p
        lib.dd_last_cuda_error.restype = ctypes.c_char_p
        for name in SYMBOLS:
            getattr(lib, name)  # AttributeError if the library does not export it
        _lib = lib
    return _lib


def library_path() -> str:
    return LIB


def dd_version() -> int:
    return int(_load().dd_version())


def dd_strerror(code: int) -> str:
    return _load().dd_strerror(code).decode()


def _chk(rc: int, what: str) -> None:
    if rc != DD_OK:
        raise DDError(rc, what)


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        return None
    if isinstance(stream, int):
        return stream or None
    return int(stream.cuda_stream) or None  # torch.cuda.Stream


class Plan:
    """Owns a dd_plan_t*.  Methods mirror the C entry points one to one."""

    def __init__(self, f_top_mhz: float, chan_width_mhz: float, nchans: int, tsamp_s: float, nsamps: int,
                 ranges: Sequence[Tuple[float, float, int, int]], nbeams: int = 1, in_bits: int = 8,
                 in_layout: int = DD_LAYOUT_CHANNEL_MAJOR, host_only: bool = False, tuning: Optional[dict] = None):
        """tuning: None (automatic) or a dict with any of the dd_tuning_t fields (mode, byte_lanes, trial_groups,
        words_per_cta, chans_per_stage, stages) -> dd_plan_create_tuned."""
        lib = _load()
        arr = (dd_range_t * max(1, len(ranges)))()
        for i, (lo, step, ndm, decim) in enumerate(ranges):
            arr[i] = dd_range_t(float(lo), float(step), int(ndm), int(decim))
        cfg = dd_config_t(float(f_top_mhz), float(chan_width_mhz), int(nchans), float(tsamp_s), int(nsamps),
                          int(nbeams), int(in_bits), len(ranges), arr, int(in_layout))
        h = ctypes.c_void_p()
        if tuning is not None:
            t = dd_tuning_t(int(tuning.get("mode", -1)), int(tuning.get("byte_lanes", -1)), int(tuning.get("trial_groups", 0)),
                            int(tuning.get("words_per_cta", 0)), int(tuning.get("chans_per_stage", 0)), int(tuning.get("stages", 0)))
            _chk(lib.dd_plan_create_tuned(ctypes.byref(cfg), ctypes.byref(t), 1 if host_only else 0, ctypes.byref(h)),
                 "dd_plan_create_tuned")
        elif host_only:
            _chk(lib.dd_plan_create_host(ctypes.byref(cfg), ctypes.byref(h)), "dd_plan_create_host")
        else:
            _chk(lib.dd_plan_create(ctypes.byref(cfg), ctypes.byref(h)), "dd_plan_create")
        self._h = h
        self.nranges = len(ranges)
        self.nchans, self.nbeams, self.in_bits, self.nsamps = int(nchans), int(nbeams), int(in_bits), int(nsamps)
        self.ranges = [(float(a), float(b), int(c), int(d)) for a, b, c, d in ranges]

    @classmethod
    def from_workload(cls, w, in_layout: int = DD_LAYOUT_CHANNEL_MAJOR, ascending: bool = False,
                      host_only: bool = False, tuning: Optional[dict] = None) -> "Plan":
        """ascending=True describes the same band listed from its lowest channel upwards (the data must then be
        given in that order)."""
        f0, cw = w.f_top_mhz, w.chan_width_mhz
        if ascending:
            f0, cw = f0 + (w.nchans - 1) * cw, -cw
        return cls(f0, cw, w.nchans, w.tsamp_s, w.nsamps,
                   [(r.dm_lo, r.dm_step, r.ndm, r.decim) for r in w.ranges], w.nbeams, w.in_bits, in_layout, host_only,
                   tuning)

    # -- dd_plan_destroy
    def destroy(self) -> None:
        if getattr(self, "_h", None):
            if getattr(self, "_owned", True):
                _load().dd_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # -- dd_execute / dd_execute_host
    def execute(self, in_dev, out_dev, stream=None) -> None:
        """in_dev / out_dev: torch CUDA tensors (or raw device pointers as int)."""
        ip = in_dev if isinstance(in_dev, int) else in_dev.data_ptr()
        op = out_dev if isinstance(out_dev, int) else out_dev.data_ptr()
        _chk(_load().dd_execute(self._h, ip, op, _stream_ptr(stream)), "dd_execute")

    def execute_host(self, in_host, out_host, stream=None) -> None:
        """in_host / out_host: host buffers (numpy arrays, pinned torch tensors, or int addresses)."""
        def addr(a):
            if isinstance(a, int):
                return a
            if hasattr(a, "data_ptr"):
                return a.data_ptr()
            return a.ctypes.data
        _chk(_load().dd_execute_host(self._h, addr(in_host), addr(out_host), _stream_ptr(stream)), "dd_execute_host")

    def execute_host_async(self, in_host, out_host, stream=None) -> None:
        """dd_execute_host without the final wait (page-locked buffers; consecutive calls need different out_host)."""
        def addr(a):
            if isinstance(a, int):
                return a
            if hasattr(a, "data_ptr"):
                return a.data_ptr()
            return a.ctypes.data
        _chk(_load().dd_execute_host_async(self._h, addr(in_host), addr(out_host), _stream_ptr(stream)),
             "dd_execute_host_async")

    def host_wait(self) -> None:
        _chk(_load().dd_host_wait(self._h), "dd_host_wait")

    def set_host_pieces(self, pieces: int) -> None:
        _chk(_load().dd_plan_set_host_pieces(self._h, pieces), "dd_plan_set_host_pieces")

    # -- queries
    def out_elems(self) -> int:
        v = ctypes.c_int64()
        _chk(_load().dd_plan_out_elems(self._h, ctypes.byref(v)), "dd_plan_out_elems")
        return v.value

    def beam_stride(self) -> int:
        v = ctypes.c_int64()
        _chk(_load().dd_plan_beam_stride(self._h, ctypes.byref(v)), "dd_plan_beam_stride")
        return v.value

    def range_info(self, r: int) -> dict:
        vals = [ctypes.c_int64() for _ in range(5)]
        _chk(_load().dd_plan_range_info(self._h, r, *[ctypes.byref(v) for v in vals]), "dd_plan_range_info")
        keys = ["ns", "maxd", "nout", "pitch", "offset"]
        d = {k: v.value for k, v in zip(keys, vals)}
        d["ndm"] = self.ranges[r][2]
        d["decim"] = self.ranges[r][3]
        return d

    def get_delays(self, r: int):
        import numpy as np
        buf = np.empty((self.ranges[r][2], self.nchans), dtype=np.int32)
        _chk(_load().dd_plan_get_delays(self._h, r, buf.ctypes.data), "dd_plan_get_delays")
        return buf

    def work(self) -> Tuple[int, int]:
        a, b = ctypes.c_int64(), ctypes.c_int64()
        _chk(_load().dd_plan_work(self._h, ctypes.byref(a), ctypes.byref(b)), "dd_plan_work")
        return a.value, b.value

    def launches(self) -> int:
        v = ctypes.c_int32()
        _chk(_load().dd_plan_launches(self._h, ctypes.byref(v)), "dd_plan_launches")
        return v.value

    def executed_adds(self) -> int:
        v = ctypes.c_int64()
        _chk(_load().dd_plan_executed_adds(self._h, ctypes.byref(v)), "dd_plan_executed_adds")
        return v.value

    def pair_info(self, r: int) -> dict:
        vals = [ctypes.c_int32() for _ in range(4)]
        _chk(_load().dd_plan_pair_info(self._h, r, *[ctypes.byref(v) for v in vals]), "dd_plan_pair_info")
        return {k: v.value for k, v in zip(["enabled", "pairs_per_stage", "row_superwords", "npairs"], vals)}

    def workspace_bytes(self) -> int:
        v = ctypes.c_int64()
        _chk(_load().dd_plan_workspace_bytes(self._h, ctypes.byref(v)), "dd_plan_workspace_bytes")
        return v.value

    def set_workspace(self, dev, nbytes: int = 0) -> None:
        ptr = None if dev is None else (dev if isinstance(dev, int) else dev.data_ptr())
        if dev is not None and not isinstance(dev, int) and not nbytes:
            nbytes = dev.numel() * dev.element_size()
        _chk(_load().dd_plan_set_workspace(self._h, ptr, int(nbytes)), "dd_plan_set_workspace")
        self._ws_ref = dev  # keep the tensor alive

    def set_kernel(self, variant: int) -> None:
        _chk(_load().dd_plan_set_kernel(self._h, int(variant)), "dd_plan_set_kernel")

    def tile_info(self, r: int) -> dict:
        vals = [ctypes.c_int32() for _ in range(5)]
        _chk(_load().dd_plan_tile_info(self._h, r, *[ctypes.byref(v) for v in vals]), "dd_plan_tile_info")
        return {k: v.value for k, v in zip(["dm_per_cta", "words_per_cta", "lanes", "flush_chans", "mode"], vals)}

    def delta_chunks(self, r: int) -> int:
        v = ctypes.c_int32()
        _chk(_load().dd_plan_delta_chunks(self._h, r, ctypes.byref(v)), "dd_plan_delta_chunks")
        return int(v.value)

    def tile_shape(self, r: int) -> dict:
        vals = [ctypes.c_int32() for _ in range(7)]
        _chk(_load().dd_plan_tile_shape(self._h, r, *[ctypes.byref(v) for v in vals]), "dd_plan_tile_shape")
        keys = ["trial_groups", "chans_per_stage", "stages", "row_superwords", "cpad", "nblocks", "tiled"]
        return {k: v.value for k, v in zip(keys, vals)}

    def table(self, r: int, which: int):
        """Tables of the tiled kernel (test hook): which = 0 per-trial table (uint32), 1 row starts, 2 row spans;
        3, 4, 5 the same of the pair mode, 6 delta_v per pair (after set_kernel(DD_KERNEL_SUBBAND))."""
        import numpy as np
        n = ctypes.c_int64()
        _chk(_load().dd_plan_table(self._h, r, which, None, 0, ctypes.byref(n)), "dd_plan_table")
        buf = np.empty(n.value // 4, dtype=np.uint32 if which in (0, 3) else np.int32)
        _chk(_load().dd_plan_table(self._h, r, which, buf.ctypes.data, n.value, ctypes.byref(n)), "dd_plan_table")
        return buf

    # -- single-pulse search on the DM-time plane
    def sps_rows(self) -> int:
        v = ctypes.c_int64()
        _chk(_load().dd_sps_rows(self._h, ctypes.byref(v)), "dd_sps_rows")
        return v.value

    def sps_execute(self, plane_dev, nwidths: int, threshold: float, snr_dev, tmax_dev, count_dev, stream=None) -> None:
        """All buffers are torch CUDA tensors (or raw device pointers): float32 / int32 / int32 [rows][nwidths]."""
        ptr = lambda a: a if isinstance(a, int) else a.data_ptr()  # noqa: E731
        _chk(_load().dd_sps_execute(self._h, ptr(plane_dev), int(nwidths), float(threshold), ptr(snr_dev), ptr(tmax_dev),
                                    ptr(count_dev), _stream_ptr(stream)), "dd_sps_execute")

    def sps_candidates(self, plane_dev, nwidths: int, threshold: float, count_dev, offsets_dev, cand_dev, max_cands: int,
                       stream=None) -> None:
        """offsets_dev: int64 [rows*nwidths + 1]; cand_dev: max_cands entries of dd_sps_cand_t (16 bytes each:
        int32 row, int32 width_log2, int32 t, float32 snr), e.g. an int32 tensor [max_cands][4]."""
        ptr = lambda a: None if a is None else (a if isinstance(a, int) else a.data_ptr())  # noqa: E731
        _chk(_load().dd_sps_candidates(self._h, ptr(plane_dev), int(nwidths), float(threshold), ptr(count_dev),
                                       ptr(offsets_dev), ptr(cand_dev), int(max_cands), _stream_ptr(stream)), "dd_sps_candidates")

    def set_row_stats(self, stats_dev) -> None:
        """stats_dev: int64 CUDA tensor of sps_rows()*2 elements (or None to switch the epilogue statistics off)."""
        ptr = None if stats_dev is None else (stats_dev if isinstance(stats_dev, int) else stats_dev.data_ptr())
        _chk(_load().dd_plan_set_row_stats(self._h, ptr), "dd_plan_set_row_stats")
        self._stats_ref = stats_dev

    def set_profiling(self, max_executes: int) -> None:
        _chk(_load().dd_plan_set_profiling(self._h, int(max_executes)), "dd_plan_set_profiling")

    def kernel_times(self, slot: int) -> List[dict]:
        cap = 3 * self.nranges
        ms = (ctypes.c_float * cap)()
        kind = (ctypes.c_int32 * cap)()
        rng = (ctypes.c_int32 * cap)()
        n = ctypes.c_int32()
        _chk(_load().dd_plan_kernel_times(self._h, slot, cap, ms, kind, rng, ctypes.byref(n)), "dd_plan_kernel_times")
        names = {0: "pack", 1: "tiled", 2: "direct", 3: "pairs"}
        return [{"ms": float(ms[i]), "kind": names[kind[i]], "range": int(rng[i])} for i in range(n.value)]

    # -- convenience for callers holding torch tensors
    def view_range(self, out, r: int, beam: int = 0):
        """View of the valid [ndm_r][nout_r] block of range r, beam `beam`, inside the flat output."""
        info = self.range_info(r)
        base = beam * self.beam_stride() + info["offset"]
        flat = out.reshape(-1)[base: base + info["ndm"] * info["pitch"]]
        return flat.reshape(info["ndm"], info["pitch"])[:, : info["nout"]]


class Stream:
    """Owns a dd_stream_t*: dedispersion of a sequence of blocks with a carried halo (dd_stream_* of include/dd.h).
    `nsamps` of the description is the block length."""

    def __init__(self, f_top_mhz: float, chan_width_mhz: float, nchans: int, tsamp_s: float, block_samps: int,
                 ranges: Sequence[Tuple[float, float, int, int]], nbeams: int = 1, in_bits: int = 8,
                 in_layout: int = DD_LAYOUT_CHANNEL_MAJOR):
        lib = _load()
        arr = (dd_range_t * max(1, len(ranges)))()
        for i, (lo, step, ndm, decim) in enumerate(ranges):
            arr[i] = dd_range_t(float(lo), float(step), int(ndm), int(decim))
        cfg = dd_config_t(float(f_top_mhz), float(chan_width_mhz), int(nchans), float(tsamp_s), int(block_samps),
                          int(nbeams), int(in_bits), len(ranges), arr, int(in_layout))
        h = ctypes.c_void_p()
        _chk(lib.dd_stream_create(ctypes.byref(cfg), ctypes.byref(h)), "dd_stream_create")
        self._h = h
        plan = Plan.__new__(Plan)           # non-owning view of the window plan, for the queries
        plan._h = ctypes.c_void_p(lib.dd_stream_plan(h))
        plan._owned = False
        plan.nranges = len(ranges)
        plan.nchans, plan.nbeams, plan.in_bits = int(nchans), int(nbeams), int(in_bits)
        plan.ranges = [(float(a), float(b), int(c), int(d)) for a, b, c, d in ranges]
        self.plan = plan
        b, hs, n = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        _chk(lib.dd_stream_info(h, ctypes.byref(b), ctypes.byref(hs), ctypes.byref(n)), "dd_stream_info")
        self.block, self.hist = b.value, hs.value
        plan.nsamps = self.block + self.hist

    def push(self, block_dev, out_dev, stream=None) -> None:
        bp = block_dev if isinstance(block_dev, int) else block_dev.data_ptr()
        op = out_dev if isinstance(out_dev, int) else out_dev.data_ptr()
        _chk(_load().dd_stream_push(self._h, bp, op, _stream_ptr(stream)), "dd_stream_push")

    def destroy(self) -> None:
        if getattr(self, "_h", None):
            self.plan._h = None
            _load().dd_stream_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


# ---- pulsar-side post-processing of dedispersed series (dd_post_* / dd_resample_* of include/dd.h) -------------------
def _p(a):
    return None if a is None else (a if isinstance(a, int) else a.data_ptr())


def post_downsample(in_dev, nrows: int, in_pitch: int, n: int, factor: int, out_dev, out_pitch: int, stream=None) -> None:
    _chk(_load().dd_post_downsample(_p(in_dev), nrows, in_pitch, n, factor, _p(out_dev), out_pitch, _stream_ptr(stream)),
         "dd_post_downsample")


def post_dered(in_dev, nrows: int, in_pitch: int, n: int, window: int, median_dev, out_dev, out_pitch: int, stream=None) -> None:
    _chk(_load().dd_post_dered(_p(in_dev), nrows, in_pitch, n, window, _p(median_dev), _p(out_dev), out_pitch,
                               _stream_ptr(stream)), "dd_post_dered")


class Resample:
    """Owns a dd_resample_t*: re-sampling of series of n samples for one (f0, f1, f2) (Eqs 3.1-3.6)."""

    def __init__(self, f0: float, f1: float, f2: float, tsamp_s: float, n: int, host_only: bool = False):
        lib = _load()
        h = ctypes.c_void_p()
        fn = lib.dd_resample_create_host if host_only else lib.dd_resample_create
        _chk(fn(float(f0), float(f1), float(f2), float(tsamp_s), int(n), ctypes.byref(h)), "dd_resample_create")
        self._h = h
        m, rev = ctypes.c_int64(), ctypes.c_int32()
        _chk(lib.dd_resample_info(h, ctypes.byref(m), ctypes.byref(rev)), "dd_resample_info")
        self.n, self.out_len, self.reversed = int(n), m.value, bool(rev.value)

    def edges(self):
        import numpy as np
        u = np.empty(self.out_len + 1, dtype=np.float64)
        _chk(_load().dd_resample_get_edges(self._h, u.ctypes.data), "dd_resample_get_edges")
        return u

    def execute(self, in_dev, nrows: int, in_pitch: int, out_dev, out_pitch: int, stream=None) -> None:
        _chk(_load().dd_resample_execute(self._h, _p(in_dev), nrows, in_pitch, _p(out_dev), out_pitch, _stream_ptr(stream)),
             "dd_resample_execute")

    def destroy(self) -> None:
        if getattr(self, "_h", None):
            _load().dd_resample_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
