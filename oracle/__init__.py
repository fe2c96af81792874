"""CPU oracle for brute-force incoherent dedispersion -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_2605_03531_b200 (the CUDA path) and never
imports it.  See oracle/oracle_dedisp.c for the definition it implements and the paper passages
it follows (PAPER.md:256-263 Eq. 1.1, :317, :421, :431); oracle/oracle_sps.c for the boxcar single-pulse
search on the DM-time plane; oracle/oracle_post.c for downsampling, running-median
de-reddening and re-sampling of dedispersed series.
"""
from .oracle import (  # noqa: F401
    build,
    channel_freqs,
    decimate,
    dedisperse,
    delay_table,
    downsample,
    num_threads,
    range_sizes,
    resample,
    resample_edges,
    running_median,
    sps,
    sps_candidates,
)
