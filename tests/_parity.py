"""Shared helpers of the GPU parity tests: tolerances and oracle-side evaluation."""
import numpy as np

from oracle.check import REL, check_float_maps  # noqa: F401  (the criterion lives beside the oracle)


def oracle_maps(oracle, frames, ref, s_first=1, nthreads=None, scale=1.0):
    nt = oracle.max_threads() if nthreads is None else nthreads
    return oracle.qld(frames, ref, s_first=s_first, nthreads=nt, scale=scale)


def forced(Q, which, tile):
    """Q.QLD with the tile shape of a kernel forced through qld_debug_set_tile (tile = "SEG,KC" for which = "stream",
    "T,STAGES,KC" for "tc"; empty: the automatic choice)."""
    import functools
    if not tile:
        return Q.QLD
    return functools.partial(Q.QLD, debug_tile=(which,) + tuple(int(t) for t in str(tile).split(",")))
