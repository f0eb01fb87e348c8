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


def expected_int_rows(oracle, x, ref, s_first=1, mode="INT_BINS"):
    """What qld_get_bins must hold, from the oracle: difference rows B_r - B_{r+den/2} (even den) or the bins (odd den); in
    INT_REFS mode, for den = 3 or 6 without a phase offset, the two integer-reference sums: row 0 = sum x (2/sqrt3) sin theta,
    row 1 = sum x 2 cos theta -- the integer tables are derived from the oracle's own reference tables (and must be integers)."""
    import numpy as np
    den, num = ref["den"], ref["num"]
    if mode == "INT_REFS" and den in (3, 6) and not ref.get("phase") and not ref.get("phase_quarter"):
        sn, cs = oracle.ref_tables({"num": num, "den": den}, s_first, x.shape[0])
        wi, wq = sn * (2.0 / np.sqrt(3.0)), cs * 2.0
        assert np.abs(wi - np.rint(wi)).max() < 1e-12 and np.abs(wq - np.rint(wq)).max() < 1e-12
        I, Q = oracle.demod_int(x, np.rint(wi).astype(np.int64), np.rint(wq).astype(np.int64))
        return np.stack([I, Q])
    B = oracle.bins(x, num, den, s_first=s_first)
    return B[:den // 2] - B[den // 2:] if den % 2 == 0 else B
