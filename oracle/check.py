"""Parity criterion for float maps -- TEST INFRASTRUCTURE, like the rest of oracle/.

Used by tests/, __graft_entry__.smoke() and bench.py's parity report (outside the timed region).  Compares maps a
caller obtained from anywhere with oracle maps; it holds no arithmetic of the method itself."""
import numpy as np

REL = 1e-5   # BASELINE.json north_star: "within 1e-5 relative (amplitude maps, fp32 accumulation)"


def check_float_maps(gpu, ora, rel=REL, what=""):
    """gpu, ora: (I, Q, amp, phase) arrays.  |d amp| <= rel*max(amp_or, median amp_or); I, Q likewise with
    max(|.|, median amp); phase: wrapped difference <= rel*max(1, median/amp_or) rad.  Returns the strict
    point-wise maximum relative amplitude error (reported, not gated)."""
    gI, gQ, gA, gP = [None if g is None else np.asarray(g, dtype=np.float64) for g in gpu]
    oI, oQ, oA, oP = [np.asarray(o, dtype=np.float64) for o in ora]
    med = float(np.median(oA))
    floor = med if med > 0 else 1.0
    f32 = 2.0 ** -23      # the maps are stored as float32: half an ulp of rounding on top of the bound
    if gA is not None:
        err = np.abs(gA - oA)
        bound = rel * np.maximum(oA, floor) + f32 * oA
        assert (err <= bound).all(), f"{what} amplitude: worst {float((err / np.maximum(oA, floor)).max()):.3e}"
    for g, o, nm in ((gI, oI, "I"), (gQ, oQ, "Q")):
        if g is not None:
            err = np.abs(g - o)
            bound = rel * np.maximum(np.abs(o), floor) + f32 * np.abs(o)
            assert (err <= bound).all(), f"{what} {nm}: worst {float((err / np.maximum(np.abs(o), floor)).max()):.3e}"
    if gP is not None:
        d = np.abs(np.remainder(gP - oP + np.pi, 2 * np.pi) - np.pi)
        bound = rel * np.maximum(1.0, floor / np.maximum(oA, 1e-300)) + 4 * f32
        ok = (d <= bound) | (oA == 0)
        assert ok.all(), f"{what} phase: worst {float(d.max()):.3e}"
    if gA is not None and (oA > 0).any():
        return float((np.abs(gA - oA)[oA > 0] / oA[oA > 0]).max())
    return 0.0
