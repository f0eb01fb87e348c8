"""CPU oracle for QLD (arXiv 1511.03390) -- TEST INFRASTRUCTURE, not part of the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may
import this package.  The arithmetic lives in qld_oracle.c (plain C, long double / int64, frame
order as in PAPER.md:169); this file is the ctypes marshalling around it plus the few lines that
express a sliding window and K references as repeated calls of the single-window definition
("sliding sequence"; "a series of QLDs ... at different frequencies").
It shares nothing with paper_1511_03390_b200/csrc and does not import the binding.

Beyond the hot path it also holds the oracles of the "next" rows: cnr / cnr_regions (Eq. (1),
PAPER.md:101-109), bin_amplitudes / dominant_bin and display_map, in plain numpy.
Parity unpinned (inputs or rule not given by the paper): the paper's CNR values 8.8 / 6.6 and the
display mapping (PAPER.md:169 names none; G22); everything else is pinned in tests/test_oracle_*.py.

Conventions: frame index s starts at 1; I = sum x sin
(in-phase, the reference sinusoid), Q = sum x cos (the 90-degree shifted one);
amplitude R = sqrt(I^2 + Q^2) with no normalisation; phase = atan2(Q, I).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qld_oracle.c")
_SO = os.path.join(_HERE, "libqld_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile qld_oracle.c with gcc (no fast-math: long double and rounding semantics matter)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", "-std=c11", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        l = C.CDLL(build())
        dp, i64, i32p, i64p, vp = C.POINTER(C.c_double), C.c_int64, C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.c_void_p
        l.qldo_ref_real.argtypes = [C.c_double, C.c_double, i64, i64, dp, dp]
        l.qldo_ref_real.restype = None
        l.qldo_ref_rational.argtypes = [i64, i64, i64, C.c_double, i64, i64, dp, dp]
        l.qldo_ref_rational.restype = None
        l.qldo_bin_index.argtypes = [i64, i64, i64, i64, i32p]
        l.qldo_bin_index.restype = None
        l.qldo_demod_f64.argtypes = [vp, C.c_int, i64, i64, i64, dp, dp, dp, dp, C.c_int]
        l.qldo_demod_i64.argtypes = [vp, C.c_int, i64, i64, i64, i64p, i64p, i64p, i64p, C.c_int]
        l.qldo_bins_i64.argtypes = [vp, C.c_int, i64, i64, i64, i32p, i64, i64p]
        l.qldo_finalise.argtypes = [dp, dp, i64, C.c_double, dp, dp]
        l.qldo_finalise.restype = None
        l.qldo_max_threads.restype = C.c_int
        _lib = l
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


_DT = {np.dtype(np.uint8): 0, np.dtype(np.uint16): 1, np.dtype(np.float64): 2}


def max_threads() -> int:
    return int(lib().qldo_max_threads())


def ref_tables(ref: dict, s_first: int, n: int) -> Tuple[np.ndarray, np.ndarray]:
    """sin(theta_s), cos(theta_s) for s = s_first .. s_first+n-1 as float64 arrays.

    ref = {"nu": float, "num": int, "den": int, "phase": float, "phase_quarter": int}; den > 0
    means nu == num/den exactly (angles reduced in integers)."""
    sn = np.empty(n, dtype=np.float64)
    cs = np.empty(n, dtype=np.float64)
    den = int(ref.get("den", 0) or 0)
    if den > 0:
        lib().qldo_ref_rational(int(ref["num"]), den, int(ref.get("phase_quarter", 0)), float(ref.get("phase", 0.0)),
                                int(s_first), int(n), _dp(sn), _dp(cs))
    else:
        ph = float(ref.get("phase", 0.0)) + int(ref.get("phase_quarter", 0)) * (np.pi / 2)
        lib().qldo_ref_real(float(ref["nu"]), ph, int(s_first), int(n), _dp(sn), _dp(cs))
    return sn, cs


def _as_stack(frames: np.ndarray) -> Tuple[np.ndarray, int, int]:
    f = np.ascontiguousarray(frames)
    if f.dtype not in _DT:
        raise TypeError(f"unsupported dtype {f.dtype}")
    n = f.shape[0]
    hw = int(np.prod(f.shape[1:])) if f.ndim > 1 else 1
    return f.reshape(n, hw), n, hw


def demod(frames: np.ndarray, sin_tab: np.ndarray, cos_tab: np.ndarray, nthreads: int = 1):
    """I = sum_s x_s sin_s, Q = sum_s x_s cos_s per pixel (float64), for one window.

    frames: [N, ...pixels]; tables: length N (entry i belongs to frames[i])."""
    f, n, hw = _as_stack(frames)
    assert len(sin_tab) == n and len(cos_tab) == n
    sn = np.ascontiguousarray(sin_tab, dtype=np.float64)
    cs = np.ascontiguousarray(cos_tab, dtype=np.float64)
    I = np.empty(hw, dtype=np.float64)
    Q = np.empty(hw, dtype=np.float64)
    rc = lib().qldo_demod_f64(f.ctypes.data, _DT[f.dtype], n, hw, hw, _dp(sn), _dp(cs), _dp(I), _dp(Q), int(nthreads))
    assert rc == 0
    return I.reshape(frames.shape[1:]), Q.reshape(frames.shape[1:])


def demod_int(frames: np.ndarray, isin: Sequence[int], icos: Sequence[int], nthreads: int = 1):
    """The same sums with integer-valued reference tables, exact in int64."""
    f, n, hw = _as_stack(frames)
    a = np.ascontiguousarray(isin, dtype=np.int64)
    b = np.ascontiguousarray(icos, dtype=np.int64)
    assert len(a) == n and len(b) == n
    I = np.empty(hw, dtype=np.int64)
    Q = np.empty(hw, dtype=np.int64)
    p = C.POINTER(C.c_int64)
    rc = lib().qldo_demod_i64(f.ctypes.data, _DT[f.dtype], n, hw, hw, a.ctypes.data_as(p), b.ctypes.data_as(p),
                              I.ctypes.data_as(p), Q.ctypes.data_as(p), int(nthreads))
    assert rc == 0
    return I.reshape(frames.shape[1:]), Q.reshape(frames.shape[1:])


def bin_index(num: int, den: int, s_first: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.int32)
    lib().qldo_bin_index(int(num), int(den), int(s_first), int(n), out.ctypes.data_as(C.POINTER(C.c_int32)))
    return out


def bins(frames: np.ndarray, num: int, den: int, s_first: int = 1) -> np.ndarray:
    """Phase-bin sums B[r] = sum_{s: (num*s mod den) == r} x_s, int64 [den, ...pixels]."""
    f, n, hw = _as_stack(frames)
    idx = bin_index(num, den, s_first, n)
    B = np.empty((den, hw), dtype=np.int64)
    rc = lib().qldo_bins_i64(f.ctypes.data, _DT[f.dtype], n, hw, hw, idx.ctypes.data_as(C.POINTER(C.c_int32)),
                             int(den), B.ctypes.data_as(C.POINTER(C.c_int64)))
    assert rc == 0
    return B.reshape((den,) + tuple(frames.shape[1:]))


def finalise(I: np.ndarray, Q: np.ndarray, scale: float = 1.0):
    """amplitude = scale * sqrt(I^2 + Q^2), phase = atan2(Q, I) (0 where I = Q = 0)."""
    i = np.ascontiguousarray(I, dtype=np.float64).reshape(-1)
    q = np.ascontiguousarray(Q, dtype=np.float64).reshape(-1)
    R = np.empty_like(i)
    ph = np.empty_like(i)
    lib().qldo_finalise(_dp(i), _dp(q), i.size, float(scale), _dp(R), _dp(ph))
    return R.reshape(np.shape(I)), ph.reshape(np.shape(I))


def qld(frames: np.ndarray, ref: dict, s_first: int = 1, nthreads: int = 1, scale: float = 1.0):
    """One window, one reference: returns (I, Q, amplitude, phase); frames[i] is frame s_first+i."""
    sn, cs = ref_tables(ref, s_first, frames.shape[0])
    I, Q = demod(frames, sn, cs, nthreads)
    R, ph = finalise(I, Q, scale)
    return I * scale, Q * scale, R, ph


def qld_multi(frames: np.ndarray, refs: Sequence[dict], s_first: int = 1, nthreads: int = 1):
    """K references = K independent single-reference QLDs (reading G13)."""
    return [qld(frames, r, s_first, nthreads) for r in refs]


def qld_sliding(stream: np.ndarray, ref: dict, N: int, hop: int, nthreads: int = 1, windows: Optional[Sequence[int]] = None):
    """Sliding sequence: window w covers absolute frames w*hop+1 .. w*hop+N and is
    recomputed from the definition every time, references indexed by absolute frame number
    (reading G10).  stream[i] is frame i+1.  Yields (w, I, Q, amplitude, phase)."""
    n_win = (stream.shape[0] - N) // hop + 1
    for w in (range(n_win) if windows is None else windows):
        a = w * hop
        yield (w,) + qld(stream[a:a + N], ref, s_first=a + 1, nthreads=nthreads)


# ---------------------------------------------------------------------------------------------------
# Contrast-to-noise ratio (Eq. (1), Fig. 6) -- SURVEY.md 8(f1), the step after the path
# ---------------------------------------------------------------------------------------------------
def cnr_regions(H: int, W: int, y0: int, x0: int, m: int):
    """Boolean masks (source, surround) of Fig. 6: the m x m source square with top-left corner
    (y0, x0) and the m-pixel wide square slice around it, i.e. the 3m x 3m square minus the source: 8 m^2 pixels
    (PAPER.md:109).  The slice must lie inside the frame."""
    if m < 1 or y0 - m < 0 or x0 - m < 0 or y0 + 2 * m > H or x0 + 2 * m > W:
        raise ValueError("cnr: the surrounding slice must lie inside the frame")
    src = np.zeros((H, W), dtype=bool)
    big = np.zeros((H, W), dtype=bool)
    src[y0:y0 + m, x0:x0 + m] = True
    big[y0 - m:y0 + 2 * m, x0 - m:x0 + 2 * m] = True
    return src, big & ~src


def cnr(image: np.ndarray, y0: int, x0: int, m: int):
    """Eq. (1): CNR = (mean_s - mean_surr) / sqrt(mean over the slice of (I(j,k) - mean_surr)^2), fp64, term by term
    as printed.  Returns (cnr, mean_s, mean_surr, rms); IEEE semantics when the slice is flat (rms = 0)."""
    img = np.asarray(image, dtype=np.float64)
    src, ring = cnr_regions(img.shape[0], img.shape[1], y0, x0, m)
    mean_s = img[src].sum() / float(m * m)
    r = img[ring]
    mean_surr = r.sum() / float(8 * m * m)
    rms = np.sqrt(((r - mean_surr) ** 2).sum() / float(8 * m * m))
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = np.float64(mean_s - mean_surr) / np.float64(rms)
    return float(ratio), float(mean_s), float(mean_surr), float(rms)


# ---------------------------------------------------------------------------------------------------
# Unknown-frequency search -- SURVEY.md 8(f2), the step before the path
# ---------------------------------------------------------------------------------------------------
def bin_amplitudes(frames: np.ndarray, q_lo: int, q_hi: int, nthreads: int = 1) -> np.ndarray:
    """R_q for every DFT bin q = q_lo..q_hi of the N-frame stack: one QLD per bin at nu = q/N ("a series
    of QLDs ... at different frequencies"), each from the definition.  Returns [q_hi - q_lo + 1, ...pixels] float64."""
    N = frames.shape[0]
    if q_lo < 1 or q_hi < q_lo or 2 * q_hi >= N:
        raise ValueError("bins must satisfy 1 <= q_lo <= q_hi < N/2")
    return np.stack([qld(frames, {"num": q, "den": N}, nthreads=nthreads)[2] for q in range(q_lo, q_hi + 1)])


def dominant_bin(frames: np.ndarray, q_lo: int, q_hi: int, nthreads: int = 1):
    """Per pixel: the largest R_q over the bins and its bin (the lowest bin on a tie).  Also returns the runner-up
    amplitude so that a caller can tell near-ties (where another bin is an equally valid answer)."""
    A = bin_amplitudes(frames, q_lo, q_hi, nthreads)
    idx = np.argmax(A, axis=0)
    best = np.take_along_axis(A, idx[None], axis=0)[0]
    if A.shape[0] > 1:
        second = np.partition(A, -2, axis=0)[-2]
    else:
        second = np.zeros_like(best)
    return best, (idx + q_lo).astype(np.int32), second


# ---------------------------------------------------------------------------------------------------
# Display mapping -- SURVEY.md 8(f3), the step after the path; the paper does not say how the 32-bit
# image is mapped to the screen: linear min-max to 8 bits is this build's reading (G22): "parity unpinned"
# against the paper, pinned against the arithmetic below by closed forms.
# ---------------------------------------------------------------------------------------------------
def display_map(image: np.ndarray):
    """u8 = rint(255 (x - lo) / (hi - lo)) with lo, hi the smallest / largest non-NaN value; zeros for a flat map and
    for NaNs.  Returns (u8 image, lo, hi)."""
    x = np.asarray(image, dtype=np.float64)
    ok = ~np.isnan(x)
    lo, hi = (float(x[ok].min()), float(x[ok].max())) if ok.any() else (np.inf, -np.inf)
    out = np.zeros(x.shape, dtype=np.uint8)
    if hi > lo:
        with np.errstate(invalid="ignore"):
            t = np.rint(255.0 * (x - lo) / (hi - lo))
        out[ok] = np.clip(t[ok], 0, 255).astype(np.uint8)
    return out, lo, hi
