"""Pins for the CPU oracle: closed forms, library routines, brute force -- never the oracle's own formula.

Each test names the mistake it would catch.  Citations: PAPER.md line numbers; readings G* in DESIGN.md.
"""
import math
import os
from fractions import Fraction

import mpmath
import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")


def _ref(nu=None, num=0, den=0, phase=0.0, pq=0):
    return {"nu": (num / den if den else nu), "num": num, "den": den, "phase": phase, "phase_quarter": pq}


def _golden():
    rows = []
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if not line:
            continue
        t = line.split()
        rows.append((t[0], int(t[1]), int(t[2]), int(t[3]), float(t[4]), float(t[5])))
    return rows


# ---------------------------------------------------------------- reference tables
def test_tables_quarter_period_exact(oracle):
    """nu = 1/4, s from 1: sin = 1,0,-1,0,...  cos = 0,-1,0,1,...; catches an s = 0 origin and libm residue."""
    sn, cs = oracle.ref_tables(_ref(num=1, den=4), 1, 8)
    assert sn.tolist() == [1, 0, -1, 0, 1, 0, -1, 0]
    assert cs.tolist() == [0, -1, 0, 1, 0, -1, 0, 1]
    sn, cs = oracle.ref_tables(_ref(num=1, den=4, pq=1), 1, 4)      # +pi/2: sin -> cos, cos -> -sin
    assert sn.tolist() == [0, -1, 0, 1] and cs.tolist() == [-1, 0, 1, 0]


def test_tables_sixth_period_exact_halves(oracle):
    sn, cs = oracle.ref_tables(_ref(num=1, den=6), 1, 6)
    h = math.sqrt(3.0) / 2.0
    assert cs.tolist() == [0.5, -0.5, -1.0, -0.5, 0.5, 1.0]
    assert np.allclose(sn, [h, h, 0, -h, -h, 0], rtol=0, atol=1e-16) and sn[2] == 0 and sn[5] == 0


@pytest.mark.parametrize("nu", [0.0937, 0.31830988618, 0.4999, 1.0 / 6.0])
def test_tables_real_vs_mpmath_large_s(oracle, nu):
    """Angle reduction must hold for frame indices deep into a long stream (cfg3: 16384; here up to 1e9)."""
    mpmath.mp.dps = 60
    for s0 in (1, 1000, 16384, 10 ** 6, 10 ** 9):
        sn, cs = oracle.ref_tables(_ref(nu=nu, phase=0.3), s0, 3)
        for i in range(3):
            turns = mpmath.mpf(Fraction(nu).numerator) / Fraction(nu).denominator * (s0 + i)
            th = 2 * mpmath.pi * (turns - mpmath.floor(turns)) + mpmath.mpf(0.3)
            assert abs(sn[i] - float(mpmath.sin(th))) < 4e-16
            assert abs(cs[i] - float(mpmath.cos(th))) < 4e-16


def test_tables_rational_equals_real_for_small_s(oracle):
    a = oracle.ref_tables(_ref(num=3, den=16), 1, 64)
    b = oracle.ref_tables(_ref(nu=3 / 16), 1, 64)
    assert np.allclose(a[0], b[0], atol=1e-15) and np.allclose(a[1], b[1], atol=1e-15)


def test_bin_index(oracle):
    assert oracle.bin_index(1, 6, 1, 8).tolist() == [1, 2, 3, 4, 5, 0, 1, 2]
    assert oracle.bin_index(5, 16, 3, 4).tolist() == [(5 * s) % 16 for s in range(3, 7)]


# ---------------------------------------------------------------- closed forms
def test_golden_closed_forms(oracle):
    for kind, N, num, den, level, expect in _golden():
        s = np.arange(1, N + 1, dtype=np.float64)
        for phi in (0.0, 0.7, 2.1, -1.3):
            if kind in ("tone", "norm"):
                x = level * np.sin(2 * np.pi * num * s / den + phi)
            else:
                x = np.full(N, level)
            if kind == "norm":
                # G3: the optional normalisation multiplies I, Q and R by 2/N, once each -- a scale that is dropped,
                # applied twice, or applied to R but not to I/Q fails here (R = A, not A*N/2 or 4A/N)
                I, Q, R, ph = oracle.qld(x[:, None], _ref(num=num, den=den), scale=2.0 / N)
                assert abs(R[0] - level) <= 1e-12 * level, (kind, N, R[0], level)
                assert abs(I[0] - level * math.cos(phi)) < 1e-12 and abs(Q[0] - level * math.sin(phi)) < 1e-12
                assert abs(math.remainder(ph[0] - phi, 2 * math.pi)) < 1e-12       # the phase does not depend on the scale
                I1, Q1 = oracle.demod(x[:, None], *oracle.ref_tables(_ref(num=num, den=den), 1, N))
                R2, ph2 = oracle.finalise(I1, Q1, scale=2.0 / N)                   # the same through finalise alone
                assert abs(R2[0] - level) <= 1e-12 * level and abs(math.remainder(ph2[0] - phi, 2 * math.pi)) < 1e-12
                continue
            I, Q, R, ph = oracle.qld(x[:, None], _ref(num=num, den=den))
            assert abs(R[0] - expect) <= 1e-11 * max(1.0, expect), (kind, N, num, den, phi, R[0], expect)
            if kind == "tone":   # G5: I = (AN/2) cos phi, Q = (AN/2) sin phi, phase map = phi
                assert abs(I[0] - expect * math.cos(phi)) < 1e-10 and abs(Q[0] - expect * math.sin(phi)) < 1e-10
                assert abs(math.remainder(ph[0] - phi, 2 * math.pi)) < 1e-12


def _G(u, N):
    """sum_{s=1..N} e^{ius} in closed form (geometric series)."""
    if abs(math.remainder(u, 2 * math.pi)) < 1e-15:
        return complex(N)
    return np.exp(1j * u * (N + 1) / 2) * math.sin(N * u / 2) / math.sin(u / 2)


@pytest.mark.parametrize("N,nu,nu_src,A,phi", [(1024, 0.0937, 0.0937, 5.0, 0.7), (1024, 0.0937, 0.0937, 5.0, 2.1),
                                              (82, 0.23, 0.31, 1.0, 0.4), (41, 0.23, 0.20, 1.0, 1.0), (257, 0.123, 0.4, 3.0, -2.0)])
def test_general_tone_closed_form(oracle, N, nu, nu_src, A, phi):
    """Z = Q + iI = sum x e^{i theta}; tone A sin(w's+phi):  Z = (A/2i)[e^{i phi} G(w+w') - e^{-i phi} G(w-w')].
    Covers non-integer N*nu (cfg2) and the paper's "incorrect frequency" leakage."""
    s = np.arange(1, N + 1, dtype=np.float64)
    x = A * np.sin(2 * np.pi * nu_src * s + phi)
    I, Q, R, _ = oracle.qld(x[:, None], _ref(nu=nu))
    w, ws = 2 * np.pi * nu, 2 * np.pi * nu_src
    Z = (A / 2j) * (np.exp(1j * phi) * _G(w + ws, N) - np.exp(-1j * phi) * _G(w - ws, N))
    assert abs(Q[0] - Z.real) < 1e-9 and abs(I[0] - Z.imag) < 1e-9 and abs(R[0] - abs(Z)) < 1e-9


def test_constant_background_leakage_cfg2(oracle):
    """G9: nothing is subtracted; D leaks as D |sin(pi N nu)/sin(pi nu)| when N*nu is not an integer."""
    mpmath.mp.dps = 40
    N, nu, D = 1024, 0.0937, 2000
    nu_x = mpmath.mpf(Fraction(nu).numerator) / Fraction(nu).denominator
    expect = float(D * abs(mpmath.sin(mpmath.pi * N * nu_x) / mpmath.sin(mpmath.pi * nu_x)))
    x = np.full((N, 1), D, dtype=np.uint16)
    _, _, R, _ = oracle.qld(x, _ref(nu=nu))
    assert abs(R[0] - expect) < 1e-9 and 1100 < expect < 1108        # SURVEY: about 0.552 * D


# ---------------------------------------------------------------- DFT identities
@pytest.mark.parametrize("dtype,N,shape", [(np.uint8, 16, (3, 5)), (np.uint16, 30, (2, 7)), (np.uint16, 64, (4, 3))])
def test_dft_bin_identity(oracle, dtype, N, shape):
    """nu = q/N: Z = e^{2 pi i q/N} conj(X[q]) with X = numpy.fft.fft along time; R = |X[q]| (the paper's FFT image)."""
    rng = np.random.default_rng(5)
    hi = 256 if dtype == np.uint8 else 4096
    x = rng.integers(0, hi, size=(N,) + shape).astype(dtype)
    X = np.fft.fft(x.astype(np.float64), axis=0)
    tot = 0.0
    for q in range(N):
        if q == 0:
            I, Q = oracle.demod(x, np.zeros(N), np.ones(N))
        else:
            I, Q, R, _ = oracle.qld(x, _ref(num=q, den=N))
        Z = np.exp(2j * np.pi * q / N) * np.conj(X[q])
        assert np.allclose(Q, Z.real, rtol=0, atol=1e-8) and np.allclose(I, Z.imag, rtol=0, atol=1e-8)
        tot = tot + I ** 2 + Q ** 2
    # Parseval: sum_q R_q^2 = N sum_s x_s^2
    assert np.allclose(tot, N * (x.astype(np.float64) ** 2).sum(axis=0), rtol=1e-12)


# ---------------------------------------------------------------- integer paths, brute force
def test_quarter_rate_brute_force_python_ints(oracle):
    """nu = 1/4, phase 0: I = sum_{s=1 mod 4} x - sum_{s=3 mod 4} x ; Q = sum_{s=0 mod 4} x - sum_{s=2 mod 4} x."""
    rng = np.random.default_rng(7)
    N, shape = 23, (3, 4)
    x = rng.integers(0, 65536, size=(N,) + shape).astype(np.uint16)
    sn, cs = oracle.ref_tables(_ref(num=1, den=4), 1, N)
    I, Q = oracle.demod_int(x, sn.astype(np.int64), cs.astype(np.int64))
    for j in range(shape[0]):
        for k in range(shape[1]):
            col = [int(v) for v in x[:, j, k]]
            bi = sum(col[s - 1] for s in range(1, N + 1) if s % 4 == 1) - sum(col[s - 1] for s in range(1, N + 1) if s % 4 == 3)
            bq = sum(col[s - 1] for s in range(1, N + 1) if s % 4 == 0) - sum(col[s - 1] for s in range(1, N + 1) if s % 4 == 2)
            assert int(I[j, k]) == bi and int(Q[j, k]) == bq
    # the float path on the same exact table must give the same integers
    If, Qf = oracle.demod(x, sn, cs)
    assert (If == I).all() and (Qf == Q).all()


def test_bins_brute_force_and_recombination(oracle):
    rng = np.random.default_rng(8)
    N, num, den = 50, 5, 12
    x = rng.integers(0, 4096, size=(N, 2, 3)).astype(np.uint16)
    B = oracle.bins(x, num, den, s_first=4)
    for r in range(den):
        ss = [i for i in range(N) if (num * (4 + i)) % den == r]
        assert (B[r] == x[ss].astype(np.int64).sum(axis=0)).all()
    assert (B.sum(axis=0) == x.astype(np.int64).sum(axis=0)).all()
    # S = sum_r B_r sin(2 pi r/den + phi) equals the direct sum
    I, Q, _, _ = oracle.qld(x, _ref(num=num, den=den, phase=0.4), s_first=4)
    r = np.arange(den)
    Ib = np.tensordot(np.sin(2 * np.pi * r / den + 0.4), B.astype(np.float64), axes=1)
    Qb = np.tensordot(np.cos(2 * np.pi * r / den + 0.4), B.astype(np.float64), axes=1)
    assert np.allclose(I, Ib, rtol=0, atol=1e-8) and np.allclose(Q, Qb, rtol=0, atol=1e-8)


# ---------------------------------------------------------------- structure: axes, linearity, invariances
def test_sixth_period_integer_references(oracle):
    """nu = 1/6 (BASELINE.json configs[3]) and nu = 1/3: (2/sqrt3) sin theta_s and 2 cos theta_s are integers, so two exact sums
    carry the whole result: 2Q = 2B0 + B1 - B2 - 2B3 - B4 + B5 and (2/sqrt3) I = B1 + B2 - B4 - B5 in terms of
    the phase bins -- brute force in Python integers, and against the float definition."""
    rng = np.random.default_rng(6)
    N = 61
    x = rng.integers(0, 65536, size=(N, 7)).astype(np.uint16)
    for den, s_first in ((6, 1), (6, 1000), (3, 5)):
        sn, cs = oracle.ref_tables(_ref(num=1, den=den), s_first, N)
        wi, wq = np.rint(sn * 2 / math.sqrt(3)).astype(np.int64), np.rint(cs * 2).astype(np.int64)
        assert np.abs(wi - sn * 2 / math.sqrt(3)).max() < 1e-15 and np.abs(wq - cs * 2).max() < 1e-15
        assert set(wi.tolist()) <= {-1, 0, 1} and set(np.abs(wq).tolist()) <= {1, 2}
        I2, Q2 = oracle.demod_int(x, wi, wq)
        for p in range(x.shape[1]):                                    # brute force, Python integers
            assert int(I2[p]) == sum(int(x[i, p]) * int(wi[i]) for i in range(N))
            assert int(Q2[p]) == sum(int(x[i, p]) * int(wq[i]) for i in range(N))
        B = oracle.bins(x, 1, den, s_first=s_first).astype(np.int64)
        if den == 6:
            assert np.array_equal(Q2, 2 * B[0] + B[1] - B[2] - 2 * B[3] - B[4] + B[5])
            assert np.array_equal(I2, B[1] + B[2] - B[4] - B[5])
        I, Q, _, _ = oracle.qld(x, _ref(num=1, den=den), s_first=s_first)
        assert np.allclose(I, I2 * (math.sqrt(3) / 2), rtol=1e-13, atol=1e-6) and np.allclose(Q, Q2 / 2, rtol=1e-13, atol=1e-6)


def test_pixel_axis_not_transposed(oracle):
    """Pixel p carries amplitude p+1 at its own phase; R[p] = (p+1) N/2.  A frame/pixel transposition or a
    wrong stride breaks this."""
    N, H, W = 48, 3, 5
    s = np.arange(1, N + 1, dtype=np.float64)[:, None, None]
    amp = (np.arange(H * W).reshape(H, W) + 1.0)[None]
    phi = (0.37 * np.arange(H * W).reshape(H, W))[None]
    x = amp * np.sin(2 * np.pi * s / 8 + phi)
    I, Q, R, ph = oracle.qld(x, _ref(num=1, den=8))
    assert R.shape == (H, W) and np.allclose(R, amp[0] * N / 2, atol=1e-10)
    assert np.allclose(np.remainder(ph - phi[0] + np.pi, 2 * np.pi) - np.pi, 0, atol=1e-12)


def test_linearity_and_multi_reference(oracle):
    rng = np.random.default_rng(9)
    N = 37
    x = rng.integers(0, 4096, (N, 6)).astype(np.float64)
    y = rng.integers(0, 4096, (N, 6)).astype(np.float64)
    r = _ref(nu=0.217, phase=0.2)
    Ix, Qx, _, _ = oracle.qld(x, r)
    Iy, Qy, _, _ = oracle.qld(y, r)
    Iz, Qz, _, _ = oracle.qld(2.5 * x - 0.5 * y, r)
    assert np.allclose(Iz, 2.5 * Ix - 0.5 * Iy, atol=1e-8) and np.allclose(Qz, 2.5 * Qx - 0.5 * Qy, atol=1e-8)
    multi = oracle.qld_multi(x, [r, _ref(nu=0.31)])
    assert np.array_equal(multi[0][0], Ix) and not np.allclose(multi[1][0], Ix)


def test_invariances(oracle):
    rng = np.random.default_rng(10)
    N, nu = 64, 0.0937
    x = rng.integers(0, 4096, (N, 9)).astype(np.uint16)
    I0, Q0, R0, _ = oracle.qld(x, _ref(nu=nu))
    # reference phase rotates (I, Q), leaves R: Z' = e^{i a} Z
    a = 0.9
    I1, Q1, R1, _ = oracle.qld(x, _ref(nu=nu, phase=a))
    Z0, Z1 = Q0 + 1j * I0, Q1 + 1j * I1
    assert np.allclose(R1, R0, rtol=1e-13) and np.allclose(Z1, np.exp(1j * a) * Z0, atol=1e-8)
    # index origin shift by m rotates by 2 pi nu m (G4, G10)
    m = 1000
    I2, Q2, R2, _ = oracle.qld(x, _ref(nu=nu), s_first=1 + m)
    assert np.allclose(R2, R0, rtol=1e-12) and np.allclose(Q2 + 1j * I2, np.exp(2j * np.pi * nu * m) * Z0, atol=1e-7)
    # real data: R(nu) = R(1 - nu)
    _, _, R3, _ = oracle.qld(x, _ref(nu=1 - nu))
    assert np.allclose(R3, R0, rtol=1e-12)


def test_degenerate_cases(oracle):
    x = np.array([[7, 200]], dtype=np.uint8)                      # N = 1: R = x_1 (G15)
    _, _, R, _ = oracle.qld(x, _ref(nu=0.0937))
    assert np.allclose(R, [7, 200], rtol=1e-15)
    z = np.zeros((16, 4), dtype=np.uint16)
    I, Q, R, ph = oracle.qld(z, _ref(num=1, den=8))
    assert not I.any() and not Q.any() and not R.any() and not ph.any()   # phase fixed to 0 at R = 0 (G16)
    sat = np.full((64, 4), 65535, dtype=np.uint16)                # saturated constant, N*nu integer: exactly 0
    sn, cs = oracle.ref_tables(_ref(num=1, den=4), 1, 64)
    I, Q = oracle.demod_int(sat, sn.astype(np.int64), cs.astype(np.int64))
    assert not I.any() and not Q.any()


def test_supplied_tables_half_rate_and_dc(oracle):
    """Reading G18: with caller-supplied tables the definition is computed whatever the arrays hold.  nu = 1/2: sin(pi s) = 0,
    cos(pi s) = (-1)^s, so a source A sin(pi s + phi) = A (-1)^s sin phi gives I = 0, Q = A N sin phi, R = A N |sin phi| --
    phase immunity is lost (why qld_create rejects nu = 1/2 without tables).  nu = 0: sin = 0, cos = 1: Q = sum x."""
    N, A = 64, 3.0
    s = np.arange(1, N + 1)
    alt = np.where(s % 2 == 0, 1.0, -1.0)
    for phi in (0.0, 0.4, 1.3, -2.0):
        x = (A * alt * math.sin(phi))[:, None]
        I, Q = oracle.demod(x, np.zeros(N), alt)
        R, _ = oracle.finalise(I, Q)
        assert I[0] == 0.0 and abs(Q[0] - A * N * math.sin(phi)) < 1e-12 and abs(R[0] - A * N * abs(math.sin(phi))) < 1e-12
    rng = np.random.default_rng(0)
    xi = rng.integers(0, 4096, size=(N, 5)).astype(np.uint16)
    I, Q = oracle.demod(xi, np.zeros(N), np.ones(N))
    assert np.array_equal(Q, xi.astype(np.int64).sum(axis=0)) and not I.any()


def test_sliding_is_window_by_window_definition(oracle):
    """Window w = absolute frames w*hop+1..w*hop+N, references by absolute index (G10): equals the
    window-relative result rotated by 2 pi nu w hop; amplitude equals the window-relative amplitude."""
    rng = np.random.default_rng(11)
    N, hop, T, nu = 16, 4, 40, 1.0 / 6.0
    stream = rng.integers(0, 4096, (T, 5)).astype(np.uint16)
    out = list(oracle.qld_sliding(stream, _ref(num=1, den=6), N, hop))
    assert [o[0] for o in out] == list(range((T - N) // hop + 1))
    for w, I, Q, R, _ in out:
        Ir, Qr, Rr, _ = oracle.qld(stream[w * hop:w * hop + N], _ref(num=1, den=6))
        assert np.allclose(R, Rr, rtol=1e-12)
        assert np.allclose(Q + 1j * I, np.exp(2j * np.pi * nu * w * hop) * (Qr + 1j * Ir), atol=1e-8)


def test_threads_do_not_change_results(oracle):
    rng = np.random.default_rng(12)
    x = rng.integers(0, 4096, (33, 101)).astype(np.uint16)
    a = oracle.qld(x, _ref(nu=0.21), nthreads=1)
    b = oracle.qld(x, _ref(nu=0.21), nthreads=3)
    assert all(np.array_equal(u, v) for u, v in zip(a, b))
