"""Pins for the oracle's all-bin search: the bins are the DFT of the series (the
Fourier decomposition "is essentially a series of QLDs"; the FFT image |F|^2), so numpy's FFT -- a
different algorithm -- must agree, and a tone sitting on a bin must be found there."""
import numpy as np


def test_bins_equal_the_fft_of_the_series(oracle):
    rng = np.random.default_rng(3)
    N, H, W = 48, 5, 7
    x = rng.integers(0, 4096, size=(N, H, W)).astype(np.uint16)
    A = oracle.bin_amplitudes(x, 1, N // 2 - 1)
    F = np.abs(np.fft.rfft(x.astype(np.float64), axis=0))[1:N // 2]          # R_q = |X[q]| (DFT-bin identity)
    assert A.shape == F.shape and np.allclose(A, F, rtol=1e-11, atol=1e-7)
    best, idx, second = oracle.dominant_bin(x, 1, N // 2 - 1)
    assert np.array_equal(idx, np.argmax(F, axis=0) + 1) and np.allclose(best, F.max(axis=0), rtol=1e-11)
    assert (second <= best).all()
    # a sub-range of bins
    b2, i2, _ = oracle.dominant_bin(x, 5, 9)
    assert np.array_equal(i2, np.argmax(F[4:9], axis=0) + 5)


def test_a_tone_on_a_bin_is_found_there(oracle):
    N, q0 = 64, 11
    s = np.arange(1, N + 1)
    amp = np.array([[3.0, 10.0], [40.0, 7.5]])
    x = 100.0 + amp[None] * np.sin(2 * np.pi * q0 * s / N + 0.4)[:, None, None]
    best, idx, second = oracle.dominant_bin(x, 1, N // 2 - 1)
    assert (idx == q0).all()
    assert np.allclose(best, amp * N / 2, rtol=1e-12)                         # R = A N / 2 on the bin
    assert (second < 1e-9 * best).all()                                      # exact orthogonality of the other bins
