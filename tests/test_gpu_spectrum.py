"""unknown-frequency search (qld_dominant_bin) against the oracle's series of QLDs, one per DFT bin
(PAPER.md:49).  The maximum amplitude must agree to 1e-6; the bin must agree wherever the answer is
unique, i.e. wherever the oracle's runner-up is not within the same 1e-6 of the maximum (a near-tie makes either bin a
correct answer; then the chosen bin's own amplitude is checked instead)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Q():
    import torch
    assert torch.cuda.is_available()
    from paper_1511_03390_b200 import qld
    qld.load_library()
    return qld


def _check(Q, oracle, x, q_lo, q_hi):
    import torch
    dev = torch.from_numpy(x.view(np.int16) if x.dtype == np.uint16 else x).cuda()
    amp, bins = Q.dominant_bin(dev, q_lo, q_hi)
    amp, bins = amp.cpu().numpy().astype(np.float64), bins.cpu().numpy()
    best, idx, second = oracle.dominant_bin(x, q_lo, q_hi, nthreads=oracle.max_threads())
    assert np.all(np.abs(amp - best) <= 1e-6 * best + 2.0 ** -23 * best), float(np.abs(amp - best).max())
    unique = second < best * (1.0 - 1e-6)
    assert np.array_equal(bins[unique], idx[unique])
    if (~unique).any():                                      # near-ties: the chosen bin must be (almost) as strong
        A = oracle.bin_amplitudes(x, q_lo, q_hi, nthreads=oracle.max_threads())
        chosen = np.take_along_axis(A, (bins - q_lo)[None].astype(np.int64), axis=0)[0]
        assert np.all(chosen[~unique] >= best[~unique] * (1.0 - 2e-6))
    assert bins.min() >= q_lo and bins.max() <= q_hi
    return bins


@pytest.mark.parametrize("H,W,N,dtype,q_lo,q_hi", [(16, 64, 64, np.uint16, 1, 31), (8, 48, 40, np.uint8, 1, 19), (12, 40, 96, np.uint16, 5, 17),
                                                   (3, 7, 32, np.uint8, 1, 15), (9, 16, 50, np.uint16, 24, 24)])
def test_dominant_bin_random_stacks(Q, oracle, H, W, N, dtype, q_lo, q_hi):
    """Every pass size (8 bins, a ragged last pass, a single bin), the tensor-core path and -- for a 21-byte frame --
    the FP32 fallback."""
    rng = np.random.default_rng(H * W + N)
    hi = 256 if dtype == np.uint8 else 4096
    x = rng.integers(0, hi, size=(N, H, W)).astype(dtype)
    _check(Q, oracle, x, q_lo, q_hi)


def test_dominant_bin_finds_each_source_of_the_paper_simulation(Q, oracle):
    """The five-source scene of PAPER.md:97 with frequencies that sit on bins of an N = 100 window (20, 23, 26, 29 Hz at
    100 frames/s): inside each modulated sub-region the dominant bin is that source's own frequency."""
    from paper_1511_03390_b200 import synth
    ps = synth.paper_sim(n=96, m=8, N=100, X=2.0)
    bins = _check(Q, oracle, ps.frames, 10, 40)
    for i, (y0, x0) in enumerate(ps.boxes[:4]):
        inside = bins[y0:y0 + ps.m, x0:x0 + ps.m]
        assert (inside == round(ps.nus[i] * 100)).mean() > 0.9, (i, np.bincount(inside.reshape(-1)))


def test_dominant_bin_rejects_bad_ranges(Q):
    import torch
    x = torch.zeros((32, 4, 16), dtype=torch.uint8, device="cuda")
    for lo, hi in ((0, 5), (5, 4), (1, 16)):
        with pytest.raises(Q.QLDError) as e:
            Q.dominant_bin(x, lo, hi)
        assert e.value.status == Q.QLD_E_INVAL


@pytest.mark.timeout(600, method="thread")
@pytest.mark.parametrize("H,W,N,dtype,q_lo,q_hi", [(64, 256, 256, np.uint16, 1, 127), (96, 128, 200, np.uint8, 1, 99), (40, 200, 130, np.uint16, 3, 64),
                                                   (128, 256, 520, np.uint16, 1, 70)])
def test_dominant_bin_many_passes(Q, oracle, H, W, N, dtype, q_lo, q_hi):
    """The 32-bins-per-pass tensor-core path: several passes (the running arg-max persists across launches), a ragged last
    pass, windows that are not a multiple of the 128-frame stage, more tiles than SMs, full-range samples."""
    rng = np.random.default_rng(N + q_hi)
    hi = 256 if dtype == np.uint8 else 65536
    x = rng.integers(0, hi, size=(N, H, W)).astype(dtype)
    # a few strong tones so that the answer is unique on part of the frame
    s = np.arange(1, N + 1)[:, None, None]
    for q in (q_lo, (q_lo + q_hi) // 2, q_hi):
        x[:, : H // 4, : W // 2] = np.clip(x[:, : H // 4, : W // 2].astype(np.int64) // 2 + (hi // 5) * (1 + np.sin(2 * np.pi * q * s / N)), 0, hi - 1).astype(dtype)
    _check(Q, oracle, x, q_lo, q_hi)


@pytest.mark.timeout(600, method="thread")
def test_dominant_bin_long_window_in_groups_of_passes(Q, oracle):
    """A long window: the digit tiles of a pass take 256 bytes per frame (2 MB at N = 8192), and they are built for at most
    64 MB worth of passes at a time -- 32 here -- so the 47 passes of bins 1..1500 run as two groups through one buffer; the
    running arg-max carries across the groups, and bins of the second group must win where they are the strongest."""
    rng = np.random.default_rng(8192)
    N, H, W = 8192, 4, 8
    x = rng.integers(0, 256, size=(N, H, W)).astype(np.uint8)
    s = np.arange(1, N + 1)[:, None]
    for col, q in enumerate((3, 700, 1023, 1024, 1025, 1400, 1500, 64)):       # one strong tone per column of the first row
        x[:, 0, col:col + 1] = np.clip(100 + 80 * np.sin(2 * np.pi * q * s / N + col), 0, 255).astype(np.uint8)
    bins = _check(Q, oracle, x, 1, 1500)
    assert list(bins[0]) == [3, 700, 1023, 1024, 1025, 1400, 1500, 64]
