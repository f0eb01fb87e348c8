"""qld_dominant_bin_static: the unknown-frequency search for callers that cannot
allocate device memory.

Two kinds of caller are meant.  A live acquisition loop (the paper's real-time threads) cannot afford
cudaMalloc / cudaFree between two frame batches: both take a driver-wide lock and may wait for all work on the device, which
stalls the copy stream that is bringing in the next batch.  And a process in which something else -- a framework's caching
allocator, another library -- already holds all of HBM has no memory left for the pool allocation qld_dominant_bin makes for
its digit tiles.  qld_dominant_bin_static keeps those tiles (and its two tile counters) in a fixed 4 MiB array that is part
of the library image instead, so it allocates nothing, at the price of a size limit and of one search at a time per device.

What is checked here: on two calls in a row -- the second with a different window length, bin range, sample type and frame
size, so that it runs over whatever the first call left in the shared array -- the maps equal those of the existing
qld_dominant_bin path (same kernels, same digits: the amplitude is held to the 1e-6 of tests/test_gpu_spectrum.py and in fact
agrees to the bit, the bins exactly); a repeated call leaves the device's free memory where it was; a search beyond the 4 MiB
limit and a frame size the tensor-core route cannot take are refused with a message that says why.

This file is named to be collected last (`pytest --collect-only`): with `-x` a failure here hides no other test.  It does
not depend on what ran before it: the first call on a device looks the array's address up by itself."""
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


def _stack(N, H, W, dtype, q_tones, seed):
    """Random full-range frames with a few strong tones on part of the frame (so that the arg-max is not noise everywhere)."""
    rng = np.random.default_rng(seed)
    hi = 256 if dtype == np.uint8 else 65536
    x = rng.integers(0, hi, size=(N, H, W)).astype(dtype)
    s = np.arange(1, N + 1)[:, None, None]
    for i, q in enumerate(q_tones):
        r0 = i * (H // len(q_tones))
        block = x[:, r0:r0 + H // (2 * len(q_tones)), : W // 2].astype(np.int64) // 2
        x[:, r0:r0 + H // (2 * len(q_tones)), : W // 2] = np.clip(block + (hi // 5) * (1 + np.sin(2 * np.pi * q * s / N)), 0, hi - 1).astype(dtype)
    return x


def _same_as_existing_path(Q, x, q_lo, q_hi):
    import torch
    dev = torch.from_numpy(x.view(np.int16) if x.dtype == np.uint16 else x).cuda()
    amp = torch.full(x.shape[1:], -7.0, dtype=torch.float32, device="cuda")          # caller-owned outputs, prefilled with junk
    bins = torch.full(x.shape[1:], -7, dtype=torch.int32, device="cuda")
    Q.dominant_bin_static(dev, q_lo, q_hi, amp=amp, bins=bins)
    ref_amp, ref_bins = Q.dominant_bin(dev, q_lo, q_hi)
    torch.cuda.synchronize()
    a, b = amp.cpu().numpy().astype(np.float64), ref_amp.cpu().numpy().astype(np.float64)
    assert np.all(np.abs(a - b) <= 1e-6 * b), float(np.abs(a - b).max())            # tolerance of tests/test_gpu_spectrum.py
    assert np.array_equal(amp.cpu().numpy(), ref_amp.cpu().numpy())                  # and, the kernels being the same, to the bit
    assert np.array_equal(bins.cpu().numpy(), ref_bins.cpu().numpy())
    assert int(bins.min()) >= q_lo and int(bins.max()) <= q_hi
    return dev, amp, bins


def test_static_scratch_search_equals_the_allocating_one_on_two_calls_in_a_row(Q):
    import torch
    lib = Q.load_library()
    # call 1: five passes of 32 bins over a 520-frame window (a ragged last 128-frame stage), more tiles than SMs: 0.8 MB of digits
    N1, lo1, hi1 = 520, 1, 150
    assert lib.qld_dominant_bin_static_bytes(N1, lo1, hi1) == 256 * 640 * 5
    _same_as_existing_path(Q, _stack(N1, 128, 256, np.uint16, (3, 77, 150), seed=11), lo1, hi1)
    # call 2, straight after: shorter window, fewer bins, bytes instead of words, another frame size -- it uses the front of
    # the array the first call filled and must not see any of it
    N2, lo2, hi2 = 200, 7, 60
    dev, amp, bins = _same_as_existing_path(Q, _stack(N2, 96, 112, np.uint8, (7, 33), seed=12), lo2, hi2)
    # a repeat of call 2 with the same caller-owned outputs: same maps again, and the device's free memory does not move
    keep_amp, keep_bins = amp.clone(), bins.clone()
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    Q.dominant_bin_static(dev, lo2, hi2, amp=amp, bins=bins)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    assert torch.equal(amp, keep_amp) and torch.equal(bins, keep_bins)


def test_static_scratch_search_refuses_what_does_not_fit(Q):
    import torch
    lib = Q.load_library()
    # all 1023 bins of an N = 2048 window need 16 MiB of digit tiles: over the 4 MiB the library holds
    assert lib.qld_dominant_bin_static_bytes(2048, 1, 1023) == 16 << 20 > Q.QLD_SEARCH_STATIC_BYTES
    x = torch.zeros((2048, 8, 32), dtype=torch.uint8, device="cuda")
    with pytest.raises(Q.QLDError) as e:
        Q.dominant_bin_static(x, 1, 1023)
    assert e.value.status == Q.QLD_E_NOMEM and "QLD_SEARCH_STATIC_BYTES" in str(e.value)
    # ... while a quarter of the bins of the same window fits exactly (4 MiB) and agrees with the allocating path
    assert lib.qld_dominant_bin_static_bytes(2048, 1, 256) == Q.QLD_SEARCH_STATIC_BYTES
    a, b = Q.dominant_bin_static(x, 1, 256)
    ra, rb = Q.dominant_bin(x, 1, 256)
    assert torch.equal(a, ra) and torch.equal(b, rb)
    # a 21-byte frame would need qld_dominant_bin's context route, which allocates: refused, with the reason
    y = torch.zeros((32, 3, 7), dtype=torch.uint8, device="cuda")
    with pytest.raises(Q.QLDError) as e:
        Q.dominant_bin_static(y, 1, 15)
    assert e.value.status == Q.QLD_E_UNSUPPORTED and "16" in str(e.value)
    # bad ranges as in qld_dominant_bin
    for lo, hi in ((0, 5), (5, 4), (1, 16)):
        with pytest.raises(Q.QLDError) as e:
            Q.dominant_bin_static(torch.zeros((32, 4, 16), dtype=torch.uint8, device="cuda"), lo, hi)
        assert e.value.status == Q.QLD_E_INVAL
    assert lib.qld_dominant_bin_static_bytes(32, 1, 16) == Q.QLD_E_INVAL
    # a success clears the message
    Q.dominant_bin_static(torch.zeros((32, 8, 32), dtype=torch.uint8, device="cuda"), 1, 15)
    assert lib.qld_dominant_bin_static_error() == b""
