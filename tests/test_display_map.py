"""SURVEY.md 8(f3), second half: the headless stand-in for the paper's display step.  The mapping itself
is this build's reading (G22: linear min-max to 8 bits; the paper gives none -- "parity unpinned" against the
paper); the oracle's arithmetic is pinned by closed forms, the CUDA path must equal the oracle byte for byte."""
import numpy as np
import pytest


def test_oracle_closed_forms(oracle):
    ramp = np.arange(256, dtype=np.float32).reshape(16, 16) * 3.0 - 100.0          # 256 equally spaced levels
    out, lo, hi = oracle.display_map(ramp)
    assert (lo, hi) == (-100.0, 665.0) and np.array_equal(out.reshape(-1), np.arange(256))
    two = np.array([[5.0, 9.0], [9.0, 5.0]], dtype=np.float32)
    assert np.array_equal(oracle.display_map(two)[0], [[0, 255], [255, 0]])
    assert np.array_equal(oracle.display_map(np.array([0.0, 1.0, 2.0]))[0], [0, 128, 255])    # 127.5 rounds to even: 128
    assert not oracle.display_map(np.full((4, 4), 7.0))[0].any()                              # flat map
    withnan = np.array([np.nan, 1.0, 3.0, 2.0])
    out, lo, hi = oracle.display_map(withnan)
    assert (lo, hi) == (1.0, 3.0) and np.array_equal(out, [0, 0, 255, 128])
    # affine invariance of the image
    rng = np.random.default_rng(0)
    x = rng.normal(size=(32, 32))
    assert np.array_equal(oracle.display_map(x)[0], oracle.display_map(4.0 * x + 10.0)[0])


@pytest.mark.gpu
@pytest.mark.parametrize("shape", [(1, 1), (3, 7), (480, 640), (1024, 1280)])
def test_gpu_display_map_equals_oracle(oracle, shape):
    import torch
    from paper_1511_03390_b200 import qld
    rng = np.random.default_rng(shape[0])
    x = (rng.normal(1000.0, 300.0, size=shape) * rng.choice([1.0, -1.0], size=shape)).astype(np.float32)
    if x.size > 10:
        x.reshape(-1)[5] = np.nan
    out, r = qld.display_map(torch.from_numpy(x).cuda())
    eo, lo, hi = oracle.display_map(x)
    assert np.array_equal(out.cpu().numpy(), eo)
    if x.size > 1:
        assert tuple(r.cpu().numpy()) == (np.float32(lo), np.float32(hi))
    flat = torch.full(shape, 3.5, dtype=torch.float32, device="cuda")
    assert not qld.display_map(flat)[0].any()
