"""Pins for the oracle's contrast-to-noise ratio (Eq. (1), Fig. 6).  The paper's own CNR values
(8.8 / 6.6) cannot be regenerated (frame size, source size, noise level and sampling interval are not
given): "parity unpinned" for those.  What the text fixes is pinned here: the geometry of Fig. 6, and closed forms."""
import numpy as np
import pytest


def test_fig6_geometry(oracle):
    # a 14 x 16 frame with a 4 x 4 source; the surround is "8 such 4x4 squares" = 8 m^2 = 128 pixels
    src, ring = oracle.cnr_regions(14, 16, 5, 6, 4)
    assert src.sum() == 16 and ring.sum() == 8 * 16 and not (src & ring).any()
    ys, xs = np.nonzero(src | ring)
    assert (ys.min(), ys.max(), xs.min(), xs.max()) == (1, 12, 2, 13)          # the 3m x 3m square, m pixels wide around the source
    # a one-pixel source: the surround is its 8 neighbours
    src, ring = oracle.cnr_regions(3, 3, 1, 1, 1)
    assert ring.sum() == 8 and src[1, 1] and not ring[1, 1]
    for bad in ((14, 16, 3, 6, 4), (14, 16, 5, 9, 4), (14, 16, 5, 6, 0)):     # slice leaves the frame / m < 1
        with pytest.raises(ValueError):
            oracle.cnr_regions(*bad)


def test_closed_forms(oracle):
    H, W, m, y0, x0 = 40, 48, 5, 12, 20
    src, ring = oracle.cnr_regions(H, W, y0, x0, m)
    img = np.full((H, W), 123.0)                        # pixels outside both regions must not matter
    img[src] = 9.0
    # surround alternates b +- d in equal numbers (8 m^2 is even): mean b, rms d  ->  CNR = (c - b) / d
    vals = np.where(np.arange(ring.sum()) % 2 == 0, 4.0 + 0.5, 4.0 - 0.5)
    img[ring] = vals
    c, ms, mr, rms = oracle.cnr(img, y0, x0, m)
    assert (ms, mr, rms) == (9.0, 4.0, 0.5) and c == 10.0
    # a source dimmer than its surround gives a negative CNR (numerator is signed in Eq. (1))
    img[src] = 3.0
    assert oracle.cnr(img, y0, x0, m)[0] == -2.0
    # affine invariance: CNR(a I + k) = CNR(I) for a > 0
    rng = np.random.default_rng(0)
    img = rng.normal(10.0, 2.0, size=(H, W))
    img[src] += 7.0
    base = oracle.cnr(img, y0, x0, m)[0]
    assert abs(oracle.cnr(3.5 * img + 11.0, y0, x0, m)[0] - base) < 1e-12 * abs(base)
    # a flat surround: IEEE division (inf), 0/0 -> nan
    flat = np.zeros((H, W)); flat[src] = 1.0
    assert oracle.cnr(flat, y0, x0, m)[0] == np.inf and np.isnan(oracle.cnr(np.zeros((H, W)), y0, x0, m)[0])


def test_gaussian_surround_statistics(oracle):
    # surround ~ N(b, sigma^2), source mean c: CNR -> (c - b) / sigma within sampling error (8 m^2 = 20000 samples)
    rng = np.random.default_rng(1)
    m = 50
    img = rng.normal(5.0, 2.0, size=(3 * m, 3 * m))
    img[m:2 * m, m:2 * m] = rng.normal(11.0, 2.0, size=(m, m))
    c = oracle.cnr(img, m, m, m)[0]
    assert abs(c - 3.0) < 0.06


def test_golden_fixture(oracle):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cnr_fig6.txt")
    n = 0
    for line in open(path):
        f = line.split("#")[0].split()
        if not f:
            continue
        if f[0] == "geom":
            H, W, y0, x0, m, ns, nr = (int(v) for v in f[1:8])
            src, ring = oracle.cnr_regions(H, W, y0, x0, m)
            assert (src.sum(), ring.sum()) == (ns, nr) == (m * m, 8 * m * m)
        else:
            c, b, d, exp = (float(v) for v in f[1:5])
            H, W, y0, x0, m = 20, 22, 6, 8, 4
            src, ring = oracle.cnr_regions(H, W, y0, x0, m)
            img = np.full((H, W), -7.0)
            img[src] = c
            img[ring] = np.where(np.arange(ring.sum()) % 2 == 0, b + d, b - d)
            assert oracle.cnr(img, y0, x0, m)[0] == exp
        n += 1
    assert n == 6
