"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (frames filled on the device,
attached in place, accumulation chosen by AUTO unless stated): sampled pixels -- random ones plus the pixels with
the strongest modulation -- are recomputed one by one by the oracle from the seeded generator (synth.series)."""
import numpy as np
import pytest

from _parity import check_float_maps

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Q():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1511_03390_b200 import qld
    qld.load_library()
    return qld


def _sample_pixels(scene, n_random=1500, n_strong=300, seed=0):
    rng = np.random.default_rng(seed)
    pix = set(rng.integers(0, scene.HW, size=n_random).tolist())
    pix.update([0, scene.W - 1, scene.HW - scene.W, scene.HW - 1])            # corners: first / last tile, ragged ends
    if scene.weights.shape[0]:
        strength = np.abs(scene.weights).sum(axis=0)
        pix.update(np.argsort(strength)[-n_strong:].tolist())
    return np.array(sorted(pix), dtype=np.int64)


def _oracle_on_pixels(oracle, scene, pix, ref, s_first, N):
    from paper_1511_03390_b200 import synth
    x = synth.series(scene, pix, s_first, N).reshape(N, 1, len(pix))
    return x, tuple(m.reshape(-1) for m in oracle.qld(x, ref, s_first=s_first, nthreads=oracle.max_threads()))


def _gpu_on_pixels(ctx, k, pix):
    import torch
    idx = torch.from_numpy(pix).cuda()
    return tuple(None if m is None else m.reshape(-1)[idx].cpu().numpy() for m in ctx.get_maps(k))


@pytest.mark.parametrize("name,accum_name,kernel", [("cfg1", "AUTO", "k_demod_stream"), ("cfg1", "FP32", "k_demod_stream"),
                                                   ("cfg2", "AUTO", "k_demod_stream"), ("cfg2", "FIXED", "k_demod_tc"),
                                                   ("cfg4", "AUTO", "k_demod_tc"), ("cfg4", "FP32", "k_demod_stream"), ("cfg4", "FIXED", "k_demod_tc")])
def test_whole_window_full_size_sampled(Q, oracle, name, accum_name, kernel):
    import torch
    from paper_1511_03390_b200 import synth
    wl = synth.BUILDERS[name]()
    sc, N, K = wl.scene, wl.N, len(wl.refs)
    refs = [dict(r) for r in wl.refs]
    frames = Q.synth_fill(sc, 1, N)
    ctx = Q.QLD(sc.H, sc.W, sc.dtype, N, refs, ring_frames=-1, accum=getattr(Q, "QLD_ACC_" + accum_name), max_value=sc.maxval)
    ctx.attach_frames_device(frames)
    ctx.demod(Q.QLD_WHOLE)
    ctx.sync()
    if kernel:
        assert ctx.last_kernel() == kernel
    mode = ctx.accum_name()
    pix = _sample_pixels(sc, n_random=1500 if K == 1 else 400, n_strong=300 if K == 1 else 200)
    for k in range(K):
        x, ora = _oracle_on_pixels(oracle, sc, pix, refs[k], 1, N)
        # the generator's device twin wrote exactly these bytes
        raw = frames.view(torch.int16) if frames.dtype == torch.uint16 else frames      # uint16 has no CUDA index kernel
        got_bytes = raw.reshape(N, -1)[:, torch.from_numpy(pix).cuda()].cpu().numpy().view(x.dtype)
        assert np.array_equal(got_bytes.reshape(x.shape), x)
        got = _gpu_on_pixels(ctx, k, pix)
        # the floor of the tolerance is the median amplitude of the sampled pixels (background-dominated, as the map's)
        check_float_maps(got, ora, rel=1e-6 if mode in ("INT_BINS", "FIXED") else 1e-5, what=f"{name} {mode} k={k}")
        if mode == "INT_BINS" and k == 0:
            den = refs[0]["den"]
            B = oracle.bins(x, refs[0]["num"], den)
            rows = ctx.get_bins(0).reshape(den // 2, -1)[:, torch.from_numpy(pix).cuda()].cpu().numpy()
            assert np.array_equal(rows.reshape(den // 2, 1, -1), B[:den // 2] - B[den // 2:])
    ctx.destroy()
    del frames
    torch.cuda.empty_cache()


@pytest.mark.parametrize("slide_hop", [0, 32])
@pytest.mark.parametrize("accum_name", ["AUTO", "FP32"])
def test_sliding_full_size_sampled(Q, oracle, accum_name, slide_hop):
    """cfg3's frame size, window, hop and batch; the first 12 hops of the stream, zero-copy ring as in bench.py."""
    import torch
    from paper_1511_03390_b200 import synth
    wl = synth.cfg3()
    sc, N, hop = wl.scene, wl.N, wl.hop
    ref = dict(wl.refs[0])
    n_hops = 12
    T = N + n_hops * hop
    ring = torch.empty((T, sc.H, sc.W), dtype=torch.uint16, device="cuda")
    for a in range(0, T, 128):
        Q.synth_fill(sc, a + 1, min(128, T - a), out=ring[a:a + 128])
    ctx = Q.QLD(sc.H, sc.W, sc.dtype, N, [ref], ring_frames=T, accum=getattr(Q, "QLD_ACC_" + accum_name), max_value=sc.maxval,
                external_store=True, slide_hop=slide_hop)
    ctx.attach_frames_device(ring)
    ctx.commit_frames(N)
    ctx.demod(Q.QLD_SLIDE, hop)
    rng = np.random.default_rng(3)
    # random pixels plus pixels on the path of the moving disk (rows around H/2)
    pix = np.unique(np.concatenate([rng.integers(0, sc.HW, size=600),
                                    (sc.H // 2 + rng.integers(-30, 31, size=600)) * sc.W + rng.integers(0, sc.W, size=600)]))
    for w in range(n_hops + 1):
        if w > 0:
            ctx.commit_frames(hop)
            ctx.demod(Q.QLD_SLIDE, hop)
            assert ctx.last_kernel() == "k_demod_stream"
        if w in (0, 1, 5, n_hops):
            ctx.sync()
            x, ora = _oracle_on_pixels(oracle, sc, pix, ref, w * hop + 1, N)
            got = _gpu_on_pixels(ctx, 0, pix)
            check_float_maps(got, ora, rel=1e-6 if ctx.accum_name() == "INT_BINS" else 1e-5, what=f"cfg3 window {w}")
            if ctx.accum_name() == "INT_BINS":
                B = oracle.bins(x, 1, 6, s_first=w * hop + 1)
                rows = ctx.get_bins(0).reshape(3, -1)[:, torch.from_numpy(pix).cuda()].cpu().numpy()
                assert np.array_equal(rows.reshape(3, 1, -1), B[:3] - B[3:]), f"window {w}"
    ctx.destroy()
