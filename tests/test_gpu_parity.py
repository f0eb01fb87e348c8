"""GPU parity: the CUDA path behind the C ABI against the CPU oracle, element by element, on the same bytes.

Bars (BASELINE.json north_star): integer paths bit-exact; float paths within 1e-5 relative (floored at the
map median).  Every call goes through paper_1511_03390_b200.qld (ctypes -> libqld.so).
"""
import numpy as np
import pytest

from _parity import check_float_maps, expected_int_rows, forced, oracle_maps

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Q():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1511_03390_b200 import qld
    qld.load_library()          # raises if libqld.so is missing: no fallback
    return qld


def _maps(ctx, k=0):
    return tuple(None if m is None else m.cpu().numpy() for m in ctx.get_maps(k))


def _rand_stack(rng, N, H, W, dtype, hi=None):
    hi = hi or (256 if dtype == np.uint8 else 4096)
    base = rng.integers(hi // 4, hi // 2, size=(1, H, W))
    return np.clip(base + rng.normal(0, hi / 64, size=(N, H, W)), 0, hi - 1).astype(dtype)


# ------------------------------------------------------------------------------------------------ A1
@pytest.mark.parametrize("ref", [{"nu": 0.0937}, {"nu": 0.31, "phase": 1.1}, {"num": 1, "den": 6},
                                 {"num": 3, "den": 16, "phase_quarter": 1}])
def test_reference_tables_match_oracle(Q, oracle, ref):
    N = 300
    ctx = Q.QLD(4, 4, "u16", N, [ref], accum=Q.QLD_ACC_FP32)
    sn, cs = ctx.read_ref_table(0, 1, N)
    osn, ocs = oracle.ref_tables(ref, 1, N)
    # fp64 sincospi of an exactly reduced angle, rounded once to fp32: at most 1 ulp from the rounded oracle value
    assert np.abs(sn.astype(np.float64) - osn).max() <= 2.0 ** -24 * 1.01
    assert np.abs(cs.astype(np.float64) - ocs).max() <= 2.0 ** -24 * 1.01
    assert (sn == osn.astype(np.float32)).mean() > 0.99 and (cs == ocs.astype(np.float32)).mean() > 0.99
    ctx.destroy()


def test_reference_tables_deep_in_a_stream(Q, oracle):
    """Ring context: tables are filled per push by absolute frame index; check around frame 10^5."""
    N, cap, H, W = 8, 64, 2, 8
    ref = {"nu": 0.0937, "phase": 0.2}
    ctx = Q.QLD(H, W, "u16", N, [ref], ring_frames=cap, accum=Q.QLD_ACC_FP32)
    z = np.zeros((32, H, W), np.uint16)
    pushed = 0
    while pushed < 100000:
        ctx.push_frames(z)
        pushed += 32
        if pushed % 32 == 0:
            ctx.demod(Q.QLD_WHOLE)
    ctx.sync()
    sn, cs = ctx.read_ref_table(0, pushed - 31, 32)
    osn, ocs = oracle.ref_tables(ref, pushed - 31, 32)
    assert np.abs(sn - osn).max() < 1e-7 and np.abs(cs - ocs).max() < 1e-7
    ctx.destroy()


# ------------------------------------------------------------------------------------------------ A3 / A4 / A6
@pytest.mark.parametrize("H,W", [(1, 1), (3, 17), (17, 3), (64, 64), (5, 48)])
@pytest.mark.parametrize("N", [1, 2, 5, 63, 64, 65, 200])
@pytest.mark.parametrize("dtype,full_range", [(np.uint8, False), (np.uint16, False), (np.uint16, True), (np.uint8, True)])
def test_whole_window_fp32_shapes(Q, oracle, H, W, N, dtype, full_range):
    """full_range: samples uniform over 0..65535 (0..255), far from the pedestal (the pixel's first sample): the worst
    case for the pedestal-subtracted fp32 sums."""
    rng = np.random.default_rng(H * 1000 + W * 10 + N)
    if full_range:
        x = rng.integers(0, 65536 if dtype == np.uint16 else 256, size=(N, H, W)).astype(dtype)
    else:
        x = _rand_stack(rng, N, H, W, dtype)
    ref = {"nu": 0.0937, "phase": 0.3}
    ctx = Q.QLD(H, W, "u8" if dtype == np.uint8 else "u16", N, [ref], accum=Q.QLD_ACC_FP32)
    ctx.push_frames(x)
    ctx.demod(Q.QLD_WHOLE)
    ctx.sync()
    check_float_maps(_maps(ctx), oracle_maps(oracle, x, ref), what=f"{H}x{W} N={N}")
    ctx.destroy()


@pytest.mark.parametrize("K", [1, 2, 3, 8])
@pytest.mark.parametrize("dtype", [np.uint8, np.uint16])
def test_multi_reference_equals_single_runs(Q, oracle, K, dtype):
    """A6 / G13: K references on shared loads == K independent QLDs."""
    rng = np.random.default_rng(K)
    H, W, N = 24, 40, 130
    x = _rand_stack(rng, N, H, W, dtype)
    refs = [{"nu": 0.05 + 0.05 * k, "phase": 0.1 * k} for k in range(K)]
    ctx = Q.QLD(H, W, "u8" if dtype == np.uint8 else "u16", N, refs, accum=Q.QLD_ACC_FP32)
    ctx.push_frames(x)
    ctx.demod(Q.QLD_WHOLE)
    ctx.sync()
    for k in range(K):
        check_float_maps(_maps(ctx, k), oracle_maps(oracle, x, refs[k]), what=f"K={K} k={k}")
    ctx.destroy()


def test_normalisation_and_map_selection(Q, oracle):
    rng = np.random.default_rng(3)
    H, W, N = 16, 32, 64
    x = _rand_stack(rng, N, H, W, np.uint16)
    ref = {"nu": 0.125}
    ctx = Q.QLD(H, W, "u16", N, [ref], accum=Q.QLD_ACC_FP32, norm=Q.QLD_NORM_AMPLITUDE, maps=Q.QLD_MAP_AMP)
    ctx.push_frames(x)
    ctx.demod()
    ctx.sync()
    I, Qm, A, P = _maps(ctx)
    assert I is None and Qm is None and P is None
    check_float_maps((None, None, A, None), oracle_maps(oracle, x, ref, scale=2.0 / N))
    ctx.destroy()


@pytest.mark.parametrize("accum_name", ["FP32", "FIXED"])
@pytest.mark.parametrize("H,W,N,dtype", [(16, 64, 64, np.uint16), (7, 24, 33, np.uint8), (128, 320, 48, np.uint16)])
def test_supplied_reference_tables(Q, oracle, accum_name, H, W, N, dtype):
    """qld_set_ref_tables ("creates tables of sine and cosine functions"): nu = 1/2, nu = 0 (reading G18) and an
    arbitrary table; the sums are the definition on whatever the arrays hold."""
    rng = np.random.default_rng(N)
    x = _rand_stack(rng, N, H, W, dtype, hi=256 if dtype == np.uint8 else 65536)
    s = np.arange(1, N + 1)
    tabs = [(np.zeros(N), np.where(s % 2 == 0, 1.0, -1.0)),                 # nu = 1/2
            (np.zeros(N), np.ones(N)),                                       # nu = 0: Q = sum x
            (np.sin(0.61 * s + 0.2) * np.hanning(N + 2)[1:-1], np.cos(0.61 * s + 0.2) * np.hanning(N + 2)[1:-1])]   # a windowed reference
    refs = [{"nu": 0.5}, {"nu": 0.0}, {"nu": 0.3}]
    try:
        ctx = Q.QLD(H, W, "u8" if dtype == np.uint8 else "u16", N, refs, accum=getattr(Q, "QLD_ACC_" + accum_name), ref_tables_supplied=True)
    except Q.QLDError as e:
        assert accum_name == "FIXED" and e.status == Q.QLD_E_UNSUPPORTED and (H * W * x.itemsize) % 16 != 0
        return
    ctx.push_frames(x)
    with pytest.raises(Q.QLDError) as e:
        ctx.demod()                                            # tables missing
    assert e.value.status == Q.QLD_E_STATE
    for k, (sn, cs) in enumerate(tabs):
        ctx.set_ref_tables(k, sn, cs)
    with pytest.raises(Q.QLDError) as e:
        ctx.set_ref_tables(0, np.full(N, 1.5), np.zeros(N))
    assert e.value.status == Q.QLD_E_INVAL
    ctx.demod()
    ctx.sync()
    for k, (sn, cs) in enumerate(tabs):
        I, Qo = oracle.demod(x, sn, cs, nthreads=oracle.max_threads())
        R, ph = oracle.finalise(I, Qo)
        check_float_maps(_maps(ctx, k), (I, Qo, R, ph), rel=1e-5 if accum_name == "FP32" else 1e-6, what=f"supplied tables k={k}")
    if accum_name == "FP32":
        Qsum = _maps(ctx, 1)[1]
        assert np.array_equal(Qsum, x.astype(np.float64).sum(axis=0).astype(np.float32))      # nu = 0: the plain sum, exact below 2^24... rounded once
    ctx.destroy()
    with pytest.raises(Q.QLDError) as e:
        Q.QLD(H, W, "u16", N, [{"nu": 0.5}])                   # without tables nu = 1/2 stays rejected
    assert e.value.status == Q.QLD_E_INVAL


def test_closed_form_tone_on_gpu(Q):
    """A pure 100-count tone on a 1000-count pedestal at nu = 1/8, N = 256: R = A N/2 = 12800, phase = phi."""
    N, H, W = 256, 4, 16
    s = np.arange(1, N + 1)[:, None, None]
    phi = np.linspace(-3, 3, H * W).reshape(1, H, W)
    x = np.rint(1000 + 100 * np.sin(2 * np.pi * s / 8 + phi)).astype(np.uint16)
    ctx = Q.QLD(H, W, "u16", N, [{"num": 1, "den": 8}], accum=Q.QLD_ACC_FP32)
    ctx.push_frames(x)
    ctx.demod()
    ctx.sync()
    I, Qm, A, P = _maps(ctx)
    # the samples are rounded to integers and the rounding error repeats with the 8-sample period, so it adds
    # coherently: up to 0.5 * N/2 = 64 counts (0.5 %), not the GPU's doing
    assert np.abs(A - 12800).max() < 64.5
    assert np.abs(np.remainder(P - phi[0] + np.pi, 2 * np.pi) - np.pi).max() < 64.5 / 12800
    ctx.destroy()


# ------------------------------------------------------------------------------------------------ A3' integer paths
@pytest.mark.parametrize("dtype,hi", [(np.uint8, 256), (np.uint16, 65536)])
@pytest.mark.parametrize("H,W,N", [(64, 64, 64), (3, 17, 65), (16, 48, 1000)])
def test_quarter_rate_integer_reference_bit_exact(Q, oracle, dtype, hi, H, W, N):
    """nu = 1/4, phase 0: references are {0, +-1}; I, Q and the amplitude are bit-exact."""
    rng = np.random.default_rng(N)
    x = rng.integers(0, hi, size=(N, H, W)).astype(dtype)
    ref = {"num": 1, "den": 4}
    ctx = Q.QLD(H, W, "u8" if dtype == np.uint8 else "u16", N, [ref], accum=Q.QLD_ACC_INT_BINS)
    ctx.push_frames(x)
    ctx.demod()
    ctx.sync()
    sn, cs = oracle.ref_tables(ref, 1, N)
    oI, oQ = oracle.demod_int(x, sn.astype(np.int64), cs.astype(np.int64))
    I, Qm, A, P = _maps(ctx)
    assert np.array_equal(I, oI.astype(np.float32)) and np.array_equal(Qm, oQ.astype(np.float32))
    p2 = (oI * oI + oQ * oQ)
    assert p2.max() < 2 ** 53
    assert np.array_equal(A, np.sqrt(p2.astype(np.float64)).astype(np.float32))
    bins = ctx.get_bins(0).cpu().numpy()
    assert np.array_equal(bins[0], oQ) and np.array_equal(bins[1], oI)       # D_0 = Q, D_1 = I (include/qld.h)
    ctx.destroy()


@pytest.mark.parametrize("num,den", [(1, 6), (1, 8), (2, 5), (3, 16), (1, 3)])
def test_phase_bins_bit_exact(Q, oracle, num, den):
    rng = np.random.default_rng(den)
    H, W, N = 20, 24, 257
    x = rng.integers(0, 4096, size=(N, H, W)).astype(np.uint16)
    ref = {"num": num, "den": den, "phase": 0.0}
    ctx = Q.QLD(H, W, "u16", N, [ref], accum=Q.QLD_ACC_INT_BINS, max_value=4095)
    ctx.push_frames(x)
    ctx.demod()
    ctx.sync()
    B = oracle.bins(x, num, den)
    bins = ctx.get_bins(0).cpu().numpy()
    if den % 2 == 0:
        assert np.array_equal(bins, B[:den // 2] - B[den // 2:])
    else:
        assert np.array_equal(bins, B)
    # maps: fp64 combination of exact integers, stored as fp32: 1e-6 relative to the map scale
    check_float_maps(_maps(ctx), oracle_maps(oracle, x, ref), rel=1e-6, what=f"bins {num}/{den}")
    ctx.destroy()


def test_auto_picks_bins_for_small_rational_and_fp32_otherwise(Q):
    a = Q.QLD(8, 8, "u8", 64, [{"num": 1, "den": 4}])
    b = Q.QLD(8, 8, "u16", 64, [{"nu": 0.0937}])
    x = np.zeros((64, 8, 8), np.uint8)
    a.push_frames(x); a.demod(); a.sync()
    assert a.get_bins(0).shape[0] == 2
    with pytest.raises(Q.QLDError):
        b.get_bins(0)
    a.destroy(); b.destroy()


# ------------------------------------------------------------------------------------------------ A5 sliding window
@pytest.mark.parametrize("accum_name", ["INT_BINS", "FP32"])
@pytest.mark.parametrize("hop,cap", [(8, 72), (8, 77), (5, 71), (64, 130)])   # cap >= N + hop + batch - 1
def test_sliding_equals_direct_recompute(Q, oracle, accum_name, hop, cap):
    """Every window equals the oracle's direct recomputation; ring wrap-around, hop not dividing the ring,
    partial pushes; the bins path is bit-exact at every hop."""
    rng = np.random.default_rng(hop + cap)
    H, W, N, T = 12, 16, 64, 400
    stream = _rand_stack(rng, T, H, W, np.uint16)
    ref = {"num": 1, "den": 6}
    accum = getattr(Q, "QLD_ACC_" + accum_name)
    ctx = Q.QLD(H, W, "u16", N, [ref], ring_frames=cap, accum=accum, max_value=4095)
    pushed, w = 0, 0
    batch = 3 if hop == 5 else hop                         # pushes need not align with hops
    while True:
        # push as much as the ring allows, in `batch`-sized pieces
        while pushed + batch <= T:
            try:
                ctx.push_frames(stream[pushed:pushed + batch])
                pushed += batch
            except Q.QLDError as e:
                assert e.status == Q.QLD_E_OVERRUN
                break
        try:
            ctx.demod(Q.QLD_SLIDE, hop)
        except Q.QLDError as e:
            assert e.status == Q.QLD_E_STATE
            break
        ctx.sync()
        a = w * hop
        ora = oracle_maps(oracle, stream[a:a + N], ref, s_first=a + 1)
        if accum_name == "INT_BINS":
            B = oracle.bins(stream[a:a + N], 1, 6, s_first=a + 1)
            assert np.array_equal(ctx.get_bins(0).cpu().numpy(), B[:3] - B[3:]), f"window {w}"
            check_float_maps(_maps(ctx), ora, rel=1e-6, what=f"window {w}")
        else:
            check_float_maps(_maps(ctx), ora, what=f"window {w}")
        w += 1
    assert pushed + batch > T and w == (pushed - N) // hop + 1
    ctx.destroy()


def test_sliding_fp32_real_nu_with_resync(Q, oracle):
    rng = np.random.default_rng(77)
    H, W, N, hop, T = 8, 32, 128, 16, 1024
    stream = _rand_stack(rng, T, H, W, np.uint16)
    ref = {"nu": 0.0937}
    for resync in (0, 7):
        ctx = Q.QLD(H, W, "u16", N, [ref], ring_frames=N + 2 * hop, accum=Q.QLD_ACC_FP32, resync_hops=resync)
        ctx.push_frames(stream[:N])
        ctx.demod(Q.QLD_SLIDE, hop)
        for w in range(1, (T - N) // hop + 1):
            ctx.push_frames(stream[N + (w - 1) * hop:N + w * hop])
            ctx.demod(Q.QLD_SLIDE, hop)
            if w % 9 == 0 or w == (T - N) // hop:
                ctx.sync()
                check_float_maps(_maps(ctx), oracle_maps(oracle, stream[w * hop:w * hop + N], ref, s_first=w * hop + 1),
                                 what=f"resync={resync} window {w}")
        ctx.destroy()


# ------------------------------------------------------------------------------------------------ boundary behaviour on the device
def test_state_errors_reset_and_attach(Q, oracle):
    import torch
    H, W, N = 8, 16, 32
    rng = np.random.default_rng(1)
    x = _rand_stack(rng, N, H, W, np.uint16)
    ref = {"nu": 0.2}
    ctx = Q.QLD(H, W, "u16", N, [ref], accum=Q.QLD_ACC_FP32)
    with pytest.raises(Q.QLDError) as e:
        ctx.demod()
    assert e.value.status == Q.QLD_E_STATE
    ctx.push_frames(x[:10])                                   # partial pushes
    with pytest.raises(Q.QLDError):
        ctx.demod()
    ctx.push_frames(x[10:])
    with pytest.raises(Q.QLDError) as e:
        ctx.push_frames(x[:1])                                # store full
    assert e.value.status == Q.QLD_E_OVERRUN
    with pytest.raises(Q.QLDError) as e:
        ctx.demod(Q.QLD_SLIDE, 4)                             # not a ring context
    assert e.value.status == Q.QLD_E_STATE
    ctx.demod(); ctx.sync()
    first = _maps(ctx)
    assert ctx.counters() == (N, 1) and ctx.kernel_launches() >= 2
    ctx.reset()
    assert ctx.counters() == (0, 0)
    pinned = torch.from_numpy(x[::-1].copy()).pin_memory()    # pinned host buffer, reversed stack
    ctx.push_frames(pinned)
    assert ctx.push_done(block=True)
    ctx.demod(); ctx.sync()
    check_float_maps(_maps(ctx), oracle_maps(oracle, x[::-1].copy(), ref))
    # attach a device stack in place
    ctx.reset()
    dev = torch.from_numpy(x).cuda()
    ctx.attach_frames_device(dev)
    ctx.demod(); ctx.sync()
    again = _maps(ctx)
    assert all(np.array_equal(a, b) for a, b in zip(first, again))      # same bytes, same kernel: deterministic
    host = torch.empty((H, W), dtype=torch.float32).pin_memory()
    ctx.read_map(0, Q.QLD_MAP_AMP, host); ctx.sync()
    assert np.array_equal(host.numpy(), again[2])
    ctx.destroy(); ctx.destroy()                                         # double destroy is a no-op


def test_device_generator_is_bit_identical_to_numpy(Q):
    from paper_1511_03390_b200 import synth
    for wl in (synth.cfg0(), synth.cfg1(H=60, W=80, N=16), synth.cfg2(H=64, W=80, N=16),
               synth.cfg3(H=64, W=64, n_stream=48, N=16, hop=4, batch=4), synth.cfg4(H=64, W=64, N=16)):
        n = min(16, wl.scene.n_frames)
        dev = Q.synth_fill(wl.scene, 3 if wl.scene.n_frames > 20 else 1, n)
        host = synth.frames(wl.scene, 3 if wl.scene.n_frames > 20 else 1, n)
        assert np.array_equal(dev.cpu().numpy(), host), wl.name


# ------------------------------------------------------------------------------------------------ TMA-fed kernel
# k_demod_stream takes over for large frames; qld_debug_set_tile(SEG, KC) forces it (and its tile shape) on small ones.
STREAM_TILES = ["512,16", "1024,16", "2048,16", "2048,32", "256,32", "1024,64"]


@pytest.mark.parametrize("tile", STREAM_TILES)
@pytest.mark.parametrize("H,W,N,dtype", [(16, 200, 70, np.uint16), (9, 136, 16, np.uint16), (50, 128, 9, np.uint8), (37, 48, 129, np.uint16),
                                         (25, 64, 3, np.uint16), (33, 256, 100, np.uint8), (128, 320, 40, np.uint16)])
def test_stream_kernel_fp32_tiles(Q, oracle, tile, H, W, N, dtype):
    """Every tile shape (column groups x time slices), ragged last tile, ragged last stage, fewer frames than a stage."""
    mk = forced(Q, "stream", tile)
    rng = np.random.default_rng(H + W + N)
    x = _rand_stack(rng, N, H, W, dtype)
    ref = {"nu": 0.0937, "phase": 0.3}
    ctx = mk(H, W, "u8" if dtype == np.uint8 else "u16", N, [ref], accum=Q.QLD_ACC_FP32)
    ctx.push_frames(x)
    ctx.demod(Q.QLD_WHOLE)
    ctx.demod(Q.QLD_WHOLE)             # second launch: cached tensor map, tile counter reset
    ctx.sync()
    check_float_maps(_maps(ctx), oracle_maps(oracle, x, ref), what=f"stream {tile} {H}x{W} N={N}")
    ctx.destroy()


@pytest.mark.parametrize("tile", ["512,16", "2048,16"])
@pytest.mark.parametrize("K", [2, 3, 8])
@pytest.mark.parametrize("dtype", [np.uint8, np.uint16])
def test_stream_kernel_multi_reference(Q, oracle, tile, K, dtype):
    mk = forced(Q, "stream", tile)
    rng = np.random.default_rng(K)
    H, W, N = 24, 256, 130
    x = _rand_stack(rng, N, H, W, dtype)
    refs = [{"nu": 0.05 + 0.05 * k, "phase": 0.1 * k} for k in range(K)]
    ctx = mk(H, W, "u8" if dtype == np.uint8 else "u16", N, refs, accum=Q.QLD_ACC_FP32)
    ctx.push_frames(x)
    ctx.demod(Q.QLD_WHOLE)
    ctx.sync()
    for k in range(K):
        check_float_maps(_maps(ctx, k), oracle_maps(oracle, x, refs[k]), what=f"stream K={K} k={k}")
    ctx.destroy()


@pytest.mark.parametrize("tile", ["512,16", "2048,16", "1024,32"])
@pytest.mark.parametrize("den,dtype", [(4, np.uint8), (6, np.uint16), (8, np.uint8), (5, np.uint16), (16, np.uint16)])
def test_stream_kernel_integer_bins_bit_exact(Q, oracle, tile, den, dtype):
    """A3' through the TMA-fed kernel: int32 phase bins bit-exact against the int64 oracle."""
    mk = forced(Q, "stream", tile)
    rng = np.random.default_rng(den)
    H, W, N = 20, 192, 150
    hi = 256 if dtype == np.uint8 else 65536
    x = rng.integers(0, hi, size=(N, H, W)).astype(dtype)
    ref = {"num": 1, "den": den}
    ctx = mk(H, W, "u8" if dtype == np.uint8 else "u16", N, [ref], accum=Q.QLD_ACC_INT_BINS)
    ctx.push_frames(x)
    ctx.demod(Q.QLD_WHOLE)
    ctx.sync()
    rows = ctx.get_bins(0).cpu().numpy().astype(np.int64)
    bins = oracle.bins(x, 1, den)
    if den % 2 == 0:
        exp = bins[: den // 2] - bins[den // 2:]
    else:
        exp = bins
    assert np.array_equal(rows, exp)
    check_float_maps(_maps(ctx), oracle_maps(oracle, x, ref), rel=1e-6, what=f"stream bins den={den}")
    ctx.destroy()


@pytest.mark.parametrize("tile", ["512,16", "2048,16"])
def test_stream_kernel_ring_wraparound(Q, oracle, tile):
    """QLD_WHOLE on a ring whose window straddles the wrap: two runs of slots, weights by absolute frame index."""
    mk = forced(Q, "stream", tile)
    rng = np.random.default_rng(7)
    H, W, N, cap = 16, 128, 40, 56
    total = 152
    x = _rand_stack(rng, total, H, W, np.uint16)
    ref = {"nu": 0.0937, "phase": 0.3}
    ctx = mk(H, W, "u16", N, [ref], ring_frames=cap, accum=Q.QLD_ACC_FP32)
    pushed = 0
    for b in (40, 8, 16, 8, 16, 16, 16, 16, 16):
        ctx.push_frames(x[pushed:pushed + b])
        pushed += b
        ctx.demod(Q.QLD_WHOLE)
        ctx.sync()
        win = x[pushed - N:pushed]
        check_float_maps(_maps(ctx), oracle_maps(oracle, win, ref, s_first=pushed - N + 1), what=f"ring whole at {pushed}")
    ctx.destroy()


@pytest.mark.parametrize("tile", ["512,16", "2048,16", "1024,32"])
@pytest.mark.parametrize("accum_name,ref", [("INT_BINS", {"num": 1, "den": 6}), ("FP32", {"num": 1, "den": 6}), ("FP32", {"nu": 0.0937, "phase": 0.3}),
                                            ("INT_BINS", {"num": 1, "den": 4})])
@pytest.mark.parametrize("hop,cap", [(32, 170), (40, 173), (64, 192)])
def test_stream_kernel_sliding_update(Q, oracle, tile, accum_name, ref, hop, cap):
    """A5 through the TMA-fed kernel: runs {expired, -w} + {new, +w} added to the stored accumulators; hops that are
    and are not multiples of a stage, expired and new runs that wrap around the ring; bins bit-exact at every hop."""
    mk = forced(Q, "stream", tile)
    rng = np.random.default_rng(hop + cap)
    H, W, N, T = 12, 128, 96, 96 + 9 * hop
    stream = _rand_stack(rng, T, H, W, np.uint16)
    ctx = mk(H, W, "u16", N, [ref], ring_frames=cap, accum=getattr(Q, "QLD_ACC_" + accum_name), max_value=4095)
    ctx.push_frames(stream[:N])
    ctx.demod(Q.QLD_SLIDE, hop)
    for w in range(0, (T - N) // hop + 1):
        if w > 0:
            ctx.push_frames(stream[N + (w - 1) * hop:N + w * hop])
            ctx.demod(Q.QLD_SLIDE, hop)
            assert ctx.last_kernel() == "k_demod_stream"
        ctx.sync()
        a = w * hop
        ora = oracle_maps(oracle, stream[a:a + N], ref, s_first=a + 1)
        if accum_name == "INT_BINS":
            den = ref["den"]
            B = oracle.bins(stream[a:a + N], 1, den, s_first=a + 1)
            assert np.array_equal(ctx.get_bins(0).cpu().numpy(), B[:den // 2] - B[den // 2:]), f"window {w}"
            check_float_maps(_maps(ctx), ora, rel=1e-6, what=f"window {w}")
        else:
            check_float_maps(_maps(ctx), ora, what=f"window {w}")
    ctx.destroy()


@pytest.mark.parametrize("tile", ["512,16", "2048,16", "1024,32"])
@pytest.mark.parametrize("accum_name,ref", [("INT_BINS", {"num": 1, "den": 6}), ("FP32", {"nu": 0.0937, "phase": 0.3}), ("INT_BINS", {"num": 3, "den": 8})])
@pytest.mark.parametrize("hop,cap", [(32, 170), (64, 200)])
def test_block_partial_sliding(Q, oracle, tile, accum_name, ref, hop, cap):
    """8(f3): slide_hop > 0 keeps the per-batch partial sums and reads only the new frames; every window equals the
    oracle's direct recomputation (bins bit-exact), through ring wrap-around and more hops than partial slots."""
    mk = forced(Q, "stream", tile)
    rng = np.random.default_rng(hop + cap)
    H, W, N, T = 12, 128, 128, 128 + 9 * hop
    stream = _rand_stack(rng, T, H, W, np.uint16)
    ctx = mk(H, W, "u16", N, [ref], ring_frames=cap, accum=getattr(Q, "QLD_ACC_" + accum_name), max_value=4095, slide_hop=hop,
                resync_hops=5 if accum_name == "FP32" else 0)
    ctx.push_frames(stream[:N])
    ctx.demod(Q.QLD_SLIDE, hop)
    with pytest.raises(Q.QLDError) as e:
        ctx.demod(Q.QLD_SLIDE, hop // 2)                        # only the configured hop
    assert e.value.status == Q.QLD_E_INVAL
    for w in range(0, (T - N) // hop + 1):
        if w > 0:
            ctx.push_frames(stream[N + (w - 1) * hop:N + w * hop])
            ctx.demod(Q.QLD_SLIDE, hop)
        ctx.sync()
        a = w * hop
        ora = oracle_maps(oracle, stream[a:a + N], ref, s_first=a + 1)
        if accum_name == "INT_BINS":
            den, num = ref["den"], ref["num"]
            B = oracle.bins(stream[a:a + N], num, den, s_first=a + 1)
            assert np.array_equal(ctx.get_bins(0).cpu().numpy(), B[:den // 2] - B[den // 2:]), f"window {w}"
            check_float_maps(_maps(ctx), ora, rel=1e-6, what=f"window {w}")
        else:
            check_float_maps(_maps(ctx), ora, what=f"window {w}")
    ctx.destroy()


def test_block_partial_sliding_rejects_what_it_cannot_do(Q):
    with pytest.raises(Q.QLDError) as e:
        Q.QLD(12, 128, "u16", 100, [{"num": 1, "den": 6}], ring_frames=200, slide_hop=32)       # hop does not divide N
    assert e.value.status == Q.QLD_E_UNSUPPORTED
    with pytest.raises(Q.QLDError) as e:
        Q.QLD(12, 128, "u16", 128, [{"num": 1, "den": 6}], slide_hop=32)                        # not a ring
    assert e.value.status == Q.QLD_E_INVAL
    ctx = Q.QLD(12, 128, "u16", 128, [{"num": 1, "den": 6}], ring_frames=200, slide_hop=32)      # a frame too small for the TMA kernel
    ctx.push_frames(np.zeros((128, 12, 128), np.uint16))
    with pytest.raises(Q.QLDError) as e:
        ctx.demod(Q.QLD_SLIDE, 32)
    assert e.value.status == Q.QLD_E_UNSUPPORTED
    ctx.destroy()


# ------------------------------------------------------------------------------------------------ A2 zero-copy ingest
@pytest.mark.parametrize("accum_name", ["INT_BINS", "FP32"])
def test_commit_frames_into_attached_ring(Q, oracle, accum_name):
    """external_store ring: the producer writes frames in place on its own stream, qld_commit_frames announces
    them; windows (with ring wrap-around) equal the oracle's direct recomputation; overrun and state errors."""
    import torch
    rng = np.random.default_rng(5)
    H, W, N, hop, cap, T = 8, 32, 48, 8, 64, 200
    stream = _rand_stack(rng, T, H, W, np.uint16)
    dev_stream = torch.from_numpy(stream.view(np.int16)).cuda()
    ring = torch.zeros((cap, H, W), dtype=torch.int16, device="cuda")
    ref = {"num": 1, "den": 6}
    ctx = Q.QLD(H, W, "u16", N, [ref], ring_frames=cap, accum=getattr(Q, "QLD_ACC_" + accum_name), max_value=4095,
                external_store=True)
    with pytest.raises(Q.QLDError) as e:
        ctx.commit_frames(4)                                   # nothing attached yet
    assert e.value.status == Q.QLD_E_STATE
    with pytest.raises(Q.QLDError) as e:
        ctx.push_frames(stream[:4])                            # copies are refused on an external store
    assert e.value.status == Q.QLD_E_STATE
    ctx.attach_frames_device(ring)
    producer = torch.cuda.Stream()

    def produce(first, n):                                     # frames first+1 .. first+n written in place
        with torch.cuda.stream(producer):
            for s in range(first, first + n):
                ring[s % cap].copy_(dev_stream[s], non_blocking=True)
        ctx.commit_frames(n, producer)

    produce(0, N)
    with pytest.raises(Q.QLDError) as e:
        ctx.commit_frames(cap - N + 1)                         # would overwrite frame 1 before window 0 exists
    assert e.value.status == Q.QLD_E_OVERRUN
    ctx.demod(Q.QLD_SLIDE, hop)
    pushed, w = N, 0
    while True:
        ctx.sync()
        a = w * hop
        check_float_maps(_maps(ctx), oracle_maps(oracle, stream[a:a + N], ref, s_first=a + 1),
                         rel=1e-6 if accum_name == "INT_BINS" else 1e-5, what=f"window {w}")
        if pushed + hop > T:
            break
        produce(pushed, hop)
        pushed += hop
        ctx.demod(Q.QLD_SLIDE, hop)
        w += 1
    assert w == (T - N) // hop and ctx.counters() == (pushed, w + 1)
    ctx.reset()                                                # the ring stays attached
    produce(0, N)
    ctx.demod(Q.QLD_WHOLE)
    ctx.sync()
    check_float_maps(_maps(ctx), oracle_maps(oracle, stream[:N], ref), what="after reset")
    ctx.destroy()


# ------------------------------------------------------------------------------------------------ A5 through the copy engines
@pytest.mark.timeout(300, method="thread")
@pytest.mark.parametrize("accum_name,refs", [("INT_BINS", [{"num": 1, "den": 6}]), ("INT_BINS", [{"num": 1, "den": 4}]), ("INT_BINS", [{"num": 3, "den": 8}]),
                                             ("INT_BINS", [{"num": 1, "den": 4}, {"num": 1, "den": 4, "phase_quarter": 1}]),
                                             ("FP32", [{"nu": 0.0937, "phase": 0.3}]), ("FP32", [{"nu": 0.21}, {"num": 1, "den": 6}])])
@pytest.mark.parametrize("hop,cap,partial", [(32, 170, True), (32, 170, False), (40, 173, False), (5, 140, False), (64, 200, True), (16, 150, False)])
@pytest.mark.parametrize("dtype,H,W,maps", [(np.uint16, 12, 128, "all"), (np.uint16, 37, 72, "amp"), (np.uint8, 9, 144, "all")])
def test_slide_bulk_kernel(Q, oracle, accum_name, refs, hop, cap, partial, dtype, H, W, maps):
    """k_slide_bulk (forced onto small frames): stored sums, expired partial sums and maps travel by bulk copies through
    shared memory; frames by TMA.  Ragged last tile (37 x 72 = 2664 pixels = 2 tiles + 616), hops that are not a multiple of
    a stage, runs that wrap around the ring, one and two references, all maps or the amplitude only: every window equals
    the oracle's direct recomputation, integer bins bit-exact."""
    N = 128
    T = N + 7 * hop
    rng = np.random.default_rng(hop + cap + H)
    hi = 4096 if dtype == np.uint16 else 256
    stream = _rand_stack(rng, T, H, W, dtype, hi=hi)
    try:
        ctx = Q.QLD(H, W, "u8" if dtype == np.uint8 else "u16", N, refs, ring_frames=cap, accum=getattr(Q, "QLD_ACC_" + accum_name), max_value=hi - 1,
                    slide_hop=hop if partial else 0, maps=Q.QLD_MAP_ALL if maps == "all" else Q.QLD_MAP_AMP, resync_hops=-1,
                    debug_tile=("stream", 512, 16) if partial else None)
    except Q.QLDError as e:
        assert partial and e.status == Q.QLD_E_UNSUPPORTED
        return
    ctx.debug_set_tile("slide", 1)
    ctx.push_frames(stream[:N])
    ctx.demod(Q.QLD_SLIDE, hop)
    for w in range(0, (T - N) // hop + 1):
        if w > 0:
            ctx.push_frames(stream[N + (w - 1) * hop:N + w * hop])
            ctx.demod(Q.QLD_SLIDE, hop)
            # (two fp32 references with partial sums and all maps need 100 KB of state per tile: no room for the pipeline,
            # the launcher falls back to k_demod_stream)
            assert ctx.last_kernel() == "k_slide_bulk" or (accum_name == "FP32" and len(refs) == 2 and partial and maps == "all")
        ctx.sync()
        a = w * hop
        for k, ref in enumerate(refs):
            ora = oracle_maps(oracle, stream[a:a + N], ref, s_first=a + 1)
            check_float_maps(_maps(ctx, k), ora, rel=1e-6 if accum_name == "INT_BINS" else 1e-5, what=f"window {w} k={k}")
            if accum_name == "INT_BINS":
                den, num = ref["den"], ref["num"]
                B = oracle.bins(stream[a:a + N], num, den, s_first=a + 1)
                assert np.array_equal(ctx.get_bins(k).cpu().numpy(), B[:den // 2] - B[den // 2:]), f"window {w} k={k}"
    ctx.destroy()


# ------------------------------------------------------------------------------------------------ f4: camera byte stream
@pytest.mark.timeout(300, method="thread")
@pytest.mark.parametrize("path", ["whole_fp32", "whole_bins", "stream_fp32", "stream_bins", "stream_bins_k2", "tc_fixed", "slide_small", "slide_bulk_bins",
                                  "slide_bulk_fp32", "slide_partial"])
def test_big_endian_byte_stream(Q, oracle, path):
    """QLD_U16_BE (the camera's 16-bit stream, pairs of bytes stitched into values): the bytes arrive most
    significant first and are joined inside the kernels' loads.  Oracle: stitch on the host, then the definition."""
    rng = np.random.default_rng(len(path))
    H, W, N = 24, 128, 96
    x = rng.integers(0, 65536, size=(N + 6 * 16, H, W)).astype(np.uint16)      # full range: both bytes matter
    raw = x.byteswap()                                                          # what the wire carries, viewed as uint16 words
    assert np.array_equal(raw.view(np.uint8).reshape(-1, 2)[:, 0].astype(np.uint16) * 256 + raw.view(np.uint8).reshape(-1, 2)[:, 1], x.reshape(-1))
    ring = path.startswith("slide")
    hop = 32 if path == "slide_partial" else 16               # the partial-sum seeding needs a hop of at least one stage
    kw = dict(max_value=65535)
    if path in ("whole_fp32", "stream_fp32", "slide_small", "slide_bulk_fp32"):
        refs, kw["accum"] = [{"nu": 0.0937, "phase": 0.3}], Q.QLD_ACC_FP32
    elif path == "stream_bins_k2":
        refs, kw["accum"] = [{"num": 1, "den": 4}, {"num": 1, "den": 8}], Q.QLD_ACC_INT_BINS
    elif path == "tc_fixed":
        refs, kw["accum"] = [{"nu": 0.0937}, {"num": 1, "den": 6}], Q.QLD_ACC_FIXED
    else:
        refs, kw["accum"] = [{"num": 1, "den": 6}], Q.QLD_ACC_INT_BINS
    if path.startswith("stream"):
        kw["debug_tile"] = ("stream", 1024, 16)
    if ring:
        kw["ring_frames"] = N + 40
        kw["resync_hops"] = -1
    if path == "slide_partial":
        kw["slide_hop"] = hop
        kw["debug_tile"] = ("stream", 512, 16)
    ctx = Q.QLD(H, W, "u16be", N, refs, **kw)
    if path.startswith("slide_bulk") or path == "slide_partial":
        ctx.debug_set_tile("slide", 1)
    ctx.push_frames(raw[:N])
    tol = 1e-5 if kw["accum"] == Q.QLD_ACC_FP32 else 1e-6
    if not ring:
        ctx.demod(Q.QLD_WHOLE)
        ctx.sync()
        for k, ref in enumerate(refs):
            check_float_maps(_maps(ctx, k), oracle_maps(oracle, x[:N], ref), rel=tol, what=f"{path} k={k}")
        if kw["accum"] == Q.QLD_ACC_INT_BINS:
            B = oracle.bins(x[:N], refs[0]["num"], refs[0]["den"])
            h = refs[0]["den"] // 2
            assert np.array_equal(ctx.get_bins(0).cpu().numpy(), B[:h] - B[h:])
    else:
        ctx.demod(Q.QLD_SLIDE, hop)
        for w in range(96 // hop + 1):
            if w > 0:
                ctx.push_frames(raw[N + (w - 1) * hop:N + w * hop])
                ctx.demod(Q.QLD_SLIDE, hop)
                assert (ctx.last_kernel() == "k_slide_bulk") == (path != "slide_small")
            ctx.sync()
            a = w * hop
            check_float_maps(_maps(ctx, 0), oracle_maps(oracle, x[a:a + N], refs[0], s_first=a + 1), rel=tol, what=f"{path} window {w}")
            if kw["accum"] == Q.QLD_ACC_INT_BINS:
                B = oracle.bins(x[a:a + N], 1, 6, s_first=a + 1)
                assert np.array_equal(ctx.get_bins(0).cpu().numpy(), B[:3] - B[3:]), f"window {w}"
    ctx.destroy()


@pytest.mark.timeout(300, method="thread")
@pytest.mark.parametrize("path", ["small", "stream", "bulk", "bulk_partial"])
@pytest.mark.parametrize("accum_name,refs", [("INT_BINS", [{"num": 1, "den": 6}]), ("FP32", [{"nu": 0.0937, "phase": 0.3}]),
                                             ("FP32", [{"nu": 0.21, "phase": -1.0}, {"num": 3, "den": 16}])])
def test_window_relative_maps(Q, oracle, path, accum_name, refs):
    """cfg.window_relative (reading G10): the I, Q and phase maps of every window equal the definition with the frame index
    counted from the window's own first frame (s = 1) -- a steady source shows a steady phase from window to
    window -- while the integer bins stay the absolute-index sums."""
    rng = np.random.default_rng(11)
    H, W, N, hop = 16, 128, 128, 32
    T = N + 6 * hop
    stream = _rand_stack(rng, T, H, W, np.uint16)
    kw = dict(ring_frames=N + 2 * hop + 5, accum=getattr(Q, "QLD_ACC_" + accum_name), max_value=4095, window_relative=True, resync_hops=3)
    if path in ("stream", "bulk_partial"):
        kw["debug_tile"] = ("stream", 512, 16)
    if path == "bulk_partial":
        kw["slide_hop"] = hop
    ctx = Q.QLD(H, W, "u16", N, refs, **kw)
    if path.startswith("bulk"):
        ctx.debug_set_tile("slide", 1)
    elif path == "stream":
        ctx.debug_set_tile("slide", 2)
    ctx.push_frames(stream[:N])
    ctx.demod(Q.QLD_SLIDE, hop)
    for w in range(7):
        if w > 0:
            ctx.push_frames(stream[N + (w - 1) * hop:N + w * hop])
            ctx.demod(Q.QLD_SLIDE, hop)
        ctx.sync()
        a = w * hop
        for k, ref in enumerate(refs):
            ora = oracle_maps(oracle, stream[a:a + N], ref, s_first=1)                 # window-relative: the window's first frame is s = 1
            check_float_maps(_maps(ctx, k), ora, rel=1e-6 if accum_name == "INT_BINS" else 1e-5, what=f"{path} window {w} k={k}")
        if accum_name == "INT_BINS":
            B = oracle.bins(stream[a:a + N], 1, 6, s_first=a + 1)                      # bins: absolute frame index
            assert np.array_equal(ctx.get_bins(0).cpu().numpy(), B[:3] - B[3:])
    # a whole-window demod on the ring (most recent N frames) is window-relative too
    ctx.demod(Q.QLD_WHOLE)
    ctx.sync()
    check_float_maps(_maps(ctx, 0), oracle_maps(oracle, stream[T - N:T], refs[0], s_first=1), rel=1e-6 if accum_name == "INT_BINS" else 1e-5, what="whole on ring")
    ctx.destroy()


# ------------------------------------------------------------------------------------------------ INT_REFS: two integer sums per reference
@pytest.mark.timeout(300, method="thread")
@pytest.mark.parametrize("path", ["whole_small", "whole_stream", "whole_tc", "slide_small", "slide_bulk", "slide_partial"])
@pytest.mark.parametrize("dtype", ["u8", "u16"])
@pytest.mark.parametrize("refs", [[{"num": 1, "den": 6}], [{"num": 1, "den": 3}], [{"num": 1, "den": 6}, {"num": 1, "den": 4}], [{"num": 1, "den": 6, "phase": 0.3}]])
def test_integer_reference_rows(Q, oracle, path, dtype, refs):
    """QLD_ACC_INT_REFS (and AUTO): den = 3 or 6 without a phase offset is carried by two exact int32 sums (weights 0, +-1, +-2)
    instead of three bin rows; other references of the context keep their bins (a reference with a phase offset falls back to
    bins too).  Rows bit-exact against the integer oracle, maps to 1e-6, through every kernel that takes integer weights."""
    rng = np.random.default_rng(len(path) + len(refs))
    H, W, N, hop = 16, 128, 96, 32
    npdt = np.uint8 if dtype == "u8" else np.uint16
    hi = 256 if dtype == "u8" else 65536
    x = rng.integers(0, hi, size=(N + 4 * hop, H, W)).astype(npdt)
    kw = dict(accum=Q.QLD_ACC_AUTO, max_value=hi - 1)
    if path == "whole_stream":
        kw["debug_tile"] = ("stream", 512, 16)
    if path == "whole_tc":
        kw["debug_tile"] = ("tc", 4, 5, 64)
    ring = path.startswith("slide")
    if ring:
        kw["ring_frames"] = N + 2 * hop + 3
    if path == "slide_partial":
        kw["slide_hop"] = hop
        kw["debug_tile"] = ("stream", 512, 16)
    ctx = Q.QLD(H, W, dtype, N, refs, **kw)
    any_compact = any(r["den"] in (3, 6) and not r.get("phase") and not r.get("phase_quarter") for r in refs)
    assert ctx.accum_name() == ("INT_REFS" if any_compact else "INT_BINS")     # the mode reported is the one in use
    if path in ("slide_bulk", "slide_partial"):
        ctx.debug_set_tile("slide", 1)
    ctx.push_frames(x[:N])
    n_win = 5 if ring else 1
    for w in range(n_win):
        if ring:
            if w > 0:
                ctx.push_frames(x[N + (w - 1) * hop:N + w * hop])
            ctx.demod(Q.QLD_SLIDE, hop)
        else:
            ctx.demod(Q.QLD_WHOLE)
        ctx.sync()
        a = w * hop
        for k, ref in enumerate(refs):
            exp = expected_int_rows(oracle, x[a:a + N], ref, a + 1, "INT_REFS")
            got = ctx.get_bins(k).cpu().numpy()
            compact = ref["den"] in (3, 6) and not ref.get("phase")
            assert got.shape[0] == (2 if compact else (ref["den"] // 2 if ref["den"] % 2 == 0 else ref["den"]))
            assert np.array_equal(got, exp), f"{path} window {w} k={k}"
            check_float_maps(_maps(ctx, k), oracle_maps(oracle, x[a:a + N], ref, s_first=a + 1), rel=1e-6, what=f"{path} window {w} k={k}")
    if path == "whole_tc":
        assert ctx.last_kernel() == "k_demod_tc"
    if path in ("slide_bulk", "slide_partial"):
        assert ctx.last_kernel() == "k_slide_bulk"
    ctx.destroy()


@pytest.mark.timeout(300, method="thread")
def test_concurrent_contexts_on_separate_streams(Q, oracle):
    """Three contexts on three streams at once -- two sliding rings (dependent launches of k_slide_bulk that start while the
    previous hop drains) and one whole-window tensor-core context -- interleaved for 40 hops: no launch may wait for SMs that a
    waiting launch holds, and every result equals the oracle's."""
    import torch
    rng = np.random.default_rng(77)
    H, W, N, hop, n_hops = 64, 512, 128, 32, 40
    streams = [torch.cuda.Stream() for _ in range(3)]
    data = [rng.integers(0, 4096, size=(N + n_hops * hop, H, W)).astype(np.uint16) for _ in range(2)]
    refs = [{"num": 1, "den": 6}, {"nu": 0.0937, "phase": 0.3}]
    rings = []
    for i in range(2):
        with torch.cuda.stream(streams[i]):
            ctx = Q.QLD(H, W, "u16", N, [refs[i]], ring_frames=N + 3 * hop, max_value=4095, slide_hop=hop if i == 0 else 0,
                        debug_tile=("stream", 2048, 16) if i == 0 else None)
        ctx.debug_set_tile("slide", 1)
        ctx.push_frames(data[i][:N])
        ctx.demod(Q.QLD_SLIDE, hop)
        rings.append(ctx)
    xw = rng.integers(0, 65536, size=(256, H, W)).astype(np.uint16)
    with torch.cuda.stream(streams[2]):
        whole = Q.QLD(H, W, "u16", 256, [{"nu": 0.05 + 0.05 * k} for k in range(8)], maps=Q.QLD_MAP_AMP)
    whole.push_frames(xw)
    for w in range(1, n_hops + 1):
        for i in range(2):
            rings[i].push_frames(data[i][N + (w - 1) * hop:N + w * hop])
            rings[i].demod(Q.QLD_SLIDE, hop)
        whole.demod(Q.QLD_WHOLE)
    for c in rings + [whole]:
        c.sync()
    a = n_hops * hop
    for i in range(2):
        assert rings[i].last_kernel() == "k_slide_bulk"
        check_float_maps(_maps(rings[i]), oracle_maps(oracle, data[i][a:a + N], refs[i], s_first=a + 1), rel=1e-6 if i == 0 else 1e-5, what=f"ring {i}")
    amp = whole.get_maps(7)[2].cpu().numpy()
    check_float_maps((None, None, amp, None), oracle_maps(oracle, xw, {"nu": 0.4}), rel=1e-6, what="whole")
    for c in rings + [whole]:
        c.destroy()


# ------------------------------------------------------------------------------------------------ host far ahead of the GPU
@pytest.mark.timeout(300, method="thread")
@pytest.mark.parametrize("mode", ["bins", "bins_partial", "bins_small", "fp32", "fp32_partial", "fixed", "fixed_partial"])
@pytest.mark.parametrize("ring_hops", [50, 130])
def test_many_hops_queued_behind_a_busy_gpu(Q, oracle, mode, ring_hops):
    """120 hops are pushed and requested without a single host-side wait while the compute stream is held up, so every update
    is still queued when the last push is issued -- far more than the 32 launches the context remembers.  Nothing the copy
    stream does (frames that wrap around a 50-hop ring; table entries written ahead on the roomy 130-hop ring, whose table
    ring wraps first) may overtake an update that still reads the old contents: the last window equals the oracle's direct
    recomputation -- integer rows bit for bit; FIXED from the library's own tables (never supplied, never synchronised):
    the table is the rounded oracle table up to rint ties, and the int64 sums are the oracle's within what those ties allow."""
    import torch
    H, W, N, hop, n_hops = 12, 128, 128, 32, 120
    T = N + n_hops * hop
    rng = np.random.default_rng(ring_hops + len(mode))
    stream = _rand_stack(rng, T, H, W, np.uint16)
    dev = torch.from_numpy(stream.view(np.int16)).cuda()
    fixed, fp32 = mode.startswith("fixed"), mode.startswith("fp32")
    ref = {"num": 1, "den": 6} if mode.startswith("bins") else {"nu": 0.0937, "phase": 0.3}
    accum = Q.QLD_ACC_FIXED if fixed else Q.QLD_ACC_FP32 if fp32 else Q.QLD_ACC_INT_BINS
    ctx = Q.QLD(H, W, "u16", N, [ref], ring_frames=N + ring_hops * hop, accum=accum, max_value=4095, resync_hops=-1,
                slide_hop=hop if mode.endswith("partial") else 0, debug_tile=("stream", 512, 16) if mode.endswith("partial") else None)
    ctx.debug_set_tile("slide", 2 if mode == "bins_small" else 1)
    ctx.push_frames(dev[:N])
    ctx.demod(Q.QLD_SLIDE, hop)
    torch.cuda._sleep(400_000_000)                                  # ~0.2 s on the compute stream: everything below queues up behind it
    for w in range(1, n_hops + 1):
        ctx.push_frames(dev[N + (w - 1) * hop:N + w * hop])
        ctx.demod(Q.QLD_SLIDE, hop)
    assert ctx.counters() == (T, n_hops + 1)
    ctx.sync()
    assert (ctx.last_kernel() == "k_slide_bulk") == (mode != "bins_small")
    a = n_hops * hop
    last = stream[a:a + N]
    check_float_maps(_maps(ctx), oracle_maps(oracle, last, ref, s_first=a + 1), rel=1e-5 if fp32 else 1e-6, what=mode)
    if mode.startswith("bins"):
        assert np.array_equal(ctx.get_bins(0).cpu().numpy(), expected_int_rows(oracle, last, ref, s_first=a + 1, mode=ctx.accum_name()))
    if fixed:
        sn, cs = oracle.ref_tables(ref, a + 1, N)
        os_, oc = np.rint(sn * 2.0 ** 30).astype(np.int64), np.rint(cs * 2.0 ** 30).astype(np.int64)
        gs, gc = ctx.read_ref_table_fixed(0)                        # the N most recent entries: this window's
        assert np.abs(gs - os_).max() <= 1 and np.abs(gc - oc).max() <= 1
        oI, oQ = oracle.demod_int(last, os_, oc, nthreads=oracle.max_threads())
        gI, gQ = [t.cpu().numpy() for t in ctx.get_sums_i64(0)]
        # each entry that differs (by one unit, on a rint tie) moves a sum by at most one sample value
        assert np.abs(gI - oI).max() <= 4095 * int((gs != os_).sum()) and np.abs(gQ - oQ).max() <= 4095 * int((gc != oc).sum())
    ctx.destroy()


def test_two_host_threads_with_different_tile_shapes(Q, oracle):
    """include/qld.h: distinct contexts are independent across host threads.  Two threads each build their own contexts, one
    walking the tile shapes of k_demod_stream upwards and one downwards (their shared-memory needs differ by a factor of
    eight), each on a stream of its own; a per-kernel shared-memory limit left too low by the other thread would make a launch
    fail, a shared counter or table would spoil the maps."""
    import threading
    import torch
    H, W, N = 33, 256, 100
    ref = {"nu": 0.0937, "phase": 0.3}
    xs = [_rand_stack(np.random.default_rng(70 + i), N, H, W, np.uint16) for i in range(2)]
    want = [oracle_maps(oracle, x, ref) for x in xs]
    errors, seen = [], set()

    def worker(i):
        try:
            with torch.cuda.stream(torch.cuda.Stream()):
                for rep in range(3):
                    for tile in (STREAM_TILES if i == 0 else STREAM_TILES[::-1]):
                        ctx = forced(Q, "stream", tile)(H, W, "u16", N, [ref], accum=Q.QLD_ACC_FP32)
                        ctx.push_frames(xs[i])
                        ctx.demod(Q.QLD_WHOLE)
                        ctx.sync()
                        seen.add(ctx.last_kernel())                  # (a shape the frame cannot take falls back to k_demod_whole)
                        check_float_maps(_maps(ctx), want[i], what=f"thread {i} tile {tile}")
                        ctx.destroy()
        except BaseException as e:                                   # noqa: BLE001 -- handed to the main thread
            errors.append((i, e))

    threads = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    assert "k_demod_stream" in seen, seen


@pytest.mark.parametrize("N,want", [(16384, "INT_REFS"), (24574, "INT_REFS"), (24575, "INT_BINS"), (32768, "INT_BINS")])
def test_auto_stays_exact_when_the_compact_rows_could_overflow(Q, oracle, N, want):
    """AUTO with full-range 16-bit samples and nu = 1/6 on long windows: a compact integer-reference row collects up to 4N/3 + 2/3
    sample values, so it is taken up to N = 24574 (65535 * (floor((4N + 2) / 3) + 2) < 2^31) and no further; from there the references keep
    their three difference bins (bound N/6), still exact -- AUTO must not fall to fp32.  Samples at the top of the range, so
    that a row that did overflow would show."""
    rng = np.random.default_rng(N)
    H, W = 2, 16
    x = rng.integers(65000, 65536, size=(N, H, W)).astype(np.uint16)
    ref = {"num": 1, "den": 6}
    ctx = Q.QLD(H, W, "u16", N, [ref])                                   # accum AUTO, max_value unset: 65535
    assert ctx.accum_name() == want
    ctx.push_frames(x)
    ctx.demod(Q.QLD_WHOLE)
    ctx.sync()
    assert np.array_equal(ctx.get_bins(0).cpu().numpy(), expected_int_rows(oracle, x, ref, mode=want))
    check_float_maps(_maps(ctx), oracle_maps(oracle, x, ref), rel=1e-6, what=f"N={N}")
    ctx.destroy()
    if want == "INT_BINS":                                               # asked for by name, the compact form degrades the same way
        ctx = Q.QLD(H, W, "u16", N, [ref], accum=Q.QLD_ACC_INT_REFS)
        assert ctx.accum_name() == "INT_BINS"
        ctx.destroy()
