"""GPU parity of the tcgen05 (QLD_ACC_FIXED) path: exact int64 sums against the integer oracle with the same
Q1.30 reference table (bit-exact), and the float maps against the fp64 definition."""
import numpy as np
import pytest

from _parity import check_float_maps, forced, oracle_maps

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Q():
    import torch
    assert torch.cuda.is_available()
    from paper_1511_03390_b200 import qld
    qld.load_library()
    return qld


def _q30(oracle, ref, N):
    sn, cs = oracle.ref_tables(ref, 1, N)
    return np.rint(sn * 2.0 ** 30).astype(np.int64), np.rint(cs * 2.0 ** 30).astype(np.int64)


def _maps(ctx, k=0):
    return tuple(None if m is None else m.cpu().numpy() for m in ctx.get_maps(k))


@pytest.mark.parametrize("ref", [{"nu": 0.0937}, {"nu": 0.4321, "phase": 2.0}, {"num": 1, "den": 4}, {"num": 1, "den": 6}])
def test_fixed_table_matches_rounded_oracle(Q, oracle, ref):
    N = 1000
    ctx = Q.QLD(4, 8, "u16", N, [ref], accum=Q.QLD_ACC_FIXED)
    gs, gc = ctx.read_ref_table_fixed(0)
    os_, oc = _q30(oracle, ref, N)
    assert np.abs(gs - os_).max() <= 1 and np.abs(gc - oc).max() <= 1           # a tie in rint can flip on the last bit of sin
    assert (gs == os_).mean() > 0.999 and (gc == oc).mean() > 0.999
    ctx.destroy()


@pytest.mark.parametrize("dtype,hi", [(np.uint8, 256), (np.uint16, 65536)])
@pytest.mark.parametrize("H,W,N", [(1, 16, 1), (3, 16, 5), (4, 16, 63), (8, 24, 64), (8, 40, 65), (64, 64, 200), (37, 48, 129),
                                   (128, 160, 70)])
def test_fixed_sums_bit_exact(Q, oracle, dtype, hi, H, W, N):
    """sum_s x_s R(s) with the oracle's own Q1.30 table handed to the library: bit-exact int64, full sample range."""
    rng = np.random.default_rng(H * W + N)
    x = rng.integers(0, hi, size=(N, H, W)).astype(dtype)
    ref = {"nu": 0.0937, "phase": 0.3}
    isin, icos = _q30(oracle, ref, N)
    ctx = Q.QLD(H, W, "u8" if dtype == np.uint8 else "u16", N, [ref], accum=Q.QLD_ACC_FIXED, maps=Q.QLD_MAP_ALL | Q.QLD_MAP_SUMS_I64)
    ctx.set_ref_table_fixed(0, isin, icos)
    ctx.push_frames(x)
    ctx.demod()
    ctx.sync()
    oI, oQ = oracle.demod_int(x, isin, icos)
    gI, gQ = [t.cpu().numpy() for t in ctx.get_sums_i64(0)]
    assert np.array_equal(gI, oI) and np.array_equal(gQ, oQ)
    I, Qm, A, P = _maps(ctx)
    assert np.array_equal(I, (oI.astype(np.float64) * 2.0 ** -30).astype(np.float32))
    assert np.array_equal(Qm, (oQ.astype(np.float64) * 2.0 ** -30).astype(np.float32))
    ctx.destroy()


@pytest.mark.parametrize("K", [1, 2, 3, 5, 8])
@pytest.mark.parametrize("dtype", [np.uint8, np.uint16])
def test_fixed_multi_reference(Q, oracle, K, dtype):
    rng = np.random.default_rng(K)
    H, W, N = 40, 72, 300
    hi = 256 if dtype == np.uint8 else 4096
    x = rng.integers(0, hi, size=(N, H, W)).astype(dtype)
    refs = [{"nu": 0.05 + 0.05 * k, "phase": 0.1 * k} for k in range(K)]
    ctx = Q.QLD(H, W, "u8" if dtype == np.uint8 else "u16", N, refs, accum=Q.QLD_ACC_FIXED, maps=Q.QLD_MAP_ALL | Q.QLD_MAP_SUMS_I64)
    tabs = [_q30(oracle, r, N) for r in refs]
    for k in range(K):
        ctx.set_ref_table_fixed(k, *tabs[k])
    ctx.push_frames(x)
    ctx.demod()
    ctx.sync()
    for k in range(K):
        oI, oQ = oracle.demod_int(x, *tabs[k])
        gI, gQ = [t.cpu().numpy() for t in ctx.get_sums_i64(k)]
        assert np.array_equal(gI, oI) and np.array_equal(gQ, oQ), f"k={k}"
        # and against the float definition: quantising the references to 2^-31 costs ~1e-9 relative
        check_float_maps(_maps(ctx, k), oracle_maps(oracle, x, refs[k]), rel=1e-7, what=f"K={K} k={k}")
    ctx.destroy()


@pytest.mark.parametrize("tile", ["16,3,32", "8,6,32", "4,6,64", "2,8,64", "1,8,32"])
@pytest.mark.parametrize("H,W,N,dtype", [(16, 200, 70, np.uint16), (16, 200, 64, np.uint16), (50, 128, 9, np.uint8), (37, 48, 129, np.uint16),
                                         (25, 64, 7, np.uint16), (33, 256, 100, np.uint8)])
def test_fixed_tile_shapes_bit_exact(Q, oracle, tile, H, W, N, dtype):
    """Every tile shape the launcher can pick (T spans x KC frames per stage), forced through the tuning override, on
    stacks with a ragged last tile, a ragged last 8-frame group, fewer than 8 frames, and a row pitch that is not a
    multiple of 128 bytes (the 1 KB-box path): bit-exact int64 sums."""
    mk = forced(Q, "tc", tile)
    rng = np.random.default_rng(H + W + N)
    hi = 256 if dtype == np.uint8 else 65536
    x = rng.integers(0, hi, size=(N, H, W)).astype(dtype)
    refs = [{"nu": 0.0937, "phase": 0.3}, {"num": 1, "den": 6}]
    tabs = [_q30(oracle, r, N) for r in refs]
    ctx = mk(H, W, "u8" if dtype == np.uint8 else "u16", N, refs, accum=Q.QLD_ACC_FIXED, maps=Q.QLD_MAP_ALL | Q.QLD_MAP_SUMS_I64)
    for k in range(2):
        ctx.set_ref_table_fixed(k, *tabs[k])
    ctx.push_frames(x)
    ctx.demod()
    ctx.demod()                                              # a second launch reuses the tensor maps and the tile counter
    ctx.sync()
    for k in range(2):
        oI, oQ = oracle.demod_int(x, *tabs[k])
        gI, gQ = [t.cpu().numpy() for t in ctx.get_sums_i64(k)]
        assert np.array_equal(gI, oI) and np.array_equal(gQ, oQ), f"k={k}"
    ctx.destroy()


@pytest.mark.parametrize("K", [1, 3, 8])
def test_fixed_wide_tiles_large_frame(Q, oracle, K):
    """A frame large enough that the launcher itself picks the widest tiles (T = 16 / 8 / 4 spans for K = 1 / 3 / 8),
    with a ragged last tile (4810 spans) and a ragged last frame group (N = 70)."""
    rng = np.random.default_rng(K)
    H, W, N = 481, 640, 70
    x = rng.integers(0, 4096, size=(N, H, W)).astype(np.uint16)
    refs = [{"nu": 0.05 + 0.05 * k, "phase": 0.1 * k} for k in range(K)]
    tabs = [_q30(oracle, r, N) for r in refs]
    ctx = Q.QLD(H, W, "u16", N, refs, accum=Q.QLD_ACC_FIXED, maps=Q.QLD_MAP_AMP | Q.QLD_MAP_SUMS_I64)
    for k in range(K):
        ctx.set_ref_table_fixed(k, *tabs[k])
    ctx.push_frames(x)
    ctx.demod()
    ctx.sync()
    for k in range(K):
        oI, oQ = oracle.demod_int(x, *tabs[k])
        gI, gQ = [t.cpu().numpy() for t in ctx.get_sums_i64(k)]
        assert np.array_equal(gI, oI) and np.array_equal(gQ, oQ), f"k={k}"
    ctx.destroy()


def test_fixed_own_table_meets_float_tolerance_on_cfg2_shape(Q, oracle):
    from paper_1511_03390_b200 import synth
    wl = synth.cfg2(H=64, W=160, N=1024)
    x = synth.frames(wl.scene, 1, wl.N)
    ref = dict(wl.refs[0])
    ctx = Q.QLD(64, 160, "u16", wl.N, [ref], accum=Q.QLD_ACC_FIXED)
    ctx.push_frames(x)
    ctx.demod()
    ctx.sync()
    worst = check_float_maps(_maps(ctx), oracle_maps(oracle, x, ref), rel=1e-7, what="cfg2-shaped")
    assert worst < 1e-5                                      # even the strict point-wise error
    ctx.destroy()


def test_fixed_rejects_what_it_cannot_do(Q):
    with pytest.raises(Q.QLDError) as e:
        Q.QLD(3, 17, "u8", 16, [{"nu": 0.1}], accum=Q.QLD_ACC_FIXED)            # 51 bytes per frame: not a TMA pitch
    assert e.value.status == Q.QLD_E_UNSUPPORTED
    ctx = Q.QLD(4, 16, "u8", 16, [{"nu": 0.1}], ring_frames=40, accum=Q.QLD_ACC_FIXED)    # rings: int64 sums through k_slide_bulk
    assert ctx.accum_name() == "FIXED"
    ctx.destroy()


def test_auto_moves_k_ge_2_to_the_tensor_cores(Q, oracle):
    """AUTO: K >= 2 float references on a whole-window store -> FIXED (k_demod_tc: the CUDA-core kernel is instruction bound from
    K = 2 on); on a ring, or for K = 1 (the CUDA cores sit on the HBM roof) -> FP32."""
    rng = np.random.default_rng(11)
    H, W, N = 16, 64, 96
    x = rng.integers(0, 4096, size=(N, H, W)).astype(np.uint16)
    refs = [{"nu": 0.07 + 0.09 * k, "phase": 0.2 * k} for k in range(4)]
    ctx = Q.QLD(H, W, "u16", N, refs)
    assert ctx.accum_name() == "FIXED"
    ctx.push_frames(x); ctx.demod(Q.QLD_WHOLE); ctx.sync()
    assert ctx.last_kernel() == "k_demod_tc"
    for k in range(4):
        got = tuple(m.cpu().numpy() for m in ctx.get_maps(k))
        check_float_maps(got, oracle_maps(oracle, x, refs[k]), rel=1e-6, what=f"auto fixed k={k}")
    ctx.destroy()
    for kw, n_refs, want in ((dict(ring_frames=N + 16), 4, "FP32"), (dict(), 1, "FP32"), (dict(), 2, "FIXED"), (dict(), 3, "FIXED")):
        c2 = Q.QLD(H, W, "u16", N, refs[:n_refs], **kw)
        assert c2.accum_name() == want
        c2.destroy()
    c3 = Q.QLD(3, 7, "u8", N, refs)              # 21-byte frames: not a TMA row pitch -> FP32
    assert c3.accum_name() == "FP32"
    c3.destroy()


@pytest.mark.timeout(300, method="thread")
@pytest.mark.parametrize("tile", ["", "4,5,64", "2,8,64", "8,3,64", "1,8,32"])
@pytest.mark.parametrize("H,W,N,K", [(256, 512, 128, 8), (128, 512, 64, 8), (96, 256, 32, 3)])
def test_slow_epilogue_against_a_fast_main_loop(Q, oracle, tile, H, W, N, K):
    """Few frames, many references and every output requested: the epilogue (two warp quartets that advance
    independently) is then much slower than the MMA warp, which runs several tiles' worth of hand-offs ahead of it.  The
    tile-id slots and accumulator sets must not be reused before BOTH quartets are past them (a regression: the second
    quartet once read a later tile's id -- wrong pixels, then a dead-locked barrier).  Exact int64 sums at every pixel."""
    rng = np.random.default_rng(H + N + K)
    x = rng.integers(0, 65536, size=(N, H, W)).astype(np.uint16)
    refs = [{"nu": 0.05 + 0.05 * k, "phase": 0.1 * k} for k in range(K)]
    tabs = [_q30(oracle, r, N) for r in refs]
    mk = forced(Q, "tc", tile)
    ctx = mk(H, W, "u16", N, refs, accum=Q.QLD_ACC_FIXED, maps=Q.QLD_MAP_ALL | Q.QLD_MAP_SUMS_I64)
    for k in range(K):
        ctx.set_ref_table_fixed(k, *tabs[k])
    ctx.push_frames(x)
    for _ in range(3):
        ctx.demod()
    ctx.sync()
    nt = oracle.max_threads()
    for k in range(K):
        oI, oQ = oracle.demod_int(x, *tabs[k], nthreads=nt)
        gI, gQ = [t.cpu().numpy() for t in ctx.get_sums_i64(k)]
        assert np.array_equal(gI, oI) and np.array_equal(gQ, oQ), f"k={k}"
    check_float_maps(_maps(ctx, K - 1), oracle_maps(oracle, x, refs[K - 1]), rel=1e-6, what="slow epilogue")
    ctx.destroy()


# ------------------------------------------------------------------------------------------------ FIXED on a ring (drift-free A5)
@pytest.mark.timeout(300, method="thread")
@pytest.mark.parametrize("dtype,H,W", [("u16", 12, 128), ("u16", 37, 72), ("u8", 9, 144), ("u16be", 16, 64)])
@pytest.mark.parametrize("hop,cap,partial", [(32, 170, False), (32, 170, True), (5, 140, False), (40, 173, False), (64, 200, True)])
@pytest.mark.parametrize("refs", [[{"nu": 0.0937, "phase": 0.3}], [{"nu": 0.4321}, {"num": 1, "den": 6}]])
def test_fixed_point_sliding_is_exact(Q, oracle, dtype, H, W, hop, cap, partial, refs):
    """QLD_ACC_FIXED on a ring (SURVEY.md 8(c) precision ladder item 3): Q1.30 references indexed by absolute
    frame number, int64 sums kept across hops -- every window's sums equal the integer oracle on the same table bit for bit
    (no drift to bound), the table is the rounded oracle table, and the maps meet the float definition to 1e-6."""
    N = 128
    T = N + 7 * hop
    rng = np.random.default_rng(hop + cap + H)
    npdt = np.uint8 if dtype == "u8" else np.uint16
    x = rng.integers(0, 256 if dtype == "u8" else 65536, size=(T, H, W)).astype(npdt)
    raw = x.byteswap() if dtype == "u16be" else x
    ctx = Q.QLD(H, W, dtype, N, refs, ring_frames=cap, accum=Q.QLD_ACC_FIXED, slide_hop=hop if partial else 0)
    assert ctx.accum_name() == "FIXED"
    def q30(ref, s_first, n):                                          # the oracle's table, rounded to Q1.30
        sn, cs = oracle.ref_tables(ref, s_first, n)
        return np.rint(sn * 2.0 ** 30).astype(np.int64), np.rint(cs * 2.0 ** 30).astype(np.int64)

    def push(first, n):
        """push frames first+1 .. first+n; the library's own table entries must be the rounded oracle table (+-1 on rounding
        ties); they are then replaced by the oracle's, so that the exact sums below are compared on the ORACLE's integers"""
        ctx.push_frames(raw[first:first + n])
        for k, ref in enumerate(refs):
            os_, oc = q30(ref, first + 1, n)
            if first + n >= N:
                gs, gc = ctx.read_ref_table_fixed(k)                  # the N most recent entries
                assert np.abs(gs[-n:] - os_).max() <= 1 and np.abs(gc[-n:] - oc).max() <= 1
            ctx.set_ref_table_fixed(k, os_, oc)

    push(0, N)
    ctx.demod(Q.QLD_SLIDE, hop)
    nt = oracle.max_threads()
    for w in range(0, (T - N) // hop + 1):
        if w > 0:
            push(N + (w - 1) * hop, hop)
            ctx.demod(Q.QLD_SLIDE, hop)
        ctx.sync()
        assert ctx.last_kernel() == "k_slide_bulk"
        a = w * hop
        for k, ref in enumerate(refs):
            os_, oc = q30(ref, a + 1, N)
            oI, oQ = oracle.demod_int(x[a:a + N], os_, oc, nthreads=nt)
            gI, gQ = [t.cpu().numpy() for t in ctx.get_sums_i64(k)]
            assert np.array_equal(gI, oI) and np.array_equal(gQ, oQ), f"window {w} k={k}"
            check_float_maps(_maps(ctx, k), oracle_maps(oracle, x[a:a + N], ref, s_first=a + 1), rel=1e-6, what=f"window {w} k={k}")
    ctx.destroy()


def test_fixed_point_ring_limits(Q):
    with pytest.raises(Q.QLDError) as e:
        Q.QLD(8, 64, "u16", 32, [{"nu": 0.1}, {"nu": 0.2}, {"nu": 0.3}], ring_frames=64, accum=Q.QLD_ACC_FIXED)
    assert e.value.status == Q.QLD_E_UNSUPPORTED
    with pytest.raises(Q.QLDError) as e:
        Q.QLD(3, 5, "u16", 32, [{"nu": 0.1}], ring_frames=64, accum=Q.QLD_ACC_FIXED)          # 30 bytes per frame
    assert e.value.status == Q.QLD_E_UNSUPPORTED


# ------------------------------------------------------------------------------------------------ integer bins on the tensor cores
@pytest.mark.timeout(300, method="thread")
@pytest.mark.parametrize("tile", ["8,3,64", "4,5,64", "2,8,32", "1,8,64"])
@pytest.mark.parametrize("dtype,H,W,N", [("u8", 50, 128, 70), ("u16", 37, 48, 129), ("u16", 16, 200, 64), ("u16be", 24, 128, 33), ("u8", 33, 256, 9)])
@pytest.mark.parametrize("refs", [[{"num": 1, "den": 8}], [{"num": 1, "den": 6}], [{"num": 1, "den": 4}, {"num": 3, "den": 16, "phase": 0.4}], [{"num": 2, "den": 5}]])
def test_integer_bins_on_the_tensor_cores(Q, oracle, tile, dtype, H, W, N, refs):
    """A3' as a one-digit int8 contraction (the bin indicators 0, +1, -1 are the B operand): int32 bins bit-exact against the
    int64 oracle for every tile shape, sample format and bin layout (even den: difference rows; odd den: plain bins; two
    references), maps to 1e-6."""
    rng = np.random.default_rng(H * N)
    npdt = np.uint8 if dtype == "u8" else np.uint16
    x = rng.integers(0, 256 if dtype == "u8" else 65536, size=(N, H, W)).astype(npdt)
    raw = x.byteswap() if dtype == "u16be" else x
    mk = forced(Q, "tc", tile)
    ctx = mk(H, W, dtype, N, refs, accum=Q.QLD_ACC_INT_BINS)
    ctx.push_frames(raw)
    ctx.demod()
    ctx.demod()
    ctx.sync()
    assert ctx.last_kernel() == "k_demod_tc"
    for k, ref in enumerate(refs):
        den, num = ref["den"], ref["num"]
        B = oracle.bins(x, num, den)
        exp = B[:den // 2] - B[den // 2:] if den % 2 == 0 else B
        assert np.array_equal(ctx.get_bins(k).cpu().numpy(), exp), f"k={k}"
        check_float_maps(_maps(ctx, k), oracle_maps(oracle, x, ref), rel=1e-6, what=f"tc bins k={k}")
    ctx.destroy()
