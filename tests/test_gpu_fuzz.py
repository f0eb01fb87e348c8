"""Seeded random sweep of the whole-window and sliding paths against the oracle: shapes (ragged rows, 1-pixel frames,
row pitches that do and do not suit the TMA kernels), dtypes, window lengths, reference counts, accumulation modes and
forced tile shapes, 120 cases.  Tolerances as everywhere: bins / fixed-point 1e-6, fp32 1e-5 (floored at the map median)."""
import os

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


def _case(seed):
    rng = np.random.default_rng(1000 + seed)
    dtype = np.uint8 if rng.random() < 0.4 else np.uint16
    H = int(rng.choice([1, 2, 3, 7, 12, 16, 31, 40]))
    W = int(rng.choice([1, 5, 16, 24, 48, 64, 100, 128, 200, 256]))
    N = int(rng.choice([1, 2, 7, 16, 33, 64, 100, 129, 256]))
    K = int(rng.choice([1, 1, 1, 2, 3, 4, 8]))
    kind = rng.choice(["fp32", "bins", "fixed", "auto"])
    refs = []
    for k in range(K):
        if kind == "bins" or (kind == "auto" and rng.random() < 0.5):
            den = int(rng.choice([3, 4, 5, 6, 8, 12, 16]))
            num = int(rng.integers(1, (den - 1) // 2 + 1))
            if 2 * num >= den:
                num = 1
            refs.append({"num": num, "den": den, "phase": float(rng.choice([0.0, 0.7]))})
        else:
            refs.append({"nu": float(rng.uniform(0.01, 0.49)), "phase": float(rng.uniform(-3, 3))})
    tile = rng.choice(["", "512,16", "1024,16", "2048,16", "256,32", "1024,32"])
    return rng, dtype, H, W, N, K, kind, refs, tile


@pytest.mark.parametrize("seed", range(120))
def test_random_configuration(Q, oracle, seed):
    rng, dtype, H, W, N, K, kind, refs, tile = _case(seed)
    mk = forced(Q, "stream", tile)
    hi = 256 if dtype == np.uint8 else int(rng.choice([4096, 65536]))
    x = rng.integers(0, hi, size=(N, H, W)).astype(dtype) if rng.random() < 0.5 else \
        np.clip(rng.normal(hi / 3, hi / 40, size=(N, H, W)), 0, hi - 1).astype(dtype)
    accum = {"fp32": Q.QLD_ACC_FP32, "bins": Q.QLD_ACC_INT_BINS, "fixed": Q.QLD_ACC_FIXED, "auto": Q.QLD_ACC_AUTO}[kind]
    try:
        ctx = mk(H, W, "u8" if dtype == np.uint8 else "u16", N, refs, accum=accum, max_value=hi - 1)
    except Q.QLDError as e:
        # the only legitimate refusals: bins with too many rows / an int32 bound, fixed point on a frame that is not
        # a multiple of 16 bytes
        assert e.status == Q.QLD_E_UNSUPPORTED, (kind, refs, H, W, N)
        rows = sum((r["den"] // 2 if r["den"] % 2 == 0 else r["den"]) for r in refs if "den" in r)
        assert (kind == "bins" and (rows > 16 or (hi - 1) * (N // min(r["den"] for r in refs) + 2) >= 2 ** 31)) or \
               (kind == "fixed" and (H * W * x.itemsize) % 16 != 0)
        return
    mode = ctx.accum_name()
    ctx.push_frames(x)
    ctx.demod(Q.QLD_WHOLE)
    ctx.sync()
    for k in range(K):
        got = tuple(None if m is None else m.cpu().numpy() for m in ctx.get_maps(k))
        check_float_maps(got, oracle_maps(oracle, x, refs[k]), rel=1e-5 if mode == "FP32" else 1e-6,
                         what=f"seed {seed} {mode} {ctx.last_kernel()} {H}x{W} N={N} K={K} k={k} tile={tile!r}")
    ctx.destroy()


@pytest.mark.timeout(300, method="thread")
@pytest.mark.parametrize("seed", range(80))
def test_random_sliding(Q, oracle, seed):
    rng = np.random.default_rng(5000 + seed)
    tile = rng.choice(["512,16", "1024,16", "2048,16", "1024,32", ""])
    mk = forced(Q, "stream", tile)
    H, W = int(rng.choice([4, 9, 16])), int(rng.choice([16, 64, 128, 136]))
    hop = int(rng.choice([1, 3, 8, 16, 24, 32, 64]))
    N = hop * int(rng.integers(1, 5)) if rng.random() < 0.6 else int(rng.integers(max(hop, 2), 160))
    N = max(N, hop)
    partial = bool(N % hop == 0 and hop >= 32 and tile and rng.random() < 0.6)
    cap = N + hop + int(rng.integers(1, 40))
    n_hops = 6
    T = N + n_hops * hop
    kind = rng.choice(["bins", "fp32"])
    ref = {"num": 1, "den": int(rng.choice([4, 6, 8]))} if kind == "bins" else {"nu": float(rng.uniform(0.02, 0.48)), "phase": 0.3}
    stream = np.clip(rng.normal(1500, 60, size=(T, H, W)), 0, 4095).astype(np.uint16)
    bulk = int(rng.integers(0, 3))                              # 0: automatic, 1: force k_slide_bulk, 2: never
    if (H * W * 2) % 16 != 0 and bulk == 1:
        bulk = 0
    try:
        ctx = mk(H, W, "u16", N, [ref], ring_frames=cap, accum=Q.QLD_ACC_INT_BINS if kind == "bins" else Q.QLD_ACC_FP32, max_value=4095,
                    slide_hop=hop if partial else 0)
        ctx.debug_set_tile("slide", bulk)
        ctx.push_frames(stream[:N])
        ctx.demod(Q.QLD_SLIDE, hop)
    except Q.QLDError as e:
        assert partial and e.status == Q.QLD_E_UNSUPPORTED          # hop shorter than a stage of the forced tile
        return
    for w in range(n_hops + 1):
        if w > 0:
            ctx.push_frames(stream[N + (w - 1) * hop:N + w * hop])
            ctx.demod(Q.QLD_SLIDE, hop)
        ctx.sync()
        got = tuple(m.cpu().numpy() for m in ctx.get_maps(0))
        check_float_maps(got, oracle_maps(oracle, stream[w * hop:w * hop + N], ref, s_first=w * hop + 1), rel=1e-6 if kind == "bins" else 1e-5,
                         what=f"seed {seed} window {w} {kind} {ctx.last_kernel()} {H}x{W} N={N} hop={hop} cap={cap} tile={tile!r} partial={partial} bulk={bulk}")
    ctx.destroy()
