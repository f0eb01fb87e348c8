"""The N > 1 path on CPU: two processes over gloo (127.0.0.1) exercise the sharding plumbing of
paper_1511_03390_b200.shard: row bands tile the frame, per-band results concatenate to the whole-frame
result (pixels are independent, PAPER.md:99 -- checked with the oracle), bands gather into whole maps, and the
whole-job rate is (sum of units) / (max of times).  No CUDA here; the per-band compute is the oracle, which tests may call."""
import os
import socket

import numpy as np
import pytest


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, H: int, W: int, N: int, out_dir: str):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from paper_1511_03390_b200 import shard, synth
        wl = synth.cfg2(H=H, W=W, N=N)
        frames = synth.frames(wl.scene, 1, N)                   # every rank can regenerate any frame (counter-based)
        bands = shard.row_bands(H, world)
        shard.check_partition(bands, H)
        mine = shard.band_of(frames, bands[rank])
        ref = dict(wl.refs[0])
        I, Q, A, P = oracle.qld(mine, ref) if mine.shape[1] else (np.zeros((0, W)),) * 4
        band_maps = torch.from_numpy(np.stack([I, Q, A, P]).astype(np.float64))
        whole = shard.gather_row_bands(band_maps, H, dist)
        # whole-job rate: rank r "processed" (r + 1) * 1000 units in (2 - r) seconds
        rate, units, secs = shard.whole_job_rate(1000.0 * (rank + 1), 2.0 - rank, dist)
        np.save(os.path.join(out_dir, f"whole_{rank}.npy"), whole.numpy())
        np.save(os.path.join(out_dir, f"rate_{rank}.npy"), np.array([rate, units, secs]))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("H", [9, 16])
def test_row_band_sharding_two_ranks_gloo(tmp_path, oracle, H):
    import torch.multiprocessing as mp
    from paper_1511_03390_b200 import synth
    W, N, world = 24, 40, 2
    port = _free_port()
    mp.spawn(_worker, args=(world, port, H, W, N, str(tmp_path)), nprocs=world, join=True)
    wl = synth.cfg2(H=H, W=W, N=N)
    frames = synth.frames(wl.scene, 1, N)
    ref = np.stack(oracle.qld(frames, dict(wl.refs[0])))
    for rank in range(world):
        got = np.load(tmp_path / f"whole_{rank}.npy")
        assert got.shape == ref.shape and np.array_equal(got, ref), f"rank {rank}: gathered bands differ from the whole-frame result"
        rate, units, secs = np.load(tmp_path / f"rate_{rank}.npy")
        assert units == 3000.0 and secs == 2.0 and rate == 1500.0


def test_row_bands_properties():
    from paper_1511_03390_b200 import shard
    for H in (0, 1, 7, 8, 1024, 2160):
        for world in (1, 2, 3, 4, 8):
            bands = shard.row_bands(H, world)
            shard.check_partition(bands, H)
            sizes = [b - a for a, b in bands]
            assert len(bands) == world and max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard.row_bands(8, 0)
    assert shard.stream_seed(2, 0) == 2 and shard.stream_seed(2, 3) == 3002
    # single-process fall-through: no process group needed
    assert shard.whole_job_rate(10.0, 2.0) == (5.0, 10.0, 2.0)


@pytest.mark.gpu
@pytest.mark.parametrize("name,shape,accum_name", [("cfg2", dict(H=301, W=256, N=96), "FP32"), ("cfg4", dict(H=256, W=512, N=128), "AUTO"),
                                                   ("cfg1", dict(H=203, W=320, N=64), "AUTO")])
def test_row_bands_through_libqld_on_one_gpu(name, shape, accum_name):
    """SURVEY.md 8(e) with the product, not the oracle: world = 2 row bands of one frame, each through its own libqld
    context on its own stream (what two ranks would run), concatenate to exactly the maps of one whole-frame context --
    bit for bit, because a pixel's sums depend on that pixel only.  Integer bins and the fixed-point
    contraction are exact in any order; the fp32 kernel's summation order depends on its tile shape (time slices), which
    the launcher picks from the frame size, so the FP32 case pins one shape for the three contexts."""
    import torch
    assert torch.cuda.is_available(), "needs the B200"
    from paper_1511_03390_b200 import qld, shard, synth
    wl = synth.BUILDERS[name](**shape)
    sc, N, K = wl.scene, wl.N, len(wl.refs)
    refs = [dict(r) for r in wl.refs]
    frames = qld.synth_fill(sc, 1, N)
    accum = getattr(qld, "QLD_ACC_" + accum_name)
    tile = ("stream", 1024, 16) if accum_name == "FP32" else None
    whole = qld.QLD(sc.H, sc.W, sc.dtype, N, refs, ring_frames=-1, accum=accum, max_value=sc.maxval, debug_tile=tile)
    whole.attach_frames_device(frames)
    whole.demod(qld.QLD_WHOLE)
    whole.sync()
    bands = shard.row_bands(sc.H, 2)
    shard.check_partition(bands, sc.H)
    parts, keep = [], []
    for band in bands:
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            sub = shard.band_of(frames, band)
            ctx = qld.QLD(band[1] - band[0], sc.W, sc.dtype, N, refs, ring_frames=-1, accum=accum, max_value=sc.maxval, debug_tile=tile)
            ctx.attach_frames_device(sub)
            ctx.demod(qld.QLD_WHOLE)
        keep.append((ctx, sub, st))
    for ctx, _, _ in keep:
        ctx.sync()
        assert ctx.accum_mode() == whole.accum_mode()
        parts.append([torch.stack([m for m in ctx.get_maps(k)]) for k in range(K)])
    for k in range(K):
        cat = torch.cat([p[k] for p in parts], dim=-2)
        ref = torch.stack([m for m in whole.get_maps(k)])
        assert torch.equal(cat.view(torch.int32), ref.view(torch.int32)), f"{name} k={k}: bands differ from the whole-frame maps"
    for ctx, _, _ in keep:
        ctx.destroy()
    whole.destroy()


@pytest.mark.gpu
@pytest.mark.timeout(600, method="thread")
@pytest.mark.parametrize("shard_mode,scaling", [("rows", "strong"), ("stacks", "weak")])
def test_bench_spawns_ranks_and_shards(shard_mode, scaling):
    """`python bench.py --gpus 2` outside torchrun re-executes itself with two ranks (on a one-GPU box they share the device and
    the host collectives go over gloo: a plumbing check).  --shard rows: the two ranks split ONE cfg1 frame into row bands, each
    through libqld; rank 0's band is checked against the oracle inside the bench; the line says n_gpus = 2."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--shard", shard_mode, "--workload", "cfg1", "--steps", "10",
                          "--e2e-steps", "1", "--also", "none", "--ref-rows", "16"], capture_output=True, text=True, timeout=500, env=env)
    assert out.returncode == 0, out.stderr[-800:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["n_gpus"] == 2 and line["scaling"] == scaling and line["value"] > 0 and line["parity"]["ok"]
    assert line["e2e"]["value"] > 0 and line["gpu_launches"] >= 10
    import torch
    assert ("oversubscribed" in line) == (torch.cuda.device_count() < 2)
