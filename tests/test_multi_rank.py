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
