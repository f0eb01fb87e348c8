"""Multi-GPU plumbing of the QLD hot path: host logic only, no arithmetic of the method.

Pixels are independent (R(j,k) depends only on pixel (j,k)'s time series), so the path shards with
no collective on it:

  * independent stacks / camera streams: one per rank (what `bench.py --gpus N` times, "weak" scaling);
  * one large frame: contiguous row bands, one per rank; each rank ingests only its band of every frame and
    produces its band of every map.  A consumer that wants whole maps gathers the bands afterwards
    (`gather_row_bands`, one all_gather of K*H*W*4 bytes per map, off the hot path).

`torch.distributed` (NCCL on the GPUs, gloo in the CPU tests) carries the barrier, the max-over-ranks timing and
the optional gather.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple


def row_bands(H: int, world: int) -> List[Tuple[int, int]]:
    """Contiguous row bands [r0, r1) covering 0..H, sizes differing by at most one row, larger bands first.
    Ranks beyond H get empty bands."""
    if H < 0 or world < 1:
        raise ValueError("row_bands: need H >= 0 and world >= 1")
    base, extra = divmod(H, world)
    out, r0 = [], 0
    for rank in range(world):
        n = base + (1 if rank < extra else 0)
        out.append((r0, r0 + n))
        r0 += n
    return out


def band_of(frames, band: Tuple[int, int]):
    """Rows band[0]..band[1]-1 of a [n, H, W] stack (numpy array or torch tensor), as a contiguous stack."""
    sub = frames[:, band[0]:band[1], :]
    return sub.contiguous() if hasattr(sub, "contiguous") else sub.copy()


def stream_seed(base_seed: int, rank: int) -> int:
    """Seed of the synthetic stack / stream that rank `rank` processes (rank 0 keeps the BASELINE.json seed)."""
    return int(base_seed) + 1000 * int(rank)


def whole_job_rate(units_local: float, seconds_local: float, dist=None, device=None) -> Tuple[float, float, float]:
    """(units of all ranks) / (max over ranks of the timed seconds): returns (rate, total_units, max_seconds)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return units_local / seconds_local, units_local, seconds_local
    import torch
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    t = torch.tensor([float(seconds_local)], dtype=torch.float64, device=device)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(u.item()) / float(t.item()), float(u.item()), float(t.item())


def gather_row_bands(band_map, H: int, dist=None):
    """Whole [.., H, W] map on every rank from the ranks' row bands [.., h_rank, W] (off the hot path).
    Bands may differ by one row, so they are padded to the largest band for the all_gather."""
    import torch
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return band_map
    world = dist.get_world_size()
    bands = row_bands(H, world)
    hmax = max(b[1] - b[0] for b in bands)
    lead, W = tuple(band_map.shape[:-2]), band_map.shape[-1]
    padded = torch.zeros(lead + (hmax, W), dtype=band_map.dtype, device=band_map.device)
    padded[..., :band_map.shape[-2], :] = band_map
    parts = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded)
    return torch.cat([p[..., :b[1] - b[0], :] for p, b in zip(parts, bands)], dim=-2)


def check_partition(bands: Sequence[Tuple[int, int]], H: int) -> None:
    """Raise unless the bands tile 0..H exactly, in order."""
    r = 0
    for a, b in bands:
        if a != r or b < a:
            raise AssertionError(f"bands do not tile the frame: {bands}")
        r = b
    if r != H:
        raise AssertionError(f"bands cover {r} rows of {H}")
