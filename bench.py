#!/usr/bin/env python
"""bench.py -- QLD pixel-samples/s on one node, through the C-ABI library (libqld.so).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A step is one pass of the hot path over one batch of synthetic frames of the named BASELINE.json config.
Whole-window workloads (cfg0, cfg1, cfg2, cfg4): one window of N frames -> qld_demod(QLD_WHOLE) = A3/A3'/A6
demodulation + A4 finalise (reference tables, A1, were built by qld_create).  Streaming workload (cfg3): one
batch of `hop` new frames -> qld_commit_frames (A1 table extension + A2 without a copy: frames are resident)
-> qld_demod(QLD_SLIDE) = A5 update + A4.  `value` has the frames resident in HBM; `e2e` runs the same step
from pinned host buffers: qld_push_frames (A2), qld_demod, qld_read_map of the amplitude map(s) to the host.
The headline workload is cfg4 (BASELINE.json configs[4], 17.2 GB, K = 8: the largest single-GPU config).  With the default
flags at N = 1 the other configs (cfg2, cfg3 sliding, cfg1) are run briefly first and each prints its own compact JSON line
(marked "also": "<cfg>"); the LAST line is the contract's line for the headline workload, carrying a short summary of the
others under "also".  `--gpus N` without a torchrun environment re-executes itself under torch.distributed.run with N ranks;
`--shard rows` makes the ranks split ONE frame into row bands (strong scaling) instead of running one
independent stack each (weak scaling, the default).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "qld_pixel_samples_per_s"
UNIT = "pixel-samples/s"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy read+write)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                 "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10, "applications_clocks_setting": 0x2}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.004)

    def result(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def build_workload(name: str, rank: int, shard_rows: bool = False):
    from paper_1511_03390_b200 import shard, synth
    # BASELINE.json seeds: cfgN -> seed N on rank 0; row sharding: every rank sees the same frame (same seed)
    return synth.BUILDERS[name](seed=shard.stream_seed(int(name[3]), 0 if shard_rows else rank))


def oracle_on_rows(wl, frames_rows_host, refs, nthreads):
    """Oracle (as it stands) on a host sample [N, rows, W]; returns list of (I, Q, amp, phase) and seconds."""
    import oracle
    t0 = time.perf_counter()
    out = [oracle.qld(frames_rows_host, r, s_first=1, nthreads=nthreads) for r in refs]
    return out, time.perf_counter() - t0


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only), on a bounded sample."""
    if rank != 0:
        return
    import numpy as np
    import oracle
    from paper_1511_03390_b200 import synth
    wl = build_workload(args.workload, 0)
    sc = wl.scene
    rows = max(1, min(sc.H, int(args.ref_rows) or 32))
    pix = np.arange(rows * sc.W)                       # the first `rows` rows of the frame
    x = synth.series(sc, pix, 1, wl.N).reshape(wl.N, rows, sc.W)
    nt = oracle.max_threads()
    refs = [dict(r) for r in wl.refs]
    for _ in range(args.warmup):
        oracle_on_rows(wl, x, refs, nt)
    t = 0.0
    for _ in range(args.steps):
        t += oracle_on_rows(wl, x, refs, nt)[1]
    # streaming workload: a step is one hop; the oracle recomputes the whole window for it (never incremental)
    per_step = float(wl.hop * rows * sc.W) if args.workload == "cfg3" else float(x.size)
    samples = per_step * args.steps
    val = samples / t
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f80 (x87 long double) / int64", "data": "synthetic",
            "config": {"workload": args.workload, "H": sc.H, "W": sc.W, "N": wl.N, "K": len(refs),
                       "sample": f"first {rows} rows x {sc.W} cols x {wl.N} frames per step"
                                 + (f" (one window recomputed per hop of {wl.hop} frames; value counts the hop's new samples)" if args.workload == "cfg3" else "")},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": nt, "kind": "oracle",
                             "sample": f"{rows} rows x {sc.W} x {wl.N} frames ({x.size} samples) per step"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)




ACCUM_NAMES = {"auto": 0, "fp32": 1, "bins": 2, "fixed": 3, "refs": 4}


class Env:
    """Rank / device / barrier plumbing shared by the workload runners."""

    def __init__(self, args):
        import torch
        self.torch = torch
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
        n_dev = torch.cuda.device_count()
        # fewer GPUs than ranks (a one-GPU box exercising the N > 1 code path): ranks share devices and the host-side
        # collectives go over gloo -- the ranks' kernels are independent of one another, only the timing barriers are shared.
        # Such a run checks the plumbing; its numbers are not a scaling measurement and the line says so.
        self.oversubscribed = self.world > n_dev
        self.local_dev = self.local_rank % n_dev
        torch.cuda.set_device(self.local_dev)
        self.dev = torch.device("cuda", self.local_dev)
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            if self.oversubscribed:
                dist.init_process_group("gloo")
            else:
                dist.init_process_group("nccl", device_id=self.dev)
            self.dist = dist
        self.red_dev = torch.device("cpu") if self.oversubscribed else self.dev

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def max_over_ranks(self, x: float) -> float:
        if self.dist is None:
            return x
        t = self.torch.tensor([x], device=self.red_dev, dtype=self.torch.float64)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(self, x: float) -> float:
        if self.dist is None:
            return x
        t = self.torch.tensor([x], device=self.red_dev, dtype=self.torch.float64)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        return float(t.item())

    def timed(self, step, steps: int, warmup: int, keep_busy=None, counter=None):
        """warmup untimed steps, then exactly `steps` steps between CUDA events on the launching stream (torch's
        current stream is the context's compute stream), barrier + synchronize on both sides, max over ranks.
        `counter()` (kernel launches so far) is read on both sides of the timed region.
        Returns (ms, clocks, launches)."""
        torch = self.torch
        for _ in range(warmup):
            step()
        self.barrier()
        sampler = ClockSampler(self.local_dev)
        sampler.start()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        self.barrier()
        c0 = counter() if counter else 0
        ev0.record()
        for _ in range(steps):
            step()
        ev1.record()
        self.barrier()
        ms = ev0.elapsed_time(ev1)
        launches = (counter() - c0) if counter else None
        # keep the GPU busy a little longer if the region was too short for a clock sample
        t_end = time.time() + 0.25
        while keep_busy is not None and len(sampler.samples) < 8 and time.time() < t_end:
            keep_busy()
            torch.cuda.synchronize()
        sampler.stop_flag = True
        sampler.join()
        return self.max_over_ranks(ms), sampler.result(), launches


def load_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
    `ncu --set full` summaries (profiles/r03_traffic.csv, the DRAM bytes of profiles/r03_ncu_full.md); None if absent."""
    tpath = os.path.join(ROOT, "profiles", "r03_traffic.csv")
    try:
        for line in open(tpath).read().splitlines()[1:]:
            w, k, v = line.split(",")
            if w == workload and k == kernel:
                return float(v)
    except Exception:
        pass
    return None


READ_CEILING = {}        # filled once per process by measure_read_ceiling()


def measure_read_ceiling(env, gib: int = 16, iters: int = 5):
    """what this GPU sustains on READS alone -- qld_probe_read (a plain read-only sum kernel of the library) over a
    16 GiB buffer, CUDA events around `iters` launches after 3 untimed ones.  The paths here read every sample once and write
    almost nothing, so this, not the read+write copy figure of MEASURED_PEAKS.json, is the ceiling they can approach."""
    torch = env.torch
    from paper_1511_03390_b200 import qld
    try:
        buf = torch.empty(gib << 30, dtype=torch.uint8, device=env.dev)
    except Exception as e:                                       # noqa: BLE001 -- e.g. many ranks sharing one device
        READ_CEILING.update({"read_ceiling_GBps": None, "read_ceiling_note": f"not measured: {type(e).__name__}"})
        return
    out = torch.zeros(qld.QLD_PROBE_OUT_WORDS, dtype=torch.int32, device=env.dev)
    for _ in range(3):
        qld.probe_read(buf, out)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(iters):
        qld.probe_read(buf, out)
    ev1.record()
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / iters
    READ_CEILING.update({"read_ceiling_GBps": (gib << 30) / (ms * 1e-3) / 1e9,
                         "read_ceiling_note": f"qld_probe_read (k_probe_read, read-only sum) over {gib} GiB, mean of {iters} launches, this run"})
    del buf
    torch.cuda.empty_cache()


def roofline_hbm(algo_bytes: float, ms_per_launch: float, workload: str, kernel: str, notes=None):
    peak, peak_src = load_peaks()
    achieved = algo_bytes / (ms_per_launch * 1e-3) / 1e9
    r = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
         "traffic": load_traffic(workload, kernel), "peak_source": peak_src, "algorithmic_bytes_per_launch": algo_bytes,
         "frac_of_nominal_8TBps": achieved / 8000.0, "kernel": kernel}
    if READ_CEILING.get("read_ceiling_GBps"):
        r["read_ceiling_GBps"] = READ_CEILING["read_ceiling_GBps"]
        r["frac_of_read_ceiling"] = achieved / READ_CEILING["read_ceiling_GBps"]
        r["read_ceiling_note"] = READ_CEILING["read_ceiling_note"]
    if notes:
        r["note"] = notes
    return r


def bench_whole(env: Env, args, workload: str, accum_name: str, steps: int, warmup: int, e2e_steps: int, with_cpu: bool):
    """Whole-window workloads (8(a) rows A1, A3/A3'/A6, A4; A2 in the e2e leg)."""
    torch = env.torch
    from paper_1511_03390_b200 import qld
    from paper_1511_03390_b200 import shard
    shard_rows = args.shard == "rows" and env.world > 1
    wl = build_workload(workload, env.rank, shard_rows)
    sc = wl.scene
    N, H_full, W, K = wl.N, sc.H, sc.W, len(wl.refs)
    b = 1 if sc.dtype == "u8" else 2
    refs = [dict(r) for r in wl.refs]
    accum = ACCUM_NAMES[accum_name]
    # inputs: the synthetic stack, filled on the device, resident before the timed region
    if shard_rows:
        # one frame, contiguous row bands, one per rank; this rank keeps only its band of every frame
        r_lo, r_hi = shard.row_bands(H_full, env.world)[env.rank]
        H = r_hi - r_lo
        frames = torch.empty((N, H, W), dtype=torch.uint8 if b == 1 else torch.uint16, device=env.dev)
        for a in range(0, N, 64):
            n = min(64, N - a)
            frames[a:a + n].copy_(qld.synth_fill(sc, a + 1, n, device=env.dev)[:, r_lo:r_hi, :])
    else:
        r_lo, H = 0, H_full
        frames = qld.synth_fill(sc, 1, N, device=env.dev)
    torch.cuda.synchronize()
    # BASELINE.json configs[4] asks for the K amplitude maps only; the other configs produce all four maps
    maps, map_names = (qld.QLD_MAP_AMP, "amplitude") if workload == "cfg4" else (qld.QLD_MAP_ALL, "I,Q,amplitude,phase")
    n_maps = 1 if workload == "cfg4" else 4
    ctx = qld.QLD(H, W, sc.dtype, N, refs, ring_frames=-1, accum=accum, maps=maps, max_value=sc.maxval)
    ctx.attach_frames_device(frames)

    def step():
        ctx.demod(qld.QLD_WHOLE)

    ms, clocks, launches = env.timed(step, steps, warmup, keep_busy=step, counter=ctx.kernel_launches)
    kernel = ctx.last_kernel()
    mode = ctx.accum_name()
    samples = float(N) * H * W                               # this rank's units per step
    job_samples = env.sum_over_ranks(samples)                # row bands may differ by one row
    res = {"workload": workload, "value": job_samples * steps / (ms * 1e-3), "ms_per_step": ms / steps,
           "maps_per_s": (1 if shard_rows else env.world) * K * steps / (ms * 1e-3), "clocks": clocks, "kernel": kernel,
           "scaling": "strong" if shard_rows else "weak"}
    res["gpu_launches"] = int(launches)
    algo = samples * b + n_maps * K * H * W * 4.0            # every sample once + the fp32 maps of every reference
    in_l2 = samples * b <= 126e6
    res["roofline"] = roofline_hbm(algo, ms / steps, workload, kernel,
                                   "input fits the 126 MB L2 and is re-read every step: L2-resident, not an HBM number" if in_l2 else None)
    res["dtype"] = {"INT_BINS": "int32", "INT_REFS": "int32", "FIXED": "int8 x int8 -> int32 -> int64 (tcgen05)", "FP32": "f32"}[mode]
    res["config"] = {"workload": workload, "H": H, "W": W, "N": N, "K": K, "input_dtype": sc.dtype, "accum": mode,
                     "maps": map_names, "step": "qld_demod(QLD_WHOLE) over the resident stack",
                     "cache": f"input {samples * b / 1e6:.0f} MB per step " + ("<= 126 MB L2: L2-resident" if in_l2 else "> 126 MB L2: no flush needed"),
                     "parallelism": (f"one {H_full}x{W} frame split into {env.world} row bands, one per rank (pixels are independent; no collective)"
                                     if shard_rows else f"{env.world} x independent stacks (pixels are independent; no collective)")}

    # ---- end to end through host buffers (pinned): push + demod + read amplitude maps back ---------
    if e2e_steps > 0:
        host = torch.empty((N, H, W), dtype=frames.dtype, pin_memory=True)
        host.copy_(frames)
        amp_host = torch.empty((K, H, W), dtype=torch.float32, pin_memory=True)
        torch.cuda.synchronize()
        ectx = qld.QLD(H, W, sc.dtype, N, refs, ring_frames=0, accum=accum, maps=maps, max_value=sc.maxval)
        chunk = max(1, min(N, (256 << 20) // (H * W * b)))       # pushes of about 256 MiB

        def e2e_step():
            ectx.reset()
            for a in range(0, N, chunk):
                ectx.push_frames(host[a:a + chunk])
            ectx.demod(qld.QLD_WHOLE)
            for k in range(K):
                ectx.read_map(k, qld.QLD_MAP_AMP, amp_host[k])
            ectx.sync()

        e2e_step()
        env.barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        env.barrier()
        dt = env.max_over_ranks(time.perf_counter() - t0)
        res["e2e"] = {"value": job_samples * e2e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": int(samples * b),
                      "d2h_bytes_per_step": int(K * H * W * 4), "ms_per_step": 1e3 * dt / e2e_steps,
                      "h2d_GBps": samples * b * e2e_steps / dt / 1e9, "steps": e2e_steps,
                      "note": "pinned host stack -> qld_push_frames -> qld_demod -> qld_read_map(amp) -> host"}
        ectx.destroy()
        del host

    # ---- CPU baseline (the oracle, as it stands) + parity of the timed configuration on the same rows
    if with_cpu and env.rank == 0:
        import oracle
        from oracle.check import check_float_maps
        nt = oracle.max_threads()
        # about 15 s of oracle work at ~1.4e8 sample-references per second per core
        rows = max(1, min(H, args.ref_rows or -(-int(15 * 1.4e8 * nt) // (K * N * W))))
        r0 = (H // 2 - rows // 2)
        sub = frames[:, r0:r0 + rows, :].contiguous().cpu().numpy()
        oracle_on_rows(wl, sub[:8], refs[:1], nt)                      # thread pool warm-up
        out, secs = oracle_on_rows(wl, sub, refs, nt)
        res["cpu_baseline"] = {"value": float(sub.size) / secs, "unit": UNIT, "cores": nt, "kind": "oracle",
                               "sample": f"rows {r0}..{r0 + rows - 1} x {W} cols x {N} frames x {K} refs = {sub.size} samples, {secs:.2f} s"}
        # the paper's other CPU figure (one thread): the same oracle on one core, on a sixteenth of the rows
        r1 = max(1, rows // 16)
        _, secs1 = oracle_on_rows(wl, sub[:, :r1], refs, 1)
        res["cpu_baseline"]["single_thread"] = {"value": float(sub[:, :r1].size) / secs1, "unit": UNIT, "cores": 1,
                                                "sample": f"{r1} rows x {W} x {N} frames x {K} refs, {secs1:.2f} s"}
        ctx.demod(qld.QLD_WHOLE)
        ctx.sync()
        worst = 0.0
        tol = 1e-5 if mode == "FP32" else 1e-6
        for k in range(K):
            got = tuple(None if m is None else m[r0:r0 + rows].cpu().numpy() for m in ctx.get_maps(k))
            worst = max(worst, check_float_maps(got, out[k], rel=tol, what=f"bench parity k={k}"))
        res["parity"] = {"rows_checked": rows, "refs_checked": K, "tolerance": f"{tol:g} relative, floored at the map median",
                         "strict_max_rel_err_amp": worst, "ok": True}
    ctx.destroy()
    del frames
    torch.cuda.empty_cache()
    return res


def bench_slide(env: Env, args, workload: str, accum_name: str, steps: int, warmup: int, e2e_steps: int, with_cpu: bool):
    """Streaming workload cfg3 (8(a) rows A1, A2, A5, A4): one step = one batch of `hop` new frames -> one map."""
    torch = env.torch
    from paper_1511_03390_b200 import qld, synth
    wl = build_workload(workload, env.rank)
    sc = wl.scene
    N, H, W, K, hop = wl.N, sc.H, sc.W, len(wl.refs), wl.hop
    b = 1 if sc.dtype == "u8" else 2
    tdt = torch.uint8 if b == 1 else torch.uint16
    refs = [dict(r) for r in wl.refs]
    accum = ACCUM_NAMES[accum_name]
    maps = qld.QLD_MAP_AMP                                   # BASELINE.json configs[3]: one amplitude map per hop
    # inputs resident in HBM: the first T frames of the stream, written in place into the (external) ring
    n_hops = warmup + steps
    T = min(sc.n_frames, N + n_hops * hop)
    ring = torch.empty((T, H, W), dtype=tdt, device=env.dev)
    for a in range(0, T, 256):
        qld.synth_fill(sc, a + 1, min(256, T - a), out=ring[a:a + 256])
    torch.cuda.synchronize()
    slide_hop = 0 if args.reread_expired else hop
    ctx = qld.QLD(H, W, sc.dtype, N, refs, ring_frames=T, accum=accum, maps=maps, max_value=sc.maxval, external_store=True,
                  slide_hop=slide_hop)
    ctx.attach_frames_device(ring)
    ctx.commit_frames(N)
    ctx.demod(qld.QLD_SLIDE, hop)                            # window 0 seeds the accumulators (and the partial sums)
    ctx.sync()
    seed_kernel = ctx.last_kernel()

    def step():                                              # past frame T the ring wraps: same bytes, same traffic
        ctx.commit_frames(hop)
        ctx.demod(qld.QLD_SLIDE, hop)

    ms, clocks, launches = env.timed(step, steps, warmup, keep_busy=step, counter=ctx.kernel_launches)
    kernel = ctx.last_kernel()
    mode = ctx.accum_name()
    is_int = mode in ("INT_BINS", "INT_REFS")
    n_rows = ctx.get_bins(0).shape[0] if is_int else 2 * K
    acc_bytes = 4 if is_int else 8                # int32 bins; fp64 (FP32 mode) or int64 (FIXED) stored sums
    samples = float(hop) * H * W                              # new pixel-samples consumed per step
    res = {"workload": workload, "value": env.world * samples * steps / (ms * 1e-3), "ms_per_step": ms / steps,
           "maps_per_s": env.world * K * steps / (ms * 1e-3), "clocks": clocks, "kernel": kernel, "gpu_launches": int(launches),
           "window_samples_per_s": env.world * float(N) * H * W * steps / (ms * 1e-3)}
    # Two byte counts per launch (both in the line, both recomputable from it):
    #  survey_A5: SURVEY.md 8(a)/(d) row A5, the frame re-reading update with two accumulators per pixel:
    #             2*hop*b (new + expired frames) + 2 x (4 B read + 4 B written) + 4 B map = 148 B per pixel on cfg3;
    #  moved:     what this run's update really moves.  Block-partial form (8(f3)): hop*b of NEW frames only + n_rows
    #             accumulators and n_rows expired partials read, both written back + the map.  Re-reading form: 2*hop*b +
    #             n_rows accumulators read and written + the map.
    # `achieved` / `frac` use `moved` (never bytes the kernel does not touch); `frac_survey_A5` is the equivalent figure.
    survey = H * W * (2.0 * hop * b + 16.0 + 4.0 * K)
    moved = H * W * ((1.0 if slide_hop else 2.0) * hop * b + (4.0 if slide_hop else 2.0) * n_rows * acc_bytes + 4.0 * K)
    res["roofline"] = roofline_hbm(moved, ms / steps, workload, kernel,
                                   (f"moved = per pixel {hop * b} B of new frames + {n_rows} x {acc_bytes} B accumulators and as many expired partial sums read, "
                                    f"both written back + 4 B map (block-partial update, 8(f3)); " if slide_hop else
                                    f"moved = per pixel 2 x {hop * b} B of frames (new + expired) + {n_rows} x {acc_bytes} B accumulators read and written + 4 B map; ")
                                   + f"survey_A5 = 2*hop*b + 16 + 4 = {survey / (H * W):.0f} B per pixel (SURVEY.md 8(d)); a recompute would read {N * b} B per pixel")
    peak = res["roofline"]["peak"]
    res["roofline"]["bytes_moved_per_launch"] = moved
    res["roofline"]["frac_moved"] = res["roofline"]["frac"]
    res["roofline"]["survey_A5_bytes_per_launch"] = survey
    res["roofline"]["frac_survey_A5"] = survey / (ms / steps * 1e-3) / 1e9 / peak
    res["dtype"] = {"INT_BINS": "int32", "INT_REFS": "int32", "FP32": "f32", "FIXED": "int64 (Q1.30 references)"}[mode]
    res["config"] = {"workload": workload, "H": H, "W": W, "N": N, "hop": hop, "K": K, "input_dtype": sc.dtype, "accum": mode,
                     "maps": "amplitude", "step": "qld_commit_frames(hop) + qld_demod(QLD_SLIDE, hop) over the resident ring",
                     "update": "block partial sums (cfg.slide_hop = hop): only the new frames are read" if slide_hop else "expired frames re-read",
                     "ring_frames": T, "seed_kernel": seed_kernel,
                     "cache": f"{2 * hop * H * W * b / 1e6:.0f} MB of frames per step, each read once > 126 MB L2: no flush needed"
                              if 2 * hop * H * W * b > 126e6 else f"{2 * hop * H * W * b / 1e6:.0f} MB of frames per step; new frames were "
                              "written N/hop steps (> L2) earlier, so both reads miss L2",
                     "parallelism": f"{env.world} x independent streams (pixels are independent; no collective)"}

    # ---- CPU baseline + parity: windows recomputed directly by the oracle on a band of rows ---------
    if with_cpu and env.rank == 0:
        import oracle
        from oracle.check import check_float_maps
        nt = oracle.max_threads()
        n_win = 6
        rows = max(1, min(H, args.ref_rows or -(-int(15 * 1.4e8 * nt) // (n_win * K * N * W))))
        r0 = H // 2 - rows // 2                               # the moving disk crosses these rows
        pctx = qld.QLD(H, W, sc.dtype, N, refs, ring_frames=T, accum=accum, maps=qld.QLD_MAP_ALL, max_value=sc.maxval, external_store=True,
                       slide_hop=slide_hop)
        pctx.attach_frames_device(ring)
        pctx.commit_frames(N)
        pctx.demod(qld.QLD_SLIDE, hop)
        last_w = min((T - N) // hop, warmup + steps)
        check_at = sorted(set(w for w in (0, 1, 15, 16, 17, last_w) if w <= last_w))
        secs, worst, done = 0.0, 0.0, 0
        for w in range(0, last_w + 1):
            if w > 0:
                pctx.commit_frames(hop)
                pctx.demod(qld.QLD_SLIDE, hop)
            if w in check_at:
                pctx.sync()
                sub = ring[w * hop:w * hop + N, r0:r0 + rows, :].contiguous().cpu().numpy()
                t0 = time.perf_counter()
                out = [oracle.qld(sub, r, s_first=w * hop + 1, nthreads=nt) for r in refs]
                secs += time.perf_counter() - t0
                done += 1
                for k in range(K):
                    got = tuple(None if m is None else m[r0:r0 + rows].cpu().numpy() for m in pctx.get_maps(k))
                    worst = max(worst, check_float_maps(got, out[k], rel=1e-6 if is_int else 1e-5, what=f"bench parity cfg3 window {w}"))
        res["cpu_baseline"] = {"value": done * float(hop) * rows * W / secs, "unit": UNIT, "cores": nt, "kind": "oracle",
                               "sample": f"{done} windows (w = {check_at}) recomputed directly from the definition on rows {r0}..{r0 + rows - 1}: "
                                         f"{done} x {N} x {rows} x {W} sample-products, {secs:.2f} s; value counts hop x rows x W new samples per window",
                               "window_samples_per_s": done * float(N) * rows * W / secs}
        res["parity"] = {"rows_checked": rows, "windows_checked": check_at, "tolerance": "1e-6" if is_int else "1e-5 floored",
                         "strict_max_rel_err_amp": worst, "ok": True}
        pctx.destroy()
    ctx.destroy()
    del ring
    torch.cuda.empty_cache()

    # ---- end to end, the stream as BASELINE.json configs[3] states it: every batch of the 16384-frame stream pushed from
    # pinned host memory (qld_push_frames, copy stream) into a WRAPPING library-owned ring, one slide + one amplitude map
    # read back per hop.  The timed region covers the whole stream, seeding window included.
    if e2e_steps > 0:
        import numpy as np
        batch = wl.batch
        assert batch == hop, "the e2e leg slides once per pushed batch"
        n_batches = sc.n_frames // batch
        full_stream = True
        try:
            host = torch.empty((n_batches, batch, H, W), dtype=tdt, pin_memory=True)
        except Exception:
            full_stream = False                               # not enough pinnable memory: rotate over a few batches
            host = torch.empty((4, batch, H, W), dtype=tdt, pin_memory=True)
        n_rot = host.shape[0]
        for i in range(n_rot):
            host[i].copy_(qld.synth_fill(sc, 1 + i * batch, batch, device=env.dev))
        torch.cuda.synchronize()
        ring_frames = N + hop + 2 * batch
        n_win = (sc.n_frames - N) // hop + 1
        check_at = [w for w in (0, 1, 15, 16, 17, 255, 495, 496) if w < n_win] if (full_stream and with_cpu and env.rank == 0) else []
        kept = {w: torch.empty((K, H, W), dtype=torch.float32, pin_memory=True) for w in check_at}
        amp_host = torch.empty((2, K, H, W), dtype=torch.float32, pin_memory=True)
        ectx = qld.QLD(H, W, sc.dtype, N, refs, ring_frames=ring_frames, accum=accum, maps=maps, max_value=sc.maxval, slide_hop=slide_hop)

        def run_stream():
            ectx.reset()
            w = 0
            for i in range(n_batches):
                ectx.push_frames(host[i % n_rot])
                if (i + 1) * batch >= N:
                    ectx.demod(qld.QLD_SLIDE, hop)
                    dst = kept[w] if w in kept else amp_host[w & 1]
                    for k in range(K):
                        ectx.read_map(k, qld.QLD_MAP_AMP, dst[k])
                    if w & 1:
                        ectx.sync()                           # a consumer looks at the maps every other hop
                    w += 1
            ectx.sync()
            return w

        env.barrier()
        t0 = time.perf_counter()
        n_maps_out = run_stream()
        env.barrier()
        dt = env.max_over_ranks(time.perf_counter() - t0)
        total = float(sc.n_frames) * H * W
        res["e2e"] = {"value": env.world * total / dt, "unit": UNIT, "h2d_bytes_per_step": int(batch * H * W * b),
                      "d2h_bytes_per_step": int(K * H * W * 4), "ms_per_step": 1e3 * dt / n_batches, "h2d_GBps": total * b / dt / 1e9,
                      "maps_per_s": env.world * K * n_maps_out / dt, "input_frames_per_s": env.world * sc.n_frames / dt, "steps": n_batches,
                      "maps": n_maps_out, "ring_frames": ring_frames, "stream_frames": sc.n_frames, "seconds": dt,
                      "host_stream": "the whole stream in pinned memory" if full_stream else f"{n_rot} pinned batches, rotated (same bytes per step)",
                      "note": "whole stream: pinned host batch -> qld_push_frames (copy stream, wrapping ring) -> qld_demod(QLD_SLIDE) -> "
                              "qld_read_map(amp) -> host; copies overlap the update; timed region includes the seeding window"}
        if check_at:
            import oracle
            from oracle.check import check_float_maps
            nt = oracle.max_threads()
            rows = 8
            r0 = H // 2 - rows // 2
            worst = 0.0
            hs = host.view(n_batches * batch, H, W)
            for w in check_at:
                sub = hs[w * hop:w * hop + N, r0:r0 + rows, :].numpy()
                out = oracle.qld(sub, refs[0], s_first=w * hop + 1, nthreads=nt)
                got = (None, None, kept[w][0, r0:r0 + rows].numpy(), None)
                worst = max(worst, check_float_maps(got, out, rel=1e-6 if is_int else 1e-5, what=f"e2e stream window {w}"))
            res["e2e"]["parity"] = {"windows_checked": check_at, "rows_checked": rows, "strict_max_rel_err_amp": worst, "ok": True,
                                    "note": "amplitude maps of the streamed run (ring wrapped " + str((sc.n_frames - 1) // ring_frames) + " times) vs the oracle's direct recomputation"}
        ectx.destroy()
        del host
    return res


def bench_spectrum(env: Env, args, workload: str, accum_name: str, steps: int, warmup: int, e2e_steps: int, with_cpu: bool):
    """unknown-frequency search (qld_dominant_bin) over every DFT bin 1..N/2-1 of the cfg2-shaped stack
    (1280x1024, N = 1024, uint16): 32 bins per pass on the tensor cores, arg-max fused into the epilogue."""
    torch = env.torch
    from paper_1511_03390_b200 import qld
    wl = build_workload("cfg2", env.rank)
    sc = wl.scene
    N, H, W = wl.N, sc.H, sc.W
    frames = qld.synth_fill(sc, 1, N, device=env.dev)
    q_lo, q_hi = 1, N // 2 - 1
    n_pass = -(-(q_hi - q_lo + 1) // 32)
    out = {}

    def step():
        out["amp"], out["bin"] = qld.dominant_bin(frames, q_lo, q_hi)

    steps = max(3, min(steps, 10))
    ms, clocks, _ = env.timed(step, steps, 5, keep_busy=None, counter=None)
    samples = float(N) * H * W
    stack = samples * 2
    res = {"workload": workload, "value": env.world * samples * steps / (ms * 1e-3), "ms_per_step": ms / steps, "maps_per_s": env.world * steps / (ms * 1e-3),
           "clocks": clocks, "kernel": "k_demod_tc", "gpu_launches": (n_pass + 1) * steps, "dtype": "int8 x int8 -> int32 -> int64 (tcgen05)"}
    res["roofline"] = roofline_hbm(n_pass * stack + 8.0 * H * W, ms / steps, workload, "k_demod_tc",
                                   f"{n_pass} passes over the {stack / 1e9:.2f} GB stack (32 of the {q_hi - q_lo + 1} bins per pass, 256 MMA columns); a single pass "
                                   f"would move {stack / 1e9:.2f} GB and be bound by the int8 tensor rate instead (about 5 ms for this shape)")
    res["roofline"]["traffic"] = None
    res["config"] = {"workload": "f2: qld_dominant_bin on the cfg2 stack", "H": H, "W": W, "N": N, "bins": [q_lo, q_hi], "passes": n_pass,
                     "step": "qld_dominant_bin(bins 1..N/2-1): digit tiles + one tcgen05 launch per 32 bins, blocking call",
                     "cache": f"input {stack / 1e6:.0f} MB per pass > 126 MB L2: no flush needed",
                     "parallelism": f"{env.world} x independent stacks"}
    if with_cpu and env.rank == 0:
        import numpy as np
        import oracle
        nt = oracle.max_threads()
        rng = np.random.default_rng(0)
        pix = np.unique(rng.integers(0, H * W, size=384))
        sub = frames.view(torch.int16).reshape(N, -1)[:, torch.from_numpy(pix).to(env.dev)].cpu().numpy().view(np.uint16).reshape(N, 1, -1)
        t0 = time.perf_counter()
        best, idx, second = oracle.dominant_bin(sub, q_lo, q_hi, nthreads=nt)
        secs = time.perf_counter() - t0
        amp = out["amp"].reshape(-1)[torch.from_numpy(pix).to(env.dev)].cpu().numpy().astype(np.float64)
        bins = out["bin"].reshape(-1)[torch.from_numpy(pix).to(env.dev)].cpu().numpy()
        best, idx, second = best.reshape(-1), idx.reshape(-1), second.reshape(-1)
        assert np.all(np.abs(amp - best) <= 1e-6 * best + 2.0 ** -23 * best), "f2 parity: amplitude"
        unique = second < best * (1.0 - 1e-6)
        assert np.array_equal(bins[unique], idx[unique]), "f2 parity: bin"
        res["cpu_baseline"] = {"value": float(sub.size) / secs, "unit": UNIT, "cores": nt, "kind": "oracle",
                               "sample": f"{len(pix)} random pixels x {N} frames x {q_hi - q_lo + 1} bins (one QLD per bin), {secs:.2f} s"}
        res["parity"] = {"pixels_checked": int(len(pix)), "tolerance": "amplitude 1e-6; bin equal wherever the runner-up is not within 1e-6",
                         "unique_fraction": float(unique.mean()), "ok": True}
    del frames
    torch.cuda.empty_cache()
    return res


RUNNERS = {"f2": bench_spectrum, "cfg0": bench_whole, "cfg1": bench_whole, "cfg2": bench_whole, "cfg3": bench_slide, "cfg4": bench_whole}


def spawn_ranks(n: int):
    """`python bench.py --gpus N` outside a torchrun environment: re-execute under torch.distributed.run, one rank per GPU."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def compact(r: dict) -> dict:
    """The short form of a config's result: enough to recompute every fraction from the record alone."""
    rf = r["roofline"]
    out = {"value": r["value"], "ms_per_step": r["ms_per_step"], "kernel": r["kernel"], "frac": rf["frac"], "achieved_GBps": rf["achieved"],
           "peak_GBps": rf["peak"], "bytes_per_launch": rf["algorithmic_bytes_per_launch"]}
    for k in ("frac_survey_A5", "survey_A5_bytes_per_launch", "frac_of_read_ceiling", "read_ceiling_GBps"):
        if k in rf:
            out[k] = rf[k]
    if r.get("parity"):
        out["parity_ok"] = r["parity"]["ok"]
    if r.get("e2e"):
        out["e2e_value"] = r["e2e"]["value"]
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=sorted(RUNNERS))
    ap.add_argument("--accum", default="auto", choices=sorted(ACCUM_NAMES))
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--shard", default="stacks", choices=["stacks", "rows"], help="N > 1: 'stacks' = one independent stack / stream per rank "
                    "(weak scaling); 'rows' = the ranks split ONE frame into contiguous row bands (SURVEY.md 8(e); strong scaling; "
                    "whole-window workloads)")
    ap.add_argument("--ref-rows", type=int, default=0, help="rows of the frame the CPU oracle is timed / checked on "
                    "(0: sized for about 15 s of oracle work on the host cores; 32 for --impl reference)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--reread-expired", action="store_true", help="cfg3: update the window by re-reading the expired frames "
                    "(SURVEY.md 8(a) A5 as literally stated) instead of keeping per-batch partial sums (8(f3), cfg.slide_hop: "
                    "identical results, fewer bytes, and the faster of the two on B200: the default)")
    ap.add_argument("--also", default="default", help="comma list of other workloads to run briefly first, one compact JSON line each "
                    "(default: cfg2,cfg3,cfg1,cfg0,f2 when --workload is cfg4 on one GPU; 'none' to skip)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    if args.impl == "reference":
        run_reference(args, int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")))
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args.gpus)                                  # does not return

    env = Env(args)
    if not env.oversubscribed:
        measure_read_ceiling(env)
    names = args.also
    if names == "default":
        names = "cfg2,cfg3,cfg1,cfg0,f2" if (args.workload == "cfg4" and env.world == 1 and args.accum == "auto") else "none"
    also = {}
    if names != "none":
        for w in [x for x in names.split(",") if x and x != args.workload]:
            r = RUNNERS[w](env, args, w, "auto", min(args.steps, 200) if w != "cfg2" else max(args.steps, 100), 5,
                           args.e2e_steps if w == "cfg3" else 0, not args.no_cpu_baseline)
            also[w] = compact(r)
            if env.rank == 0:
                line = {"also": w, "metric": METRIC, "unit": UNIT}
                line.update({k: r[k] for k in ("value", "ms_per_step", "maps_per_s", "window_samples_per_s", "kernel", "gpu_launches", "dtype",
                                               "config", "roofline", "parity", "cpu_baseline", "e2e", "clocks") if k in r})
                print(json.dumps(line), flush=True)

    main_res = RUNNERS[args.workload](env, args, args.workload, args.accum, args.steps, args.warmup, args.e2e_steps,
                                      not args.no_cpu_baseline)
    if env.rank == 0:
        r = main_res
        line = {}
        if also:
            line["also"] = also                                  # summaries first: the headline keys close the line
        line.update({"maps_per_s": r["maps_per_s"], "parity": r.get("parity"), "clocks": r["clocks"], "cpu_baseline": r.get("cpu_baseline"),
                     "e2e": r.get("e2e"), "roofline": r["roofline"], "gpu_launches": r["gpu_launches"], "config": r["config"],
                     "data": "synthetic", "dtype": r["dtype"], "vs_baseline": None, "scaling": r.get("scaling", "weak"),
                     "higher_is_better": True, "ms_per_step": r["ms_per_step"], "warmup": args.warmup, "steps": args.steps,
                     "n_gpus": env.world, "unit": UNIT, "value": r["value"], "metric": METRIC})
        if env.oversubscribed:
            line["oversubscribed"] = f"{env.world} ranks on {env.torch.cuda.device_count()} GPU(s): a plumbing check, not a scaling measurement"
        if "window_samples_per_s" in r:
            line["window_samples_per_s"] = r["window_samples_per_s"]
        print(json.dumps(line), flush=True)
    if env.dist is not None:
        env.dist.destroy_process_group()


if __name__ == "__main__":
    main()
