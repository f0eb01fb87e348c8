#!/usr/bin/env python
"""bench.py -- QLD pixel-samples/s on one node, through the C-ABI library (libqld.so).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A step is one pass of the hot path over one window of synthetic frames of the named BASELINE.json config:
qld_demod (reference tables were built by qld_create, A1) = A3/A3'/A6 demodulation + A4 finalise, with the
frames resident in HBM (`value`), and the same through host buffers -- qld_push_frames from pinned memory (A2),
qld_demod, qld_read_map of the amplitude map back to the host -- for `e2e`.  Prints ONE JSON line (rank 0).
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
sys.path.insert(0, os.path.join(ROOT, "tests"))

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


def build_workload(name: str, rank: int):
    from paper_1511_03390_b200 import synth
    return synth.BUILDERS[name](seed=int(name[3]) + 1000 * rank)      # BASELINE.json seeds: cfgN -> seed N


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
    samples = float(x.size) * args.steps
    val = samples / t
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f80 (x87 long double) / int64", "data": "synthetic",
            "config": {"workload": args.workload, "H": sc.H, "W": sc.W, "N": wl.N, "K": len(refs),
                       "sample": f"first {rows} rows x {sc.W} cols x {wl.N} frames per step"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": nt, "kind": "oracle",
                             "sample": f"{rows} rows x {sc.W} x {wl.N} frames ({x.size} samples) per step"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg0", "cfg1", "cfg2", "cfg4"])
    ap.add_argument("--accum", default="auto", choices=["auto", "fp32", "bins", "fixed"])
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--ref-rows", type=int, default=0, help="rows of the frame the CPU oracle is timed / checked on "
                    "(0: sized for about 15 CPU-seconds of oracle work; 32 for --impl reference)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1511_03390_b200 import qld, synth
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    wl = build_workload(args.workload, rank)
    sc = wl.scene
    N, H, W, K = wl.N, sc.H, sc.W, len(wl.refs)
    bytes_per = 1 if sc.dtype == "u8" else 2
    accum = {"auto": qld.QLD_ACC_AUTO, "fp32": qld.QLD_ACC_FP32, "bins": qld.QLD_ACC_INT_BINS, "fixed": qld.QLD_ACC_FIXED}[args.accum]

    # ---- inputs: synthetic stack filled on the device, resident before the timed region -------------
    frames = qld.synth_fill(sc, 1, N, device=dev)
    torch.cuda.synchronize()
    ctx = qld.QLD(H, W, sc.dtype, N, [dict(r) for r in wl.refs], ring_frames=-1, accum=accum, maps=qld.QLD_MAP_ALL,
                  max_value=sc.maxval)
    ctx.attach_frames_device(frames)
    is_int = False
    try:
        ctx.get_bins(0)
        is_int = True
    except qld.QLDError:
        pass

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        ctx.demod(qld.QLD_WHOLE)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    l0 = ctx.kernel_launches()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        ctx.demod(qld.QLD_WHOLE)
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = ctx.kernel_launches() - l0
    # keep the GPU busy a little longer if the region was too short for a clock sample
    t_end = time.time() + 0.25
    while len(sampler.samples) < 8 and time.time() < t_end:
        ctx.demod(qld.QLD_WHOLE)
        torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join()
    if world > 1:
        t = torch.tensor([ms], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    samples_per_step = float(N) * H * W
    value = world * samples_per_step * args.steps / (ms * 1e-3)

    # ---- roofline of the dominant kernel (the demodulation kernel is the only launch of a step) -----
    n_maps = 4
    algo_bytes = samples_per_step * bytes_per + n_maps * K * H * W * 4.0
    peak, peak_src = load_peaks()
    achieved = algo_bytes / (ms * 1e-3 / args.steps) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic_r01.json")
    if os.path.exists(tpath):
        try:
            traffic = json.load(open(tpath)).get(args.workload)
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "peak_source": peak_src, "algorithmic_bytes_per_launch": algo_bytes,
                "frac_of_nominal_8TBps": achieved / 8000.0, "kernel": "k_demod_tc" if args.accum == "fixed" else "k_demod_whole"}

    # ---- end to end through host buffers (pinned): push + demod + read amplitude map back ------------
    e2e = None
    parity = None
    if (rank == 0 or world > 1) and args.e2e_steps > 0:
        host = torch.empty((N, H, W), dtype=frames.dtype).pin_memory()
        host.copy_(frames)
        amp_host = torch.empty((K, H, W), dtype=torch.float32).pin_memory()
        torch.cuda.synchronize()
        ectx = qld.QLD(H, W, sc.dtype, N, [dict(r) for r in wl.refs], ring_frames=0, accum=accum, maps=qld.QLD_MAP_ALL,
                       max_value=sc.maxval)
        chunk = max(1, min(N, (256 << 20) // (H * W * bytes_per)))       # pushes of about 256 MiB

        def e2e_step():
            ectx.reset()
            for a in range(0, N, chunk):
                ectx.push_frames(host[a:a + chunk])
            ectx.demod(qld.QLD_WHOLE)
            for k in range(K):
                ectx.read_map(k, qld.QLD_MAP_AMP, amp_host[k])
            ectx.sync()

        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            e2e_step()
        barrier()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": world * samples_per_step * args.e2e_steps / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(samples_per_step * bytes_per), "d2h_bytes_per_step": int(K * H * W * 4),
               "ms_per_step": 1e3 * dt / args.e2e_steps, "h2d_GBps": samples_per_step * bytes_per * args.e2e_steps / dt / 1e9,
               "steps": args.e2e_steps, "note": "pinned host stack -> qld_push_frames -> qld_demod -> qld_read_map(amp) -> host"}
        ectx.destroy()
        del host

    # ---- CPU baseline (the oracle, as it stands) + parity of the timed configuration on the same rows -
    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        import oracle
        from _parity import check_float_maps
        # about 15 CPU-seconds of oracle work at ~9e7 sample-references per second per core
        rows = max(1, min(H, args.ref_rows or -(-int(1.35e9) // (K * N * W))))
        r0 = (H // 2 - rows // 2)
        sub = frames[:, r0:r0 + rows, :].contiguous().cpu().numpy()
        nt = oracle.max_threads()
        refs = [dict(r) for r in wl.refs]
        oracle_on_rows(wl, sub[:8], refs[:1], nt)                      # thread pool warm-up
        out, secs = oracle_on_rows(wl, sub, refs, nt)
        cpu = {"value": float(sub.size) / secs, "unit": UNIT, "cores": nt, "kind": "oracle",
               "sample": f"rows {r0}..{r0 + rows - 1} x {W} cols x {N} frames x {K} refs = {sub.size} samples, {secs:.2f} s"}
        ctx.demod(qld.QLD_WHOLE)
        ctx.sync()
        worst = 0.0
        for k in range(K):
            got = tuple(m[r0:r0 + rows].cpu().numpy() for m in ctx.get_maps(k))
            worst = max(worst, check_float_maps(got, out[k], rel=(1e-6 if is_int else 1e-5), what=f"bench parity k={k}"))
        parity = {"rows_checked": rows, "refs_checked": K, "tolerance": "1e-6 (bins, fp64 combine)" if is_int else "1e-5 floored at map median",
                  "strict_max_rel_err_amp": worst, "ok": True}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "int32 (phase bins)" if is_int else ("int8 x int8 -> int32/int64 (tcgen05, Q1.30 references)" if args.accum == "fixed" else "f32"), "data": "synthetic",
                "config": {"workload": args.workload, "H": H, "W": W, "N": N, "K": K, "input_dtype": sc.dtype,
                           "accum": "INT_BINS" if is_int else ("FIXED (tensor cores)" if args.accum == "fixed" else "FP32 (pedestal)"), "maps": "I,Q,amplitude,phase",
                           "cache": f"input {samples_per_step * bytes_per / 1e6:.0f} MB per step "
                                    + ("> 126 MB L2: no flush needed" if samples_per_step * bytes_per > 3e8 else "<= L2: L2-resident, not an HBM number"),
                           "parallelism": f"{world} x independent stacks (pixels are independent; no collective)"},
                "maps_per_s": value / samples_per_step, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
                "gpu_launches": int(launches), "clocks": sampler.result(), "parity": parity}
        print(json.dumps(line), flush=True)
    ctx.destroy()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
