#!/usr/bin/env python
"""bench.py -- emulated-fp64 3-D FFT (arxiv/paper_2606_23698 hot path) on B200, one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--size 1024] [--impl ours|reference]

A step is one forward complex128 3-D transform of size^3 (BASELINE.json configs[4] workload; size 1024 by
default) through the C ABI (ozfft_exec): every stage of the hot path runs in the CUDA kernels.
value = 5*N_tot*log2(N_tot) GFLOP/s (PAPER.md:859 flop convention) with the input resident in HBM;
e2e = the same through ozfft_exec_host with pinned HOST buffers (H2D + D2H inside the timed region).
N > 1 runs N independent replicas (one per rank, no collective: north_star fixes the path to one GPU;
DESIGN.md "replicas only"), value = aggregate over ranks / max time.
--impl reference times the CPU oracle (oracle/, plain C, OpenMP) on a bounded sample of the same workload.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

SEED = 4  # BASELINE.json configs[4]


def flops(n_tot):
    return 5.0 * n_tot * math.log2(n_tot)


def peaks():
    try:
        p = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], 0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(sm)}


def max_over_ranks(values, device="cpu"):
    """element-wise MAX over the ranks of the default process group (identity when not initialised):
    every multi-GPU number is the slowest rank's (timed on the device)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def kernel_source_hash():
    from paper_2606_23698_b200 import ledger
    return ledger.kernel_source_hash()


def ncu_constants(size, variant):
    """ncu-derived figures of the dominant kernel (DRAM traffic per launch, thread instructions per output-equivalent)
    from profiles/ncu_constants.json, which records the ncu command and the source hash they were measured on.
    Returns (entry or None, note): None when no entry matches this size / variant / source hash (never a stale number)."""
    try:
        db = json.load(open(os.path.join(ROOT, "profiles", "ncu_constants.json")))
    except Exception:
        return None, "profiles/ncu_constants.json missing"
    if db.get("source_hash") != kernel_source_hash():
        return None, f"stale: profiles/ncu_constants.json was captured on source hash {db.get('source_hash')}, the tree is {kernel_source_hash()}"
    e = db.get("entries", {}).get(f"{variant}:{size}")
    return (e, e.get("command", "")) if e else (None, f"no ncu capture for variant {variant} at size {size}")



def cpu_oracle_sample(size, pencils):
    """Times the oracle (as it stands, direct exact-integer route) on `pencils` length-`size` pencils of the
    workload's own data; returns (seconds, threads)."""
    from oracle import oracle
    from paper_2606_23698_b200 import inputs
    import numpy as np
    x = (2.0 * inputs.uniform01(SEED, 0, 2 * pencils * size) - 1.0).view(np.complex128).reshape(pencils, size)
    oracle.fft1d(x[:64], -1, route=0)  # page in
    t = time.perf_counter()
    oracle.fft1d(x, -1, route=0)
    return time.perf_counter() - t, oracle.num_threads()


def workload_name(size):
    """the same string in both arms (the driver compares them)"""
    return f"forward 3-D FFT {size}^3 complex128, uniform[-1,1), seed {SEED}" + (" (BASELINE.json configs[4])" if size == 1024 else "")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    size = args.size
    n_tot = size ** 3
    pencils = 262144
    total_pencils = 3 * size * size
    times = []
    threads = 1
    for i in range(args.warmup + args.steps):
        dt, threads = cpu_oracle_sample(size, pencils)
        if i >= args.warmup:
            times.append(dt)
    t_step = sum(times) / len(times)
    t_full = t_step * total_pencils / pencils  # extrapolated time of one whole transform
    val = flops(n_tot) / t_full / 1e9
    sample = f"{pencils} of {total_pencils} length-{size} pencils per step ({pencils / total_pencils:.4%} of one transform), extrapolated"
    workload = workload_name(size)
    line = {"impl": "reference", "metric": "emulated_fp64_fft3d_gflops_5NlogN", "value": val, "unit": "GFLOP/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_full * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int128", "data": "synthetic",
            "config": {"workload": workload},
            "cpu_baseline": {"value": val, "unit": "GFLOP/s", "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2606_23698_b200 import inputs, ozfft

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch with torchrun --nproc-per-node {args.gpus} "
                         f"(or run `python bench.py --gpus {args.gpus}` without WORLD_SIZE set: it spawns the ranks itself)")
    if args.dry_run:  # CPU rehearsal of the launch plumbing only (tests/test_multirank_cpu.py): no transform is run
        if world > 1:
            dist.init_process_group("gloo")
        worst = max_over_ranks([float(rank)])
        if rank == 0:
            print(json.dumps({"dry_run": True, "n_gpus": world, "max_rank_seen": worst[0]}))
        if world > 1:
            dist.destroy_process_group()
        return
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    size = args.size
    n_tot = size ** 3
    shape = (size, size, size)
    nbytes = 16 * n_tot

    # synthetic input (configs[4] recipe), generated on the host in pinned memory, rank-specific seed offset.
    # N ranks on one node need N x 2 x 16 GiB of pinned host memory for the end-to-end leg: if the node does not
    # have it, the input is streamed to the device in slabs and the e2e leg is reported as skipped (never risk the box)
    try:
        import psutil
        host_ok = psutil.virtual_memory().available > world * 2 * nbytes * 1.2
    except Exception:
        host_ok = world == 1
    if world > 1:  # one decision for all ranks (the end-to-end leg has barriers)
        flag = torch.tensor([1 if host_ok else 0], device="cuda")
        dist.all_reduce(flag, op=dist.ReduceOp.MIN)
        host_ok = bool(flag.item())
    seed = SEED + 1000 * rank
    if host_ok:
        h_in = torch.empty(shape, dtype=torch.complex128).pin_memory()
        inputs.uniform_pm1(shape, seed, out=h_in.numpy())
        h_out = torch.empty(shape, dtype=torch.complex128).pin_memory()
        d_in = h_in.cuda()
    else:
        h_in = h_out = None
        d_in = torch.empty(shape, dtype=torch.complex128, device="cuda")
        flat = d_in.view(torch.float64).view(-1)
        step = 1 << 26
        for s0 in range(0, 2 * n_tot, step):
            c = min(step, 2 * n_tot - s0)
            flat[s0:s0 + c].copy_(torch.from_numpy(2.0 * inputs.uniform01(seed, s0, c) - 1.0))
    d_out = torch.empty_like(d_in)
    plan = ozfft.Plan(size, size, size, sign=-1)
    launches = plan.num_launches
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        plan.exec(d_in, d_out)
    barrier()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    with ClockSampler(local) as cs:
        ev[0].record(stream)
        for i in range(args.steps):
            plan.exec(d_in, d_out)
            ev[i + 1].record(stream)
        barrier()
    ms = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    ms_step = sum(ms) / len(ms)
    clocks = cs.summary()

    # end to end through the public API with HOST buffers
    e2e_steps = max(1, min(args.steps, 3))
    e2e_ms, same = float("nan"), None
    if host_ok:
        plan.exec_host(h_in, h_out)  # warm-up (allocates the staging buffers)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            plan.exec_host(h_in, h_out)
        barrier()
        e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
        # sanity inside the bench: device-resident and host paths agree bit for bit
        same = bool(torch.equal(d_out.cpu().view(torch.float64), h_out.view(torch.float64)))

    # round trip (BASELINE.json configs[4]: forward then inverse)
    x_keep = d_in.view(-1)[: min(n_tot, 1 << 27)].clone()
    inv = ozfft.Plan(size, size, size, sign=+1)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    inv.exec(d_out, d_in)  # overwrites d_in with the unnormalised round trip
    e1.record(stream)
    torch.cuda.synchronize()
    inv_ms = e0.elapsed_time(e1)
    chunk = 1 << 24
    flat_rt = d_in.view(-1)
    num = den = 0.0
    for s in range(0, x_keep.numel(), chunk):
        a = flat_rt[s:s + chunk] / n_tot
        b = x_keep[s:s + chunk]
        num += float(((a - b).abs() ** 2).sum())
        den += float((b.abs() ** 2).sum())
    roundtrip = math.sqrt(num / den)
    inv.destroy()
    del x_keep

    # cuFFT Z2Z context number (not part of the path)
    cufft_ms = None
    try:
        for _ in range(2):
            y = torch.fft.fftn(d_in)
            del y
        torch.cuda.synchronize()
        e0.record(stream)
        y = torch.fft.fftn(d_in)
        e1.record(stream)
        torch.cuda.synchronize()
        cufft_ms = e0.elapsed_time(e1)
        del y
    except Exception as ex:  # out of memory at the largest size is not fatal for the bench line
        cufft_ms = None

    ms_step_max, e2e_ms_max = max_over_ranks([ms_step, e2e_ms if host_ok else 0.0], device="cuda")

    if rank == 0:
        peak, peak_src = peaks()
        variant = os.environ.get("OZFFT_VARIANT", "bf")
        schedule = os.environ.get("OZFFT_SCHEDULE", "fused") if variant == "bf" else "unfused"
        stage_gemms = 3 * (2 if size > 32 else 1)  # per transform (Eq. 12: n_out = stage GEMMs x 2 N_tot)
        n_out = 2 * stage_gemms * n_tot
        # algorithmic bytes = 32 B per element per AXIS PASS (16 read + 16 written) =
        # 96 N_tot per transform; a transform is `launches` stage launches of one kernel (two per axis when n > 32), so
        # one launch accounts for 96 N_tot / launches algorithmic bytes.  Fused schedule: one launch per axis, measured DRAM
        # traffic 1.00 x 32 N_tot (beta = 1); unfused: two launches per axis, Y' crosses HBM (beta = 2).  beta is reported
        # beside the fraction from the ncu capture recorded in profiles/ncu_constants.json.
        alg_bytes_launch = 96.0 * n_tot / launches
        launch_ms = ms_step / launches
        achieved = alg_bytes_launch / (launch_ms * 1e-3) / 1e9
        ncu, ncu_note = ncu_constants(size, variant if schedule != "unfused" or variant != "bf" else "bf-unfused")
        traffic = ncu["dram_bytes_per_launch"] if ncu else None
        tinst = ncu["thread_inst_per_output_eq"] if ncu else None
        line = {
            "metric": "emulated_fp64_fft3d_gflops_5NlogN", "value": world * flops(n_tot) / (ms_step_max * 1e-3) / 1e9,
            "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step_max,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": workload_name(size),
                       "parallelism": "replicas only" if world > 1 else "single GPU", "l2": "inputs_exceed_l2" if nbytes > (126 << 20) else "l2_resident",
                       "variant": variant, "schedule": schedule, "stage_launches_per_transform": launches, "stage_gemms_per_transform": stage_gemms},
            "ms_per_transform": ms_step_max, "ms_per_transform_min": min(ms), "inverse_ms": inv_ms,
            "roundtrip_rel_err": roundtrip, "host_and_device_paths_bit_identical": same,
            "hbm_roof": {"alg_bytes": 96.0 * n_tot,
                         "roof_ms_at_measured_peak": 96.0 * n_tot / (peak * 1e9) * 1e3, "frac_of_roof": (96.0 * n_tot / (peak * 1e9) * 1e3) / ms_step},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "beta": (traffic / alg_bytes_launch if traffic else None),
                         "kernel": {"bf": "stage_bf_kernel", "tc": "stage_tc_kernel", "simt": "stage_simt_kernel"}.get(variant, variant) + " (every launch of a transform is this kernel"
                                   + ("; fused schedule: one launch per axis, both stages, Y' in an L2-resident ring)" if schedule == "fused" else ")"),
                         "peak_source": peak_src, "alg_bytes_per_launch": alg_bytes_launch, "launch_ms": launch_ms,
                         "ncu": ncu_note},
            "clocks": clocks,
            "e2e": ({"value": world * flops(n_tot) / (e2e_ms_max * 1e-3) / 1e9, "unit": "GFLOP/s", "ms": e2e_ms_max,
                     "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes, "steps": e2e_steps} if host_ok else
                    {"value": None, "unit": "GFLOP/s", "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                     "skipped": "not enough host memory on this node for N x 2 x 16 GiB of pinned buffers"}),
            "gpu_launches": launches * args.steps,
            # the SIMT side (PAPER.md:452 names integer issue as the wall): achieved = n_out x the ncu-measured thread
            # instructions per output-equivalent / step time; peak = 148 SM x 128 lanes x 1.965 GHz.
            # null when no ncu capture matches the current kernel sources.
            "roofline_alu": ({"bound": "alu", "achieved": n_out * tinst / (ms_step * 1e-3) / 1e12,
                              "peak": 148 * 128 * 1.965e9 / 1e12, "unit": "T thread-inst/s",
                              "frac": n_out * tinst / (ms_step * 1e-3) / (148 * 128 * 1.965e9),
                              "n_out": n_out, "thread_inst_per_output_eq": tinst} if tinst else None),
            "context": {"cufft_z2z_ms": cufft_ms, "paper_projection_ms_B300": [63, 87], "paper_projection_ms_B200": [70, 96],
                        "paper_hbm_roof_ms": 12.9},
        }
        if not args.no_cpu:
            pencils = 262144
            dt, threads = cpu_oracle_sample(size, pencils)
            t_full = dt * (3 * size * size) / pencils
            line["cpu_baseline"] = {"value": flops(n_tot) / t_full / 1e9, "unit": "GFLOP/s", "cores": threads, "kind": "oracle",
                                    "sample": f"{pencils} of {3 * size * size} length-{size} pencils ({dt:.1f} s), extrapolated to one transform = {t_full:.0f} s"}
        print(json.dumps(line))
    plan.destroy()
    if world > 1:
        dist.destroy_process_group()


def run_configs(args):
    """--configs: ms per transform for all five BASELINE.json workloads (bench.py's contract line times only the headline
    one): CUDA events on the current stream, median of --steps after --warmup; 5 N log2 N GFLOP/s; fraction of the HBM roof
    (32 B per element per axis pass over the measured copy bandwidth); cuFFT Z2Z fp64 on the same tensor for context.
    One JSON line per config, variant from OZFFT_VARIANT (default: the byte-fed kernel)."""
    import torch
    from paper_2606_23698_b200 import inputs, ozfft
    hbm, _ = peaks()

    def timed(fn):
        for _ in range(max(3, args.warmup)):
            fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(args.steps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        ts.sort()
        return ts[len(ts) // 2], ts[0]

    for name, (kind, shape, dist_name, seed) in inputs.CONFIGS.items():
        h = torch.empty(shape, dtype=torch.complex128)
        if dist_name == "uniform":
            inputs.uniform_pm1(shape, seed, out=h.numpy())
        else:
            h.copy_(torch.from_numpy(inputs.make(dist_name, shape, seed)))
        x = h.cuda()
        y = torch.empty_like(x)
        if kind == "3d":
            plan = ozfft.Plan(*shape)
            flop, passes = 5.0 * x.numel() * math.log2(x.numel()), 3
            cufft = lambda: torch.fft.fftn(x)
        else:
            plan = ozfft.Plan.batched_1d(shape[1], shape[0])
            flop, passes = 5.0 * x.numel() * math.log2(shape[1]), 1
            cufft = lambda: torch.fft.fft(x, dim=1)
        med, best = timed(lambda: plan.exec(x, y))
        try:
            cmed, _ = timed(cufft)
        except Exception:
            cmed = None
        # variants other than the default: the same transform on the default kernel, compared on the device (the exact
        # variants must be bit-identical; fp64sum, the naive fp64 Phase B of PAPER.md:340-345, shows its lost bits here)
        same = diff = None
        variant = os.environ.get("OZFFT_VARIANT", "bf")
        if variant != "bf" or os.environ.get("OZFFT_SCHEDULE"):
            keep = {k: os.environ.pop(k, None) for k in ("OZFFT_VARIANT", "OZFFT_SCHEDULE")}
            ref_plan = ozfft.Plan(*shape) if kind == "3d" else ozfft.Plan.batched_1d(shape[1], shape[0])
            for k, v in keep.items():
                if v is not None:
                    os.environ[k] = v
            yref = ref_plan.exec(x)
            torch.cuda.synchronize()
            same = bool(torch.equal(y.view(torch.float64), yref.view(torch.float64)))
            num = den = 0.0
            fy, fr = y.view(-1), yref.view(-1)
            for s0 in range(0, fy.numel(), 1 << 26):
                num += float(((fy[s0:s0 + (1 << 26)] - fr[s0:s0 + (1 << 26)]).abs() ** 2).sum())
                den += float((fr[s0:s0 + (1 << 26)].abs() ** 2).sum())
            diff = math.sqrt(num / den)
            ref_plan.destroy()
            del yref
        roof_ms = 32.0 * x.numel() * passes / (hbm * 1e9) * 1e3
        print(json.dumps({"config": name, "variant": variant, "schedule": os.environ.get("OZFFT_SCHEDULE", "fused" if variant == "bf" else "unfused"),
                          "bit_identical_to_default_kernel": same, "normwise_diff_vs_default_kernel": diff, "shape": list(shape), "input": dist_name,
                          "seed": seed, "launches": plan.num_launches, "ms_median": med, "ms_best": best,
                          "gflops_5NlogN": flop / (med * 1e-3) / 1e9, "hbm_roof_ms": roof_ms, "frac_of_hbm_roof": roof_ms / med,
                          "cufft_z2z_ms": cmed}), flush=True)
        plan.destroy()
        del x, y, h
        torch.cuda.empty_cache()


def run_pipe_timers(args):
    """--pipe-timers: where the byte-fed kernel's roles wait.  Builds and loads the measuring library (build.py --timers:
    clock64 stamps around every mbarrier wait), runs one transform per axis pass and prints, per launch, the cycles per
    tile each role spent waiting (mean over the CTAs).  Not a timed run: the stamps cost issue slots."""
    import ctypes
    import numpy as np
    import torch
    from paper_2606_23698_b200 import build as b, ozfft
    ozfft._SO = b.build(timers=True)
    L = ozfft.lib()
    size = args.size
    x = torch.randn(size, size, size, dtype=torch.complex128, device="cuda")
    plan = ozfft.Plan(size, size, size)
    buf = (ctypes.c_ulonglong * (160 * 12))()
    y = plan.exec(x)
    torch.cuda.synchronize()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    names = ["z", "y", "x"]
    for axis in range(3):
        # the stamps are those of the LAST launch: the axis hook (unfused, natural order) ends with the axis' second stage
        plan.exec_axis(axis, x, y)
        torch.cuda.synchronize()
        assert L.ozfft_debug_timers(buf) == 160
        a = np.frombuffer(buf, dtype=np.uint64).reshape(160, 12)[:sms].astype(np.float64)
        t = a[:, 4].mean()
        print(json.dumps({"launch": f"{names[axis]} pass, second stage (axis hook, unfused, natural order)", "tiles_per_cta": t,
                          "issuer_wait_a_full": a[:, 0].mean() / t, "issuer_wait_b_full": a[:, 1].mean() / t, "issuer_wait_pa_empty": a[:, 2].mean() / t,
                          "issuer_total": a[:, 3].mean() / t, "epilogue_wait_pa_full": a[:, 5].mean() / t, "epilogue_wait_a_full": a[:, 6].mean() / t,
                          "epilogue_total": a[:, 7].mean() / t, "decon_wait_ring": a[:, 8].mean() / t, "decon_wait_a_empty_e_start": a[:, 9].mean() / t,
                          "decon_total": a[:, 10].mean() / t, "unit": "SM cycles per tile"}))
    plan.exec(x, y)
    torch.cuda.synchronize()
    assert L.ozfft_debug_timers(buf) == 160
    a = np.frombuffer(buf, dtype=np.uint64).reshape(160, 12)[:sms].astype(np.float64)
    t = a[:, 4].mean()
    print(json.dumps({"launch": "x pass of the one-call transform (" + os.environ.get("OZFFT_SCHEDULE", "fused") + " schedule; a fused launch holds both stages)",
                      "tiles_per_cta": t, "issuer_wait_a_full": a[:, 0].mean() / t, "issuer_wait_b_full": a[:, 1].mean() / t,
                      "issuer_wait_pa_empty": a[:, 2].mean() / t, "issuer_total": a[:, 3].mean() / t, "epilogue_wait_pa_full": a[:, 5].mean() / t,
                      "epilogue_wait_a_full": a[:, 6].mean() / t, "epilogue_total": a[:, 7].mean() / t, "decon_wait_ring": a[:, 8].mean() / t,
                      "decon_wait_a_empty_e_start": a[:, 9].mean() / t, "decon_total": a[:, 10].mean() / t, "unit": "SM cycles per tile"}))
    plan.destroy()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--size", type=int, default=1024)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    ap.add_argument("--configs", action="store_true", help="time all five BASELINE.json configs (one JSON line each) instead of the contract line")
    ap.add_argument("--pipe-timers", action="store_true", help="per-role wait cycles of the byte-fed kernel (measuring build; not a timed run)")
    ap.add_argument("--dry-run", action="store_true", help="launch plumbing only (gloo, no GPU work): used by the CPU tests")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N`: spawn the N ranks ourselves (one process per GPU, the driver's own launch line)
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.pipe_timers:
        run_pipe_timers(args)
    elif args.configs:
        run_configs(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
