#!/usr/bin/env python
"""Throughput of the APIC closed-form reconstruction on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl apic|reference] [--config 2]

A step = one pass of the whole hot path (S0-S10 of DESIGN.md) over one batch of synthetic tiles.
Default workload: BASELINE.json config 2 (64 tiles of 256x256, 8 NA-matching + 16 darkfield LEDs,
Poisson noise, 3x output grid) - the batched 256x256 configuration the north-star target is quoted
on (config 1 is a single tile, i.e. a latency case).  Prints ONE JSON line.

  value     output megapixels/s with the inputs resident in HBM (CUDA events, max over ranks)
  e2e       the same metric through apic_reconstruct_host with pinned HOST buffers (H2D + D2H inside)
  roofline  the dominant kernel (df_cols_mul: column IFFT . p . column FFT of the darkfield CG),
            timed live by CUDA events inside the library on the launching stream
  cpu_baseline  the fp64 oracle, as it stands, on this box's host cores, on a bounded sample
`--impl reference` times the oracle alone (rank 0 only under torchrun).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "reconstructed output megapixels/sec"
UNIT = "Mpx/s"
FP32_LANES_PER_SM = 128          # FMA lanes per SM (4 SMSPs x 32), B200


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="apic", choices=["apic", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (2 = default workload)")
    ap.add_argument("--tiles", type=int, default=0, help="tiles per step and per GPU (0 = the config's batch, capped at 64)")
    ap.add_argument("--chunk", type=int, default=0, help="apic_params.chunk_tiles (0 = library default)")
    ap.add_argument("--df-mode", type=int, default=0, help="darkfield scheduler: 0 team kernel (reduced grids at N=256), 1 launch per phase, 2 ticket kernel, 3 team kernel on the full grid")
    ap.add_argument("--df-team", type=int, default=0, help="apic_params.df_team: CTAs per tile of the team kernel (0 = auto)")
    ap.add_argument("--df-tol", type=float, default=-1.0, help="CG tolerance (default: the library's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--breakdown", action="store_true", help="also print the per-kernel time table to stderr")
    return ap.parse_args()


def workload_name(cfg, tiles):
    return (f"{cfg.name}: {tiles} tiles/GPU/step, {cfg.tile_n}x{cfg.tile_n} px, {cfg.n_bright} NA-matching + "
            f"{cfg.n_dark} darkfield LEDs, {len(cfg.noll_fit)} Zernike terms, {cfg.upsample}x output grid, "
            f"{cfg.noise} noise")


def host_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 0) for p in threadpool_info() if p.get("user_api") == "blas"]
        if n:
            return int(max(n))
    except Exception:
        pass
    return int(os.cpu_count() or 1)


# ------------------------------------------------------------------------------------ reference arm
def oracle_step(stack, params, geo, sets):
    from oracle import apic_oracle as O
    t0 = time.perf_counter()
    r = O.reconstruct_tile(stack, params, geo=geo, sets=sets)
    return time.perf_counter() - t0, r


def oracle_setup(cfg):
    from oracle import apic_oracle as O
    from apic_synth import led_kvectors
    kb, kd = led_kvectors(cfg)
    p = O.OracleParams(tile_n=cfg.tile_n, upsample=cfg.upsample, wavelength_um=cfg.wavelength_um,
                       pixel_um=cfg.pixel_um, na_obj=cfg.na_obj, k_bright=kb, k_dark=kd, noll=list(cfg.noll_fit))
    geo = O.Geometry(p)
    sets = O.darkfield_sets(geo)[0] if cfg.n_dark else None
    return p, geo, sets


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from apic_synth import make_tile
    p, geo, sets = oracle_setup(cfg)
    stacks = [make_tile(cfg, t)[0] for t in range(max(1, min(args.steps + args.warmup, 4)))]
    for w in range(args.warmup):
        oracle_step(stacks[w % len(stacks)], p, geo, sets)
    t0 = time.perf_counter()
    for k in range(args.steps):
        oracle_step(stacks[(args.warmup + k) % len(stacks)], p, geo, sets)
    dt = time.perf_counter() - t0
    mpx = args.steps * cfg.out_n ** 2 / 1e6 / dt
    cores = host_threads()
    sample = f"1 tile per step of {workload_name(cfg, 1)}; geometry/index sets prepared once outside the timed region"
    line = {"impl": "reference", "metric": METRIC, "value": mpx, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg, 1), "sample": sample},
            "cpu_baseline": {"value": mpx, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": mpx, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------ clocks
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_id: str):
        self.gpu_id, self.rows, self.proc, self.thread = gpu_id, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", self.gpu_id, f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------ product arm
def main():
    args = parse_args()
    from apic_synth import get_config, make_batch
    cfg = get_config(args.config)
    if args.impl == "reference":
        run_reference(args, cfg)
        return
    assert args.warmup >= 3, "timing rules: at least 3 warm-up steps"
    import torch
    import paper_2407_20469_b200 as A
    A.load()                                            # raises if libapic.so is missing: no fallback
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist = dist_mod
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass

    tiles = args.tiles or min(cfg.batch, 64)
    # seeded synthetic tiles of this rank (weak scaling: every GPU gets its own `tiles` tiles); a few
    # distinct tiles are generated and repeated to fill the batch, each GPU starting at another tile
    n_gen = min(tiles, 8)
    base = (rank * n_gen) % max(1, cfg.batch - n_gen + 1)
    stacks, truths = make_batch(cfg, range(base, base + n_gen))
    reps = -(-tiles // n_gen)
    host = np.concatenate([stacks] * reps)[:tiles]
    x = torch.from_numpy(host).cuda()
    popts = {"df_tol": args.df_tol} if args.df_tol > 0 else {}
    plan = A.Plan.from_config(cfg, max_batch=tiles, chunk_tiles=args.chunk, df_mode=args.df_mode, df_team=args.df_team, **popts)
    n, on, nz = cfg.tile_n, cfg.out_n, plan.nz
    out = (torch.empty((tiles, on, on), dtype=torch.complex64, device="cuda"),
           torch.empty((tiles, nz), dtype=torch.float32, device="cuda"),
           torch.empty((tiles, n, n), dtype=torch.complex64, device="cuda"),
           torch.empty((tiles,), dtype=torch.int32, device="cuda"))

    def barrier():
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        plan.reconstruct(x, out=out)
    barrier()
    sampler = ClockSampler(str(local))
    if os.environ.get("CUDA_VISIBLE_DEVICES"):
        vis = os.environ["CUDA_VISIBLE_DEVICES"].split(",")
        sampler.gpu_id = vis[local] if local < len(vis) else str(local)
    sampler.start()
    plan.profile_begin(stride=1 if args.df_mode != 1 else 4, max_samples=16384)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = 0
    barrier()
    e0.record()
    for _ in range(args.steps):
        plan.reconstruct(x, out=out)
        launches += plan.last_launch_count
    e1.record()
    barrier()
    prof = plan.profile_end()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    if dist:
        t = torch.tensor([ms], device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    status = out[3].cpu().numpy()
    live = int((status != 1).sum())
    mpx = world * args.steps * tiles * on * on / 1e6 / (ms / 1e3)

    # ---- roofline of the dominant kernel: executed flops / CUDA-event time
    chunk = plan.info["chunk_tiles"]
    fft_line = 5.0 * n * math.log2(n)                    # flop of one N-point complex FFT (5 N log2 N)
    sm_max = clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    peak = sms * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    total_kernel_ms = sum(v[0] / max(v[1], 1) * v[2] for v in prof.values())
    dominant = "df_persistent" if args.df_mode != 1 and cfg.n_dark else "df_cols_mul"
    if not cfg.n_dark:
        dominant = max(prof, key=lambda k: prof[k][0] / max(prof[k][1], 1) * prof[k][2])
    ms_sum, samples, nlaunch = prof[dominant]
    avg_ms = ms_sum / max(samples, 1)
    if dominant == "df_persistent":
        # executed work counted by the kernel itself: 5 L log2 L per L-point line transform of its strip tasks
        # (L = N, or the per-LED reduced grid sizes 96..256 of df_mgrid.cu at N = 256)
        flop = plan.profile_work()
        flop_per_launch = flop / max(nlaunch, 1)
        note = (f"{flop:.4g} nominal FFT flop executed (5 L log2 L per L-point line transform, counted by the kernel) "
                f"over {nlaunch} launches; pointwise work not counted")
    elif dominant == "df_cols_mul":
        n_chunks = -(-tiles // chunk)
        flop_per_launch = (2 * n * fft_line + 6.0 * n * n) * tiles / n_chunks
        note = "N columns x (IFFT + FFT) x 5 N log2 N + complex multiply, per tile of the launch"
    else:
        flop_per_launch, note = None, "no flop model for this kernel"
    achieved = flop_per_launch / (avg_ms * 1e-3) / 1e12 if (samples and flop_per_launch) else None
    share = (avg_ms * nlaunch / total_kernel_ms) if total_kernel_ms else None
    # DRAM bytes per launch of that kernel from the committed ncu --set full capture (same workload only)
    traffic = None
    if dominant == "df_persistent" and args.config == 2 and tiles == 64 and args.df_mode == 0:
        try:
            import csv
            with open(os.path.join(ROOT, "profiles", "r1b_traffic_cfg2.csv")) as fh:
                row = next(r for r in csv.DictReader(fh) if r["kernel"] == "df_mgrid_kernel")
            traffic = int(row["dram_bytes_read_per_launch"]) + int(row["dram_bytes_write_per_launch"])
        except Exception:
            traffic = None
    roofline = {"kernel": dominant, "bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": (achieved / peak) if achieved else None, "traffic": traffic,
                "traffic_note": "DRAM read + write bytes per launch, ncu --set full (profiles/r1b_cfg2_mgrid.md); the kernel's "
                                "algorithmic HBM bytes are the 16 darkfield images of each tile = 268 MB per launch, the rest "
                                "is scratch evicted from L2",
                "avg_launch_ms": avg_ms, "sampled_launches": int(samples), "launches": int(nlaunch),
                "share_of_kernel_time": share, "flop_per_launch": flop_per_launch, "flop_model": note,
                "peak_note": f"{sms} SMs x {FP32_LANES_PER_SM} FMA lanes x 2 x {sm_max:.0f} MHz (derived, DESIGN.md §5)",
                "hbm_peak_gbs_measured": peaks.get("hbm_gbs")}
    if args.breakdown and rank == 0:
        print(f"{'kernel':22s} {'launches':>9s} {'avg us':>9s} {'est ms/step':>12s} {'share':>7s}", file=sys.stderr)
        for k, v in sorted(prof.items(), key=lambda kv: -(kv[1][0] / max(kv[1][1], 1) * kv[1][2])):
            est = v[0] / max(v[1], 1) * v[2]
            print(f"{k:22s} {v[2]:9d} {1e3 * v[0] / max(v[1], 1):9.2f} {est / args.steps:12.3f} "
                  f"{est / max(total_kernel_ms, 1e-12):7.3f}", file=sys.stderr)
        print(f"sum of kernel time {total_kernel_ms / args.steps:.3f} ms/step vs step {ms / args.steps:.3f} ms",
              file=sys.stderr)

    # ---- end to end through the host-buffer entry point (pinned memory, copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        hx = torch.from_numpy(host).pin_memory()
        hf = torch.empty((tiles, on, on), dtype=torch.complex64).pin_memory()
        hz = torch.empty((tiles, nz), dtype=torch.float32).pin_memory()
        hp = torch.empty((tiles, n, n), dtype=torch.complex64).pin_memory()
        hs = torch.empty((tiles,), dtype=torch.int32).pin_memory()
        stream = torch.cuda.current_stream().cuda_stream
        plan.reconstruct_host(hx, hf, hz, hp, hs, stream)          # warm-up (allocates the staging buffers)
        k2 = max(1, min(args.steps, 3))
        barrier()
        t0 = time.perf_counter()
        for _ in range(k2):
            plan.reconstruct_host(hx, hf, hz, hp, hs, stream)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if dist:
            t = torch.tensor([dt], device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": world * k2 * tiles * on * on / 1e6 / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(hx.numel() * 4),
               "d2h_bytes_per_step": int(hf.numel() * 8 + hz.numel() * 4 + hp.numel() * 8 + hs.numel() * 4),
               "steps": k2, "api": "apic_reconstruct_host (pinned host buffers, fp32 intensities)"}
        if cfg.noise == "poisson":
            # the same step from the camera's uint16 counts (BASELINE.json config 2: "uint16 raw converted to fp32"):
            # apic_reconstruct_host_u16, half the host-to-device bytes; reported beside the fp32 number, not instead
            gains = np.array([[t.gain_bright] * cfg.n_bright + [t.gain_dark] * cfg.n_dark for t in truths])
            gains = np.concatenate([gains] * reps)[:tiles]
            raw = np.rint(host.astype(np.float64) * gains[:, :, None, None]).astype(np.uint16)
            hr = torch.from_numpy(raw).pin_memory()
            hsc = torch.from_numpy((1.0 / gains).astype(np.float32)).pin_memory()
            plan.reconstruct_host_u16(hr, hsc, hf, hz, hp, hs, stream)
            barrier()
            t0 = time.perf_counter()
            for _ in range(k2):
                plan.reconstruct_host_u16(hr, hsc, hf, hz, hp, hs, stream)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            if dist:
                t = torch.tensor([dt], device="cuda")
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                dt = float(t.item())
            e2e["u16"] = {"value": world * k2 * tiles * on * on / 1e6 / dt, "unit": UNIT,
                          "h2d_bytes_per_step": int(hr.numel() * 2 + hsc.numel() * 4),
                          "api": "apic_reconstruct_host_u16 (pinned host buffers, uint16 counts + per-image scale)"}

    # ---- the oracle on this box's host cores (rank 0, N = 1 only): one tile of the same workload
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        p, geo, sets = oracle_setup(cfg)
        dt, _ = oracle_step(host[0], p, geo, sets)
        cpu = {"value": on * on / 1e6 / dt, "unit": UNIT, "cores": host_threads(), "kind": "oracle",
               "sample": f"1 of the {tiles} tiles of the step ({dt:.1f} s), index sets prepared outside the timed region"}

    if rank == 0:
        line = {"metric": METRIC, "value": mpx, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": workload_name(cfg, tiles), "tiles_per_step_per_gpu": tiles,
                           "tiles_per_s": world * args.steps * tiles / (ms / 1e3), "chunk_tiles": chunk,
                           "live_tiles": live, "cache": "inputs larger than L2 "
                           f"({host.nbytes / 1e6:.0f} MB per step vs 126 MB L2)", "parallelism": f"tiles x{world}"},
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
                "cpu_baseline": cpu}
        print(json.dumps(line), flush=True)
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
