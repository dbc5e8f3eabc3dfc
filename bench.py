#!/usr/bin/env python
"""Throughput of the APIC closed-form reconstruction on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl apic|reference] [--config 2]

A step = one pass of the whole hot path (S0-S10 of DESIGN.md) over one batch of synthetic tiles.
Default workload: BASELINE.json config 2 (64 tiles of 256x256, 8 NA-matching + 16 darkfield LEDs,
Poisson noise, 3x output grid) - the batched 256x256 configuration the north-star target is quoted
on (config 1 is a single tile, i.e. a latency case).  Prints ONE JSON line.

  value     output megapixels/s with the inputs resident in HBM (CUDA events, max over ranks)
  e2e       the same metric through apic_submit_host / apic_wait_host with pinned HOST buffers (H2D + D2H inside;
            two batches in flight), and through the blocking apic_reconstruct_host beside it
  roofline  the dominant kernel (df_wide_kernel: the darkfield CG on reduced cyclic grids), timed live by CUDA
            events inside the library on the launching stream, against fp32 peaks MEASURED in this run
            (apic_measure_peak: FFMA and FADD register loops, shared-memory reads)
  cpu_baseline  the fp64 oracle, as it stands, on this box's host cores, on a bounded sample
`--impl reference` times the oracle alone (rank 0 only under torchrun).
`--config 4` is the slide-scale streaming run: 20,000 tiles generated on the device from a seed
(apic_synth/device.py), 40 % of them background, reconstructed in passes through apic_reconstruct_u16; every status
flag is checked against the generator's blank mask; `--oracle-sample M` also compares M live tiles with the oracle.
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
    ap.add_argument("--steps", type=int, default=0, help="timed steps (default 20; config 4: every pass of the slide)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="apic", choices=["apic", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (2 = default workload)")
    ap.add_argument("--tiles", type=int, default=0, help="tiles per step and per GPU (0 = the config's batch, capped at 64)")
    ap.add_argument("--distinct-tiles", type=int, default=0, help="distinct seeded tiles generated per GPU and repeated to fill "
                    "the step (0 = every tile of the step distinct)")
    ap.add_argument("--chunk", type=int, default=0, help="apic_params.chunk_tiles (0 = library default)")
    ap.add_argument("--df-mode", type=int, default=0, help="darkfield kernel (apic.h): 0 default (df_wide.cu, 256-thread CTAs at 128 registers), "
                    "3 full grid, 4 async-proxy staging, 5 1024-thread CTA pairs with the decimated CG loop, 6 the round-1 kernel")
    ap.add_argument("--pass-tiles", type=int, default=592, help="config 4: tiles per apic_reconstruct_u16 call (a step)")
    ap.add_argument("--oracle-sample", type=int, default=0, help="config 4: live tiles compared with the fp64 oracle after the run")
    ap.add_argument("--df-order", type=int, default=0, help="apic_params.df_order: 0 sequential (R15, the headline), 1 ring-wise (R15b)")
    ap.add_argument("--df-team", type=int, default=0, help="apic_params.df_team: CTAs per tile of the team kernel (0 = auto)")
    ap.add_argument("--df-tol", type=float, default=-1.0, help="CG tolerance (default: the library's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--breakdown", action="store_true", help="also print the per-kernel time table to stderr")
    ap.add_argument("--ncu-summary", default="", help="no run: append the kernels of an `ncu -i <rep> --page raw --csv` dump "
                    "to profiles/r3_ncu_kernels.csv (with --commit and --workload)")
    ap.add_argument("--commit", default="", help="--ncu-summary: the commit the capture was taken at")
    ap.add_argument("--workload", default="", help="--ncu-summary: workload tag, e.g. cfg2_64tiles")
    ap.add_argument("--reassemble", action="store_true", help="no reconstruction: time apic_reassemble (within-FOV reassembly of "
                    "5 x 5 tiles of 768 x 768 output pixels with 10 %% overlap) against the HBM roofline")
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
            self.rows.append([c.strip() for c in line.split(",")] + [time.perf_counter()])

    def mark(self):
        """The timed region starts now: only samples that arrive from here on count (nvidia-smi is started before the
        warm-up steps because its first sample can take longer than a short timed region)."""
        self.t_mark = time.perf_counter()

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        t_mark = getattr(self, "t_mark", None)
        rows = [r for r in self.rows if t_mark is None or r[-1] >= t_mark]
        if not rows:
            rows = self.rows[-3:]                        # a timed region shorter than the sampling period: the samples of
        for r in rows:                                   # the warm-up steps right before it (the GPU was under the same load)
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------ roofline helpers
KERNEL_SOURCES = ("df_wide.cu", "df_mgrid.cu", "df_tma.cu", "df_team.cu", "fft_xy.cuh", "fft_core.cuh")


def kernel_source_hash():
    """Identifies the darkfield kernel sources an ncu capture under profiles/ was taken with (the GPU box has no .git)."""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2407_20469_b200", "csrc", name), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def kernel_short_name(full):
    """'void apic::wd::df_wide_kernel<1, 2>(apic::wd::Args)' -> 'df_wide_kernel'; '<unnamed>::peak_alu_kernel<0>(...)' -> 'peak_alu_kernel'."""
    import re
    s = full.replace("<unnamed>", "anon")
    s = s.split("(")[0]
    s = re.sub(r"<[^<>]*>", "", s)
    return s.split("::")[-1].replace("void ", "").strip()


def ncu_capture(kernel, workload):
    """Per-launch DRAM bytes and shared-memory wavefronts of `kernel` from the committed ncu --set full summary
    (profiles/r3_ncu_kernels.csv).  A row taken with other kernel sources than the ones in the tree is refused."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "r3_ncu_kernels.csv")) as fh:
            rows = [r for r in csv.DictReader(fh) if r["kernel"] == kernel and r["workload"] == workload]
    except Exception:
        return None
    if not rows:
        return None
    r = rows[-1]
    if r["source_hash"] != kernel_source_hash():
        return {"stale": True, "source_hash": r["source_hash"]}
    return {"stale": False, "dram_bytes": int(r["dram_bytes_read"]) + int(r["dram_bytes_write"]),
            "smem_wavefronts": int(r["smem_wavefronts"]), "duration_ms": float(r["duration_ms"]), "commit": r["commit"]}


def ncu_summary(args):
    """Reduces an `ncu --page raw --csv` dump of an `ncu --set full` capture to one row per kernel launch in
    profiles/r3_ncu_kernels.csv: what bench.py's roofline line reads (traffic, smem_frac) plus the figures DESIGN.md
    quotes (issue-slot utilisation, occupancy, L2 hit rate, stall shares)."""
    import csv
    with open(args.ncu_summary) as fh:
        rows = list(csv.reader(fh))
    hdr, units = rows[0], rows[1]
    ix = {h: i for i, h in enumerate(hdr)}

    def val(r, key, scale_units=True):
        v = r[ix[key]].replace(",", "")
        if v in ("", "n/a"):
            return 0.0
        x = float(v)
        u = units[ix[key]]
        if scale_units:
            x *= {"Mbyte": 1e6, "Gbyte": 1e9, "Kbyte": 1e3, "byte": 1.0, "us": 1e-3, "ns": 1e-6, "ms": 1.0, "s": 1e3}.get(u, 1.0)
        return x

    out_path = os.path.join(ROOT, "profiles", "r3_ncu_kernels.csv")
    fields = ["kernel", "workload", "commit", "source_hash", "duration_ms", "dram_bytes_read", "dram_bytes_write",
              "smem_wavefronts", "inst_executed", "issue_active_pct", "warps_active_pct", "l2_hit_pct", "registers",
              "dyn_smem_bytes", "grid", "cluster", "stall_barrier_pct", "stall_long_sb_pct", "stall_short_sb_pct",
              "stall_wait_pct", "stall_membar_pct"]
    new = not os.path.exists(out_path)
    with open(out_path, "a", newline="") as fh:
        w = csv.DictWriter(fh, fieldnames=fields)
        if new:
            w.writeheader()
        for r in rows[2:]:
            name = kernel_short_name(r[ix["Kernel Name"]])
            stall = {k: val(r, f"smsp__average_warps_issue_stalled_{k}_per_issue_active.ratio", False)
                     for k in ("barrier", "long_scoreboard", "short_scoreboard", "wait", "membar", "no_instruction", "not_selected",
                               "selected", "math_pipe_throttle", "mio_throttle", "lg_throttle", "branch_resolving", "dispatch_stall",
                               "drain", "imc_miss", "sleeping", "tex_throttle", "misc")
                     if f"smsp__average_warps_issue_stalled_{k}_per_issue_active.ratio" in ix}
            tot = sum(stall.values()) or 1.0
            w.writerow({"kernel": name, "workload": args.workload, "commit": args.commit, "source_hash": kernel_source_hash(),
                        "duration_ms": f"{val(r, 'gpu__time_duration.sum'):.4f}",
                        "dram_bytes_read": int(val(r, "dram__bytes_read.sum")), "dram_bytes_write": int(val(r, "dram__bytes_write.sum")),
                        "smem_wavefronts": int(val(r, "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum")),
                        "inst_executed": int(val(r, "smsp__inst_executed.sum")),
                        "issue_active_pct": f"{val(r, 'smsp__issue_active.avg.pct_of_peak_sustained_active'):.2f}",
                        "warps_active_pct": f"{val(r, 'sm__warps_active.avg.pct_of_peak_sustained_active'):.2f}",
                        "l2_hit_pct": f"{val(r, 'lts__t_sector_hit_rate.pct'):.2f}",
                        "registers": int(val(r, "launch__registers_per_thread")),
                        "dyn_smem_bytes": int(val(r, "launch__shared_mem_per_block_dynamic")),
                        "grid": int(val(r, "launch__grid_size")), "cluster": int(val(r, "launch__cluster_dim_x")),
                        "stall_barrier_pct": f"{100 * stall.get('barrier', 0) / tot:.1f}",
                        "stall_long_sb_pct": f"{100 * stall.get('long_scoreboard', 0) / tot:.1f}",
                        "stall_short_sb_pct": f"{100 * stall.get('short_scoreboard', 0) / tot:.1f}",
                        "stall_wait_pct": f"{100 * stall.get('wait', 0) / tot:.1f}",
                        "stall_membar_pct": f"{100 * stall.get('membar', 0) / tot:.1f}"})
            print("appended", name, args.workload, "to", out_path)


def reassemble_bench(args):
    """apic_reassemble on FOVs shaped like the paper's (5 x 5 patches per FOV) with config 4's 10 % overlap:
    25 tiles of 768 x 768 complex64 in, one 3536 x 3536 FOV out per call; several FOVs so that the data exceeds the L2."""
    import torch
    import paper_2407_20469_b200 as A
    torch.cuda.set_device(0)
    ty = tx = 5
    t, ov, n_fov = 768, 76, 4
    g = torch.Generator(device="cuda").manual_seed(1)
    tiles = [torch.view_as_complex(torch.rand((ty, tx, t, t, 2), device="cuda", generator=g) - 0.5).contiguous() for _ in range(n_fov)]
    h = ty * (t - ov) + ov
    outs = [torch.empty((h, h), dtype=torch.complex64, device="cuda") for _ in range(n_fov)]
    steps = max(args.steps or 20, 1)
    for w in range(max(args.warmup, 3)):
        for f, o in zip(tiles, outs):
            A.reassemble(f, ov, True, out=o)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(steps):
        for f, o in zip(tiles, outs):
            A.reassemble(f, ov, True, out=o)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / (steps * n_fov)
    overlap_bytes = (ty * (tx - 1) + tx * (ty - 1)) * 2 * ov * t * 8          # the correlation pass reads every overlap twice
    algo = ty * tx * t * t * 8 + h * h * 8 + overlap_bytes
    peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
    peak = peaks.get("hbm_gbs", 6650.0)
    gbs = algo / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "reassembled FOV megapixels/sec", "value": h * h / 1e6 / (ms * 1e-3), "unit": "Mpx/s",
                      "ms_per_fov": ms, "steps": steps, "fovs_per_step": n_fov, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": f"{ty} x {tx} tiles of {t} x {t} complex64, overlap {ov}, FOV {h} x {h}, align on; "
                                             f"{n_fov} FOVs per step ({n_fov * algo / 1e6:.0f} MB > L2)"},
                      "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                                   "algorithmic_bytes_per_fov": algo, "traffic": None,
                                   "peak_note": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6650 GB/s"}}), flush=True)


def measured_peaks(A, torch, sm_mhz_max, sms):
    """fp32 FFMA / FADD rates and shared-memory read bandwidth measured on this device now; the derived figures
    (unit counts x clock) beside them."""
    fma = A.measure_peak(0) / 1e12
    fadd = A.measure_peak(1) / 1e12
    smem = A.measure_peak(2) / 1e12
    return {"fp32_fma_tflops": fma, "fp32_fadd_tflops": fadd, "smem_tbs": smem,
            "fp32_fma_tflops_derived": sms * FP32_LANES_PER_SM * 2 * sm_mhz_max * 1e6 / 1e12,
            "smem_tbs_derived": sms * 128 * sm_mhz_max * 1e6 / 1e12,
            "how": "apic_measure_peak: register-resident FFMA / FADD loops (8 independent accumulators, 4 x 512 threads per "
                   "SM) and conflict-free 16-byte shared-memory loads, best of 3 after warm-up, CUDA events"}


# ------------------------------------------------------------------------------------ product arm
def main():
    args = parse_args()
    if args.ncu_summary:
        ncu_summary(args)
        return
    if args.reassemble:
        reassemble_bench(args)
        return
    from apic_synth import get_config, make_batch, plan_args
    cfg = get_config(args.config)
    if args.impl == "reference":
        args.steps = args.steps or 20
        run_reference(args, cfg)
        return
    assert args.warmup >= 3, "timing rules: at least 3 warm-up steps"
    import torch
    import paper_2407_20469_b200 as A
    from paper_2407_20469_b200.sharding import max_over_ranks, shard_tiles
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
    ctx = dict(args=args, cfg=cfg, torch=torch, A=A, rank=rank, world=world, local=local, dist=dist, peaks=peaks,
               max_over_ranks=max_over_ranks, shard_tiles=shard_tiles)
    if args.config == 4:
        run_stream(ctx)
    else:
        args.steps = args.steps or 20
        run_batch(ctx)
    if dist:
        dist.destroy_process_group()


def make_sampler(local):
    sampler = ClockSampler(str(local))
    if os.environ.get("CUDA_VISIBLE_DEVICES"):
        vis = os.environ["CUDA_VISIBLE_DEVICES"].split(",")
        sampler.gpu_id = vis[local] if local < len(vis) else str(local)
    return sampler


def roofline_line(ctx, plan, prof, clocks, tiles, workload, step_ms, algo_hbm_bytes_per_step):
    """The dominant kernel against the measured fp32 peaks."""
    args, cfg, torch, A = ctx["args"], ctx["cfg"], ctx["torch"], ctx["A"]
    peaks = ctx["peaks"]
    sm_max = clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
    sms = torch.cuda.get_device_properties(ctx["local"]).multi_processor_count
    mp = measured_peaks(A, torch, sm_max, sms)
    total_kernel_ms = sum(v[0] / max(v[1], 1) * v[2] for v in prof.values())
    dominant = max(prof, key=lambda k: prof[k][0] / max(prof[k][1], 1) * prof[k][2])
    ms_sum, samples, nlaunch = prof[dominant]
    avg_ms = ms_sum / max(samples, 1)
    share = (avg_ms * nlaunch / total_kernel_ms) if total_kernel_ms else None
    hbm_peak = peaks.get("hbm_gbs") or peaks.get("hbm_gbs_burst")
    out = {"kernel": dominant, "avg_launch_ms": avg_ms, "sampled_launches": int(samples), "launches": int(nlaunch),
           "share_of_kernel_time": share, "measured_peaks": mp,
           "step_hbm": {"algorithmic_bytes_per_step": int(algo_hbm_bytes_per_step),
                        "achieved_gbs": algo_hbm_bytes_per_step / (step_ms * 1e-3) / 1e9, "peak_gbs": hbm_peak,
                        "frac": (algo_hbm_bytes_per_step / (step_ms * 1e-3) / 1e9 / hbm_peak) if hbm_peak else None,
                        "note": "inputs read once + outputs written once per step, over the whole step time"}}
    if dominant.startswith("df_"):
        # executed work counted by the kernel itself: 5 L log2 L per L-point line transform of its strip tasks
        # (L = N, or the per-LED reduced grid sizes 96..256 of df_mgrid.cu at N = 256); pointwise work not counted
        flop = plan.profile_work()
        flop_per_launch = flop / max(nlaunch, 1)
        achieved = flop_per_launch / (avg_ms * 1e-3) / 1e12 if samples else None
        cap = ncu_capture(dominant, workload)
        traffic, smem_frac, cap_note = None, None, "no ncu --set full capture of this kernel and workload under profiles/"
        if cap and cap.get("stale"):
            cap_note = "profiles/r3_ncu_kernels.csv was captured with other kernel sources (hash mismatch): refused"
        elif cap:
            traffic = cap["dram_bytes"]
            # 128 bytes per shared-memory wavefront, against the measured shared-memory read bandwidth
            smem_frac = cap["smem_wavefronts"] * 128.0 / (cap["duration_ms"] * 1e-3) / (mp["smem_tbs"] * 1e12)
            cap_note = f"ncu --set full at commit {cap['commit']} (profiles/r3_ncu_kernels.csv), per launch"
        out.update({"bound": "alu", "achieved": achieved, "peak": mp["fp32_fma_tflops"], "unit": "TFLOP/s",
                    "frac": (achieved / mp["fp32_fma_tflops"]) if achieved else None,
                    "frac_of_fadd_peak": (achieved / mp["fp32_fadd_tflops"]) if achieved else None,
                    "traffic": traffic, "smem_frac": smem_frac, "ncu": cap_note,
                    "flop_per_launch": flop_per_launch,
                    "flop_model": "nominal FFT flop executed, 5 L log2 L per L-point line transform, counted by the kernel; an "
                                  "add-dominated radix-16 butterfly executes ~0.66 fp32 instructions per nominal flop, so the "
                                  "instruction-issue roof in these units is ~1.5 x the FADD peak / 2 (DESIGN.md section 5)",
                    "peak_note": "fp32 FFMA rate measured in this run (flop = 2 x FMA); FADD rate beside it"})
    else:
        # HBM-bound kernels (no darkfield LEDs): the whole step against the measured copy bandwidth
        out.update({"bound": "hbm", "achieved": out["step_hbm"]["achieved_gbs"], "peak": hbm_peak, "unit": "GB/s",
                    "frac": out["step_hbm"]["frac"], "traffic": None})
    if args.breakdown and ctx["rank"] == 0:
        print(f"{'kernel':22s} {'launches':>9s} {'avg us':>9s} {'est ms/step':>12s} {'share':>7s}", file=sys.stderr)
        for k, v in sorted(prof.items(), key=lambda kv: -(kv[1][0] / max(kv[1][1], 1) * kv[1][2])):
            est = v[0] / max(v[1], 1) * v[2]
            print(f"{k:22s} {v[2]:9d} {1e3 * v[0] / max(v[1], 1):9.2f} {est / max(args.steps, 1):12.3f} "
                  f"{est / max(total_kernel_ms, 1e-12):7.3f}", file=sys.stderr)
        print(f"sum of kernel time {total_kernel_ms / max(args.steps, 1):.3f} ms/step vs step {step_ms:.3f} ms", file=sys.stderr)
    return out


def run_batch(ctx):
    args, cfg, torch, A, rank, world, local, dist = (ctx[k] for k in ("args", "cfg", "torch", "A", "rank", "world", "local", "dist"))
    from apic_synth import make_batch, plan_args
    tiles = args.tiles or min(cfg.batch, 64)
    # seeded synthetic tiles of this rank (weak scaling: every GPU gets its own `tiles` tiles), every tile of the step
    # distinct (generated on the host, outside every timed region; --distinct-tiles M repeats M tiles to fill the
    # batch, for quick runs), each GPU starting at another tile
    n_gen = min(tiles, args.distinct_tiles or tiles, max(1, cfg.batch))
    base = (rank * n_gen) % max(1, cfg.batch - n_gen + 1)
    if n_gen > 8:
        # tiles are seeded per index, so generating them side by side on the host threads changes nothing but the wait
        import concurrent.futures as cf
        with cf.ThreadPoolExecutor(max_workers=min(16, host_threads())) as ex:
            made = list(ex.map(lambda t: make_batch(cfg, [t]), range(base, base + n_gen)))
        stacks, truths = np.concatenate([m[0] for m in made]), [m[1][0] for m in made]
    else:
        stacks, truths = make_batch(cfg, range(base, base + n_gen))
    reps = -(-tiles // n_gen)
    host = np.concatenate([stacks] * reps)[:tiles]
    x = torch.from_numpy(host).cuda()
    popts = {"df_tol": args.df_tol} if args.df_tol > 0 else {}
    plan = A.Plan(*plan_args(cfg), max_batch=tiles, chunk_tiles=args.chunk, df_mode=args.df_mode, df_team=args.df_team, df_order=args.df_order, **popts)
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

    sampler = make_sampler(local)
    sampler.start()
    for _ in range(args.warmup):
        plan.reconstruct(x, out=out)
    barrier()
    sampler.mark()
    plan.profile_begin(stride=1, max_samples=16384)
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
    ms = ctx["max_over_ranks"](e0.elapsed_time(e1), dist, device="cuda")
    status = out[3].cpu().numpy()
    n_ok = int((status == 0).sum())
    if n_ok != tiles:
        raise SystemExit(f"bench: {tiles - n_ok} of {tiles} tiles were not reconstructed (status {np.unique(status).tolist()}); "
                         "the throughput of a failed step is not a result")
    mpx = world * args.steps * tiles * on * on / 1e6 / (ms / 1e3)
    chunk = plan.info["chunk_tiles"]
    workload = f"cfg{args.config}_{tiles}tiles" + (f"_mode{args.df_mode}" if args.df_mode else "")   # tag of the ncu rows under profiles/
    algo_bytes = tiles * (host[0].nbytes + on * on * 8 + n * n * 8 + nz * 4 + 4)
    roofline = roofline_line(ctx, plan, prof, clocks, tiles, workload, ms / args.steps, algo_bytes)

    # ---- end to end through the host-buffer entry points (pinned memory, copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        hx = torch.from_numpy(host).pin_memory()
        outs = [(torch.empty((tiles, on, on), dtype=torch.complex64).pin_memory(),
                 torch.empty((tiles, nz), dtype=torch.float32).pin_memory(),
                 torch.empty((tiles, n, n), dtype=torch.complex64).pin_memory(),
                 torch.empty((tiles,), dtype=torch.int32).pin_memory()) for _ in range(2)]
        hf, hz, hp, hs = outs[0]
        stream = torch.cuda.current_stream().cuda_stream
        k2 = max(6, args.steps)      # the same K as the device-timed loop (pipeline fill and drain are inside the timed region)
        ref_field = out[0].cpu().numpy()

        def timed(step_fn, drain_fn=None):
            """k2 steps after three warm-up steps (the first use of a pipeline slot allocates its workspace set and its
            staging buffers: both slots are warm before the clock starts); seconds, max over ranks."""
            for w in range(3):
                step_fn(w)
            if drain_fn:
                drain_fn()
            torch.cuda.synchronize()
            barrier()
            t0 = time.perf_counter()
            for i in range(k2):
                step_fn(i)
            if drain_fn:
                drain_fn()
            torch.cuda.synchronize()
            return ctx["max_over_ranks"](time.perf_counter() - t0, dist, device="cuda")

        def drain():
            plan.wait_host(0)
            plan.wait_host(1)

        # (1) streaming: apic_submit_host / apic_wait_host, one batch in flight per pipeline slot; every step uploads
        # its inputs from pinned memory and its results are read back to pinned memory (two output buffer sets)
        dt = timed(lambda i: plan.submit_host(i & 1, hx, *outs[i & 1]), drain)
        assert all(np.array_equal(o[0].numpy(), ref_field) for o in outs), "streaming host entry and device entry disagree"
        d2h = int(hf.numel() * 8 + hz.numel() * 4 + hp.numel() * 8 + hs.numel() * 4)
        e2e = {"value": world * k2 * tiles * on * on / 1e6 / dt, "unit": UNIT, "h2d_bytes_per_step": int(hx.numel() * 4),
               "d2h_bytes_per_step": d2h, "steps": k2, "input": "fp32 intensities",
               "api": "apic_submit_host / apic_wait_host (pinned host buffers, fp32 intensities, two batches in flight)"}
        # (2) one blocking call per step: upload, kernels and download of a step overlap only inside the call
        dt = timed(lambda i: plan.reconstruct_host(hx, hf, hz, hp, hs, stream))
        assert np.array_equal(hf.numpy(), ref_field), "host entry and device entry disagree"
        e2e["single_call"] = {"value": world * k2 * tiles * on * on / 1e6 / dt, "unit": UNIT,
                              "api": "apic_reconstruct_host (blocking, sub-batches pipelined inside the call)"}
        if cfg.noise == "poisson":
            # the same step from the camera's uint16 counts (BASELINE.json config 2: "uint16 raw converted to fp32"):
            # half the host-to-device bytes; reported beside the fp32 number, not instead
            gains = np.array([[t.gain_bright] * cfg.n_bright + [t.gain_dark] * cfg.n_dark for t in truths])
            gains = np.concatenate([gains] * reps)[:tiles]
            raw = np.rint(host.astype(np.float64) * gains[:, :, None, None]).astype(np.uint16)
            hr = torch.from_numpy(raw).pin_memory()
            hsc = torch.from_numpy((1.0 / gains).astype(np.float32)).pin_memory()
            dt = timed(lambda i: plan.submit_host_u16(i & 1, hr, hsc, *outs[i & 1]), drain)
            e2e["u16"] = {"value": world * k2 * tiles * on * on / 1e6 / dt, "unit": UNIT,
                          "h2d_bytes_per_step": int(hr.numel() * 2 + hsc.numel() * 4), "d2h_bytes_per_step": d2h,
                          "api": "apic_submit_host_u16 / apic_wait_host (uint16 counts + per-image scale, two batches in flight)"}
            dt = timed(lambda i: plan.reconstruct_host_u16(hr, hsc, hf, hz, hp, hs, stream))
            e2e["u16"]["single_call"] = {"value": world * k2 * tiles * on * on / 1e6 / dt, "unit": UNIT,
                                         "api": "apic_reconstruct_host_u16 (blocking)"}
            # BASELINE.json states this workload as "uint16 raw converted to fp32": what a user uploads is the camera's
            # counts, so the uint16 streaming entry is the declared end-to-end number and the fp32-host one sits beside it
            f32 = {k: e2e[k] for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "api", "single_call")}
            u16 = e2e["u16"]
            e2e = {"value": u16["value"], "unit": UNIT, "h2d_bytes_per_step": u16["h2d_bytes_per_step"],
                   "d2h_bytes_per_step": d2h, "steps": k2, "input": "uint16 counts + per-image fp32 scale",
                   "api": u16["api"], "single_call": u16["single_call"], "f32": f32}

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
                           "distinct_tiles": n_gen, "tiles_ok": n_ok, "df_mode": args.df_mode, "df_order": args.df_order,
                           "tiles_per_s": world * args.steps * tiles / (ms / 1e3), "chunk_tiles": chunk,
                           "cache": "inputs larger than L2 "
                           f"({host.nbytes / 1e6:.0f} MB per step vs 126 MB L2)", "parallelism": f"tiles x{world}"},
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
                "cpu_baseline": cpu}
        print(json.dumps(line), flush=True)


def run_stream(ctx):
    """BASELINE.json config 4: the slide-scale streaming run.  A step = one pass of `--pass-tiles` tiles (generated on
    the device outside the timed region, then reconstructed from uint16 counts inside it)."""
    args, cfg, torch, A, rank, world, local, dist = (ctx[k] for k in ("args", "cfg", "torch", "A", "rank", "world", "local", "dist"))
    from apic_synth import plan_args
    from apic_synth.device import DeviceGenerator
    total = args.tiles or cfg.batch
    mine = ctx["shard_tiles"](total, rank, world)                      # contiguous scan-row ranges per GPU, no collective
    P = max(1, min(args.pass_tiles, len(mine)))
    passes = [(t0, min(P, mine.stop - t0)) for t0 in range(mine.start, mine.stop, P)]
    if args.steps:
        passes = passes[:args.steps]
    bg = dict(bg_mode=1, bg_threshold=0.9)
    plan = A.Plan(*plan_args(cfg), max_batch=P, chunk_tiles=args.chunk, df_team=args.df_team, **bg)
    gen = DeviceGenerator(cfg, device=f"cuda:{local}")
    n, on, nz = cfg.tile_n, cfg.out_n, plan.nz
    out = (torch.empty((P, on, on), dtype=torch.complex64, device="cuda"), torch.empty((P, nz), dtype=torch.float32, device="cuda"),
           torch.empty((P, n, n), dtype=torch.complex64, device="cuda"), torch.empty((P,), dtype=torch.int32, device="cuda"))

    def barrier():
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
            torch.cuda.synchronize()

    raw, scale, blank = gen.generate(*passes[0])
    for _ in range(args.warmup):
        plan.reconstruct_u16(raw, scale, out=tuple(o[:raw.shape[0]] for o in out))
    barrier()
    want = args.oracle_sample if (rank == 0 and world == 1) else 0
    live_all = np.nonzero(~gen.blank[mine.start:mine.stop])[0] + mine.start
    pick = set(live_all[np.linspace(0, len(live_all) - 1, want).astype(int)].tolist()) if want else set()
    kept = []
    sampler = make_sampler(local)
    sampler.start()
    plan.profile_begin(stride=1, max_samples=16384)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in passes]
    launches, n_live, n_done, wrong, in_bytes = 0, 0, 0, 0, 0
    barrier()
    for k, (t0, cnt) in enumerate(passes):
        if k:
            raw, scale, blank = gen.generate(t0, cnt)
        o = tuple(x[:cnt] for x in out)
        torch.cuda.synchronize()
        ev[k][0].record()
        plan.reconstruct_u16(raw, scale, out=o)
        ev[k][1].record()
        launches += plan.last_launch_count
        status = o[3].cpu().numpy()
        wrong += int(np.count_nonzero((status == 1) != blank) + np.count_nonzero((status != 1) & (status != 0)))
        n_live += int((status == 0).sum())
        n_done += cnt
        in_bytes += raw.numel() * 2 + scale.numel() * 4
        for b in range(cnt):
            if t0 + b in pick:
                kept.append((t0 + b, (raw[b].cpu().numpy().astype(np.float32) * scale[b].cpu().numpy()[:, None, None]),
                             o[0][b].cpu().numpy(), o[1][b].cpu().numpy()))
    barrier()
    prof = plan.profile_end()
    clocks = sampler.stop()
    ms = ctx["max_over_ranks"](sum(a.elapsed_time(b) for a, b in ev), dist, device="cuda")
    n_live_all = ctx_sum(ctx, n_live)
    n_done_all = ctx_sum(ctx, n_done)
    wrong_all = ctx_sum(ctx, wrong)
    if wrong_all:
        raise SystemExit(f"bench --config 4: {wrong_all} status flags disagree with the generator's blank mask")
    workload = f"cfg4_{P}tiles"
    algo = in_bytes + n_live * (on * on * 8 + n * n * 8 + nz * 4)
    roofline = roofline_line(ctx, plan, prof, clocks, P, workload, ms / len(passes), algo / len(passes))
    sample = None
    if kept:
        from oracle import apic_oracle as O
        p, geo, sets = oracle_setup(cfg)
        p.bg_mode, p.bg_threshold = 1, 0.9
        worst_f = worst_c = 0.0
        for t, x, f, z in kept:
            r = O.reconstruct_tile(x, p, geo=geo, sets=sets)
            assert r.status == 0
            worst_f = max(worst_f, float(np.linalg.norm(f - r.field) / np.linalg.norm(r.field)))
            worst_c = max(worst_c, float(np.linalg.norm(z - r.zernike)))
        sample = {"tiles": [k[0] for k in kept], "worst_field_rel_l2": worst_f, "worst_pupil_rad": worst_c,
                  "within_contract": bool(worst_f <= 1e-4 and worst_c <= 1e-3)}
    if rank == 0:
        mpx_live = n_live_all * on * on / 1e6 / (ms / 1e3)
        line = {"metric": METRIC, "value": mpx_live, "unit": UNIT, "n_gpus": world, "steps": len(passes), "warmup": args.warmup,
                "ms_per_step": ms / len(passes), "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic (generated on the device from a seed, apic_synth/device.py)",
                "config": {"workload": workload_name(cfg, P) + f"; slide of {total} tiles, {world} GPU(s)",
                           "tiles_done": n_done_all, "tiles_live": n_live_all, "tiles_background": n_done_all - n_live_all,
                           "status_flags_checked": n_done_all, "status_flags_wrong": 0,
                           "value_counts": "pixels of reconstructed (non-background) tiles only",
                           "mpx_per_s_counting_skipped_tiles": n_done_all * on * on / 1e6 / (ms / 1e3),
                           "output_gpx_live": n_live_all * on * on / 1e9, "tiles_per_s": n_done_all / (ms / 1e3),
                           "chunk_tiles": plan.info["chunk_tiles"], "input": "uint16 counts + per-image scale (apic_reconstruct_u16)",
                           "cache": f"inputs larger than L2 ({raw.numel() * 2 / 1e6:.0f} MB per pass vs 126 MB L2)",
                           "oracle_sample": sample},
                "clocks": clocks, "e2e": None, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": None}
        print(json.dumps(line), flush=True)


def ctx_sum(ctx, v):
    dist = ctx["dist"]
    if not dist:
        return v
    t = ctx["torch"].tensor([float(v)], dtype=ctx["torch"].float64, device="cuda")
    dist.all_reduce(t)
    return int(t.item())


if __name__ == "__main__":
    main()
