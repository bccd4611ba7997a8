#!/usr/bin/env python
"""bench.py -- the headline measurement (BASELINE.json `metric`): 52-channel NBS correlator
time-slices/s at 32^3 x 64 in FP64 on one B200, with the dominant kernel's roofline fraction.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

A "step" is one pass of the whole hot path (blocks -> FFT -> effective blocks x product -> inverse
FFT -> F[52][256][V]) over one time slice of synthetic propagators of BASELINE.json configs[2]
(32^3 x 64, u != d != s, Gaussian entries x exp(-m t), seed 3).  N > 1: "replicas only" -- time
slices are independent (T-parallel), every rank runs its own slices, no collective on
the data path; `value` = slices of all ranks / max-over-ranks time.
`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "nbs_correlator_time_slices_per_s_52ch_32c64_fp64"  # configs[2]; other --config values rename it (metric_name)


def metric_name(cfg_index: int, cfg: dict, L: int) -> str:
    return METRIC if cfg_index == 2 else f"nbs_correlator_time_slices_per_s_52ch_{L}c{cfg['T']}_fp64"
UNIT = "time-slices/s"
# Cross-check only: 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz.  The roofline denominator is
# MEASURED in this process by nbs_probe_fp64 (register-resident DMMA.8x8x4 on all SMs, include/nbs.h).
FP64_PEAK_DERIVED_TFLOPS = 37.2
# dram__bytes_read.sum + dram__bytes_write.sum of one k_product_c launch on configs[2], parsed from the committed
# `ncu --set full` capture of the benched kernel (the .md beside it names the command and the commit)
PRODUCT_NCU_CSV = os.path.join(ROOT, "profiles", "r2_product_ncu.csv")


def product_dram_traffic():
    """(bytes per launch, source) from profiles/r2_product_ncu.csv, or (None, reason)."""
    try:
        rd = wr = None
        with open(PRODUCT_NCU_CSV) as fh:
            for line in fh:
                cells = [c.strip().strip('"') for c in line.split(",")]
                if len(cells) < 3:
                    continue
                name, unit, val = cells[0], cells[1].lower(), cells[2]
                if name not in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                    continue
                scale = {"byte": 1.0, "kbyte": 1e3, "mbyte": 1e6, "gbyte": 1e9, "tbyte": 1e12}[unit]
                if name.endswith("read.sum"):
                    rd = float(val) * scale
                else:
                    wr = float(val) * scale
        if rd is None or wr is None:
            return None, "profiles/r2_product_ncu.csv has no dram__bytes rows"
        return rd + wr, "profiles/r2_product_ncu.csv"
    except OSError:
        return None, "profiles/r2_product_ncu.csv missing"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2,
                    help="index into BASELINE.json configs (2 = 32^3 x 64, the metric; 1 = 16^3 x 32, the paper's Fig. 1-2 "
                         "lattice; 3 = 32^3 u=d=s; 4 = 96^3, tile-wise plan)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1 (T-parallel replicas, PAPER.md:133-137): weak = K slices per rank; strong = the K slices "
                         "of the job are divided over the ranks (K must be a multiple of N)")
    ap.add_argument("--lattice", type=int, default=0, help="override L (debugging only; invalidates the metric)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--oracle-sample-L", type=int, default=0,
                    help="sub-lattice of the CPU oracle's timed sample (default: 6 for cpu_baseline, 8 for --impl reference)")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([s.strip() for s in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 6 and r[2 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


# ------------------------------------------------------------------------------------------------
def oracle_leg(sample_L: int, cfg_index: int, steps: int, warmup: int) -> dict:
    """Time the CPU oracle (tier B, eq. 2.6 path) on a bounded sample of the workload: the same
    flavour recipe and all 52 channels on a sample_L^3 sub-lattice; its cost is per lattice site
    (blocks per x, products per q; numpy's FFT is negligible), so slices/s at L^3 = sites/s / L^3."""
    import numpy as np
    from oracle import nbs_oracle as O
    from paper_1604_07983_b200 import synth
    cfg = synth.CONFIGS[cfg_index]
    chans = O.channels52()
    V_full = cfg["L"] ** 3
    times, cpu = [], []
    for i in range(warmup + steps):
        S = synth.config_slice(cfg, i % cfg["T"], L=sample_L)
        c0 = os.times()
        t0 = time.perf_counter()
        B = O.all_blocks(S, O.sink_names(chans))
        F = O.correlator_fft(sample_L, B, chans)
        dt = time.perf_counter() - t0
        c1 = os.times()
        assert np.isfinite(F).all()
        if i >= warmup:
            times.append(dt)
            cpu.append((c1.user + c1.system) - (c0.user + c0.system))
    per_step = sum(times) / len(times)
    sites_per_s = sample_L ** 3 / per_step
    # threads the oracle actually kept busy: process CPU time / wall time of the timed samples
    cores = max(1.0, round(sum(cpu) / sum(times), 1))
    return {"value": sites_per_s / V_full, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"one step = the whole path on a periodic {sample_L}^3 sub-lattice ({sample_L ** 3} of the {V_full} sites "
                      f"of a slice; same flavour recipe, all 52 channels): {per_step:.1f} s measured per step; the oracle's "
                      f"cost is per site, so value = ({sample_L ** 3}/{V_full}) slices per step / measured seconds per step",
            "ms_per_step": per_step * 1e3, "ms_per_slice_extrapolated": per_step * 1e3 * V_full / sample_L ** 3,
            "host_cpus": os.cpu_count()}


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    from paper_1604_07983_b200 import synth
    cfg = dict(synth.CONFIGS[args.config])
    L = args.lattice or cfg["L"]
    V = L ** 3
    workload = f"BASELINE.json configs[{args.config}]: {L}^3 x {cfg['T']}, 52 channels, complex128, {cfg['name']}"
    metric = metric_name(args.config, cfg, L)

    if args.impl == "reference":
        if rank != 0:
            return
        steps, warm = max(1, min(args.steps, 3)), min(args.warmup, 1)
        leg = oracle_leg(args.oracle_sample_L or 8, args.config, steps, warm)
        line = {"impl": "reference", "metric": metric, "value": leg["value"], "unit": UNIT, "n_gpus": args.gpus,
                "steps": steps, "warmup": warm, "ms_per_step": leg["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": workload, "ms_per_slice_extrapolated": leg["ms_per_slice_extrapolated"]},
                "cpu_baseline": {k: leg[k] for k in ("value", "unit", "cores", "kind", "sample")},
                "e2e": {"value": leg["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
        print(json.dumps(line))
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1604_07983_b200 import nbs, replicas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()

    K, W = args.steps, max(args.warmup, 3)
    if args.scaling == "strong":
        if K % world:
            raise SystemExit("--scaling strong needs --steps to be a multiple of the number of ranks")
        K //= world  # slices of THIS rank; the job's total stays args.steps
    T = cfg["T"]
    npool = min(4 if L <= 32 else 2, K + W, T)
    # this rank's time slices: T-parallel replicas (t = rank, rank + world, ...)
    pool_t = replicas.rank_slices(rank, world, T, count=npool)
    host = []
    for t in pool_t:
        S = synth.config_slice(cfg, t, L=L)
        pinned = {}
        for f in "uds":
            spec = cfg["flavours"][f]
            if isinstance(spec, str):
                pinned[f] = pinned[spec]
            else:
                buf = torch.empty((V, 12, 12), dtype=torch.complex128).pin_memory()
                buf.copy_(torch.from_numpy(S[f]))
                pinned[f] = buf
        host.append(pinned)
    resident = []
    for h in host:
        d = {}
        for f in "uds":
            spec = cfg["flavours"][f]
            d[f] = d[spec] if isinstance(spec, str) else h[f].to(dev)
        resident.append(d)

    # configs[4] (96^3): the result of one slice is 188 GB, so it is produced sink pair by sink pair into one buffer
    # (include/nbs.h: channel ranges, nbs_pair_order); the library takes its tile-wise plan there
    big = 52 * 256 * V * 16 > 40e9
    ctx = nbs.Nbs(L, T, None, device=local,
                  workspace_budget_bytes=0 if not big else int(0.92 * torch.cuda.mem_get_info(dev)[0]) - 6 * 256 * V * 16)
    nch = ctx.nch
    flops = ctx.model_flops()
    tiled = ctx.tiled_info()
    ranges = ctx.pair_order() if big else [(0, nch)]
    nmax = max(hi - lo for lo, hi in ranges)
    out_dev = torch.empty((nmax, 256, V), dtype=torch.complex128, device=dev)
    stream = torch.cuda.Stream(device=dev)

    def step_resident(i):
        t = pool_t[i % npool]
        r = resident[i % npool]
        ctx.load(t, r["u"], r["d"], r["s"], stream=stream)
        for lo, hi in ranges:
            ctx.correlator(t, lo, hi, out=out_dev[:hi - lo], stream=stream)

    # ---------------- device-resident leg (value, roofline) ----------------
    for i in range(W):
        step_resident(i)
    torch.cuda.synchronize()
    # clocks are sampled from here on: the probes and the timed steps keep the GPU loaded without a gap
    sampler = ClockSampler(local)
    sampler.start()
    # measured FP64 peaks of this device, in this process (nbs_probe_fp64): ~0.3 s per mix
    probe = {name: ctx.probe_fp64(mode, 60000)["tflops"]
             for name, mode in (("dmma", 0), ("dfma", 1), ("dadd", 2), ("mix_16x16_kstep", 3), ("mix_64x4_kstep", 4))}
    torch.cuda.synchronize()
    ctx.set_timing(True)
    ctx.stage_times(reset=True)
    launches0 = ctx.kernel_launches()
    builds0 = ctx.tiled_info()["chunk_builds"]
    barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(K):
        step_resident(W + i)
    e1.record(stream)
    torch.cuda.synchronize()
    barrier()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    stage = ctx.stage_times(reset=True)
    ctx.set_timing(False)
    launches = ctx.kernel_launches() - launches0
    builds = ctx.tiled_info()["chunk_builds"] - builds0
    checksum = float(out_dev.view(torch.float64).abs().max().item())
    assert np.isfinite(checksum) and checksum > 0

    # ---------------- end-to-end leg: host buffers through the C ABI ----------------
    e2e = None
    if not args.no_e2e:
        # Time slices are pipelined over two CUDA streams (the library keeps two
        # workspace slots, t % 2): the 7 GB device-to-host copy of slice i runs on the copy engine
        # while the kernels of slice i + 1 run.  Every slice still pays its own H2D and D2H.
        nslots = ctx.num_slots()  # one stream per workspace slot; with one slot the slices serialise on one stream
        # slot 0's stream has the higher priority: when the empty pipeline starts, the kernels of the first slice run
        # ahead of those of the second instead of interleaving with them, so the first copy starts one slice earlier
        streams2 = [torch.cuda.Stream(device=dev, priority=-1), torch.cuda.Stream(device=dev, priority=0)] if nslots > 1 else [stream, stream]
        del out_dev
        outs_host = [torch.empty((nmax, 256, V), dtype=torch.complex128).pin_memory() for _ in range(2 if not big else 1)]
        out_host = outs_host[0]

        def step_e2e(i):
            t = pool_t[i % npool]
            h = host[i % npool]
            st = streams2[t % nslots]                                # one stream per workspace slot (t % nslots)
            ctx.load(t, h["u"], h["d"], h["s"], stream=st)          # H2D inside the library
            for lo, hi in ranges:                                    # D2H of F inside the library
                ctx.correlator(t, lo, hi, out=outs_host[t % len(outs_host)][:hi - lo], stream=st)
        step_e2e(0)
        step_e2e(1)
        torch.cuda.synchronize()
        barrier()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        Ke = K if not big else max(2, min(K, 2))  # exactly K steps; the pipeline starts empty: its fill (the kernels of the first slice before the first copy) is inside the timed region
        f0.record(streams2[0])
        if nslots > 1:
            streams2[1].wait_event(f0)
        for i in range(Ke):
            step_e2e(2 + i)
        if nslots > 1:
            join = torch.cuda.Event()
            join.record(streams2[1])
            streams2[0].wait_event(join)
        f1.record(streams2[0])
        torch.cuda.synchronize()
        barrier()
        ms_e2e = f0.elapsed_time(f1)
        nflav = len({id(v) for v in host[0].values()})
        e2e = {"ms": ms_e2e, "steps": Ke, "h2d": nflav * V * 144 * 16, "d2h": nch * 256 * V * 16}
        assert np.isfinite(out_host.view(torch.float64)[:1024]).all()

    # ---------------- max over ranks ----------------
    ms, ms_e2e_max = replicas.max_over_ranks([ms, e2e["ms"] if e2e else 0.0], device=dev)
    if e2e:
        e2e["ms"] = ms_e2e_max
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = replicas.aggregate_throughput(K, world, ms)
    prod_ms, prod_calls = stage["product"]
    prod_avg_s = prod_ms * 1e-3 / K  # per slice (the tile-wise plan launches the kernel up to 4 times per sink pair)
    alg_flops = flops["product"] * V  # 256 * sum_d K_d cMAC x 8 flop per q, standard count
    achieved = alg_flops / prod_avg_s / 1e12
    peak = probe["dmma"]
    traffic, traffic_src = product_dram_traffic()
    line = {
        "metric": metric, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
        "ms_per_step": ms / (K * world if args.scaling == "strong" else K), "higher_is_better": True,
        "scaling": args.scaling, "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload, "channels": nch, "lattice": [L, L, L, T],
                   "l2_policy": "inputs (%.0f MB per slice) and intermediates (%.1f GB per slice) exceed the 126 MB L2"
                                % (len({id(v) for v in host[0].values()}) * V * 144 * 16 / 1e6,
                                   ctx.workspace_bytes() / max(ctx.num_slots(), 1) / 1e9),
                   "parallelism": "replicas only (T-parallel), no collective" if world > 1 else "1 GPU",
                   "plan": ("tile-wise: %d chunk buffers, %.1f chunk builds per slice, %d channel ranges per slice"
                            % (tiled["chunk_slots"], builds / K, len(ranges))) if tiled["tiled"] else "resident",
                   "channel_sites_per_s": value * nch * V},
        "clocks": clocks,
        "gpu_launches": int(launches),
        "stages_ms_per_step": {k: v[0] / K for k, v in stage.items()},
        "roofline": {"bound": "alu", "kernel": "product (effective blocks x product, eqs. 4.2-4.3)",
                     "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                     "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                     "peak_source": "measured in this run: nbs_probe_fp64 mode 0 (register-resident DMMA.8x8x4, 16 warps per SM, "
                                    "all SMs), executed flops / CUDA-event time",
                     "peak_derived": FP64_PEAK_DERIVED_TFLOPS,
                     "fp64_probe_tflops": probe,
                     "flops_per_launch_algorithmic": alg_flops,
                     "flops_per_launch_executed": flops["product_executed"] * V,
                     "achieved_executed": flops["product_executed"] * V / prod_avg_s / 1e12,
                     "frac_executed": flops["product_executed"] * V / prod_avg_s / 1e12 / peak,
                     "kernel_ms": prod_avg_s * 1e3, "kernel_launches_per_step": prod_calls / K,
                     "note": "achieved/frac use SURVEY 8(d)'s standard count (256 x sum K_d x 8 flop per site); the kernel "
                             "evaluates about half of it (shared elementary correlators, source- and sink-swap relations), "
                             "so frac can exceed 1; achieved_executed/frac_executed count 8 flop per complex MAC actually "
                             "evaluated"},
    }
    if e2e:
        line["e2e"] = {"value": world * e2e["steps"] / (e2e["ms"] * 1e-3), "unit": UNIT,
                       "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"]}
    if world == 1 and not args.no_cpu_baseline:
        leg = oracle_leg(args.oracle_sample_L or 6, args.config, 1, 0)
        line["cpu_baseline"] = {k: leg[k] for k in ("value", "unit", "cores", "kind", "sample")}
    ctx.close()
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
