#!/usr/bin/env python
"""bench.py -- matrix elements per second on B200 through the C ABI (see the contract in DESIGN.md §Measurement).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--process P] [--precision fp64|mixed] [--nevt E]
  python bench.py --impl reference ...         # the CPU oracle on the host cores (reported baseline)

One "step" = one mg_sigma_batch over one batch of seeded RAMBO momenta of the BASELINE.json config
(helicity filter already done): momenta read -> external wavefunctions -> currents + amplitudes -> jamps ->
colour sum -> helicity sum -> me[nevt].  Rank 0 prints ONE JSON line.
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2510_05392_b200 import inputs  # noqa: E402

# DRAM bytes of the dominant kernel from the committed ncu --set full captures: profiles/dram_traffic.csv holds one row per
# capture (process, precision, events of the launch, dram__bytes_read.sum, dram__bytes_write.sum, capture file); the figure is
# scaled to the timed launch by the event count.  No row for the timed (process, precision) -> "traffic": null.
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "dram_traffic.csv")


def ncu_dram_bytes_per_event(process, precision):
    if not os.path.exists(TRAFFIC_CSV):
        return None, None
    last = None
    for line in open(TRAFFIC_CSV):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 6 and f[0] == process and f[1] == precision:
            last = ((float(f[3]) + float(f[4])) / float(f[2]), ", ".join(f[5:]))
    return last if last else (None, None)

HEADLINE = "gg_ttxggg"      # BASELINE.json configs[4]: the process the north star's roofline targets are set on
METRIC = "matrix elements/sec"


def read_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        return json.load(open(path)), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region"""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_rate(process, nevt_sample, seed=1):
    """the oracle as it stands on the host cores: (MEs/s, cores, seconds)"""
    import oracle
    p = inputs.momenta(process, nevt_sample, seed=seed)
    oracle.matrix_elements(process, p[:1], inputs.PARAMS)          # builds the colour matrix, loads the library
    t = time.perf_counter()
    oracle.matrix_elements(process, p, inputs.PARAMS)
    dt = time.perf_counter() - t
    return nevt_sample / dt, os.cpu_count(), dt


# sized for about 10-30 s of oracle time on the 16 host cores of the GPU box (854 MEs/s measured for gg_ttxggg)
ORACLE_SAMPLE = {"epem_mupmum": 16384, "gg_ttx": 65536, "gg_ttxg": 65536, "gg_ttxgg": 32768, "gg_ttxggg": 12288,
                 "gg_ttxgggg": 256}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    process = args.process or HEADLINE
    ns = args.nevt or ORACLE_SAMPLE[process]
    import oracle
    p = inputs.momenta(process, ns)
    oracle.matrix_elements(process, p[:1], inputs.PARAMS)
    for _ in range(min(args.warmup, 1)):
        oracle.matrix_elements(process, p[: max(1, ns // 8)], inputs.PARAMS)
    t = time.perf_counter()
    for _ in range(args.steps):
        oracle.matrix_elements(process, p, inputs.PARAMS)
    dt = time.perf_counter() - t
    val = ns * args.steps / dt
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": "MEs/s", "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"{process}, {inputs.PROCESSES[process]['nevt']} events/batch (BASELINE.json config), "
                                  f"each step a bounded sample of {ns} events", "process": process},
           "cpu_baseline": {"value": val, "unit": "MEs/s", "cores": os.cpu_count(), "kind": "oracle",
                            "sample": f"{ns} seeded RAMBO events of {process} per step"},
           "e2e": {"value": val, "unit": "MEs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


def shard_first_event(rank, nevt_per_rank):
    """weak scaling (events are independent): rank r evaluates the contiguous event
    range [r * nevt, (r + 1) * nevt) of the seeded stream; no collective on the data path"""
    return rank * nevt_per_rank


def reduce_max_ms(ms, dist, device="cpu"):
    """device time of the slowest rank (the one all-reduce of the run: a scalar, for the timing only)"""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def masks_agree(mask, dist, device="cpu"):
    """the helicity mask is a property of the process: every rank derives it from its own probe events;
    True iff all ranks found the same one"""
    if dist is None:
        return True
    import torch
    m = torch.as_tensor(np.asarray(mask, dtype=np.int32), device=device)
    lo, hi = m.clone(), m.clone()
    dist.all_reduce(lo, op=dist.ReduceOp.MIN)
    dist.all_reduce(hi, op=dist.ReduceOp.MAX)
    return bool((lo == hi).all().item())


def spawn_ranks(argv, gpus):
    """`python bench.py --gpus N` without a launcher: start N ranks of this script under torch.distributed.run (one process
    per GPU, rendezvous on 127.0.0.1) and hand their output through"""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
    return subprocess.call(cmd)


def time_process(torch, B, process, precision, nevt, steps, warmup, rank, world, flush, opts=None, dist=None, stages=True):
    """returns dict with device-timed throughput of `steps` batches (stages: also the per-stage CUDA-event times)"""
    dev = torch.cuda.current_device()
    proc = B.Process(process, precision, dev)
    for k, v in (opts or {}).items():
        proc.set_option(k, v)
    proc.set_option("timing", 1 if stages else 0)
    mom_h = inputs.momenta(process, nevt, seed=1, first_event=shard_first_event(rank, nevt))
    d_mom = torch.from_numpy(mom_h).to(f"cuda:{dev}")
    mask = proc.helicity_filter(d_mom)
    if not masks_agree(mask, dist, f"cuda:{dev}"):
        raise SystemExit("ranks disagree on the good-helicity mask")
    d_me = torch.empty(nevt, dtype=torch.float64, device=f"cuda:{dev}")
    for _ in range(warmup):
        proc.sigma_batch(d_mom, d_me)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
        torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    stage = np.zeros(3)
    for i in range(steps):
        if flush is not None:
            flush.fill_(i)                      # > L2 (126 MB): evicts momenta / tables between timed steps
        ev[i][0].record()
        proc.sigma_batch(d_mom, d_me)
        ev[i][1].record()
        ev[i][1].synchronize()
        if stages:
            stage += np.array(proc.last_stage_ms())
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    ms = reduce_max_ms(ms, dist, f"cuda:{dev}")
    if dist is not None:
        dist.barrier()
    launches_per_step = proc.last_launch_count()
    res = {"proc": proc, "ms_total": ms, "ms_per_step": ms / steps, "value": world * nevt * steps / (ms * 1e-3),
           "stage_ms": (stage / steps).tolist(), "ngood": int(mask.sum()), "launches": launches_per_step * steps,
           "d_mom": d_mom, "d_me": d_me, "mom_h": mom_h}
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--process", default=None)
    ap.add_argument("--precision", default="fp64")
    ap.add_argument("--nevt", type=int, default=None)
    ap.add_argument("--color-sum", type=int, default=None, help="0 fused ALU, 1 tensor-core kernel")
    ap.add_argument("--schedule", type=int, default=0, help="0 helicity in the grid, 1 helicity streams")
    ap.add_argument("--diagrams", type=int, default=None, help="0 thread per (event, helicity), 1 helicity-shared CTA per event")
    ap.add_argument("--chunk-mib", type=int, default=None, help="jamps buffer size inside the workspace")
    ap.add_argument("--no-extras", action="store_true", help="skip per-process table, e2e and cpu baseline")
    ap.add_argument("--ramp", action="store_true",
                    help="also report MEs/s against the number of events per batch, 32 ... full (the paper's small-grid curves, PAPER.md:174, 225)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl != "reference" else args.warmup
    if args.gpus < 1:
        raise SystemExit("--gpus must be >= 1")
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        raise SystemExit(spawn_ranks(sys.argv[1:], args.gpus))
    if int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={os.environ.get('WORLD_SIZE')}: launch one rank per GPU")
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2510_05392_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (B200); there is no CPU fallback. Use --impl reference for the oracle.")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")             # rank/transport lines (NVLink, NVLS) for whoever reads the log
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")  # stdout carries the JSON line only
        import torch.distributed as dist_
        dist_.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
        dist = dist_

    process = args.process or HEADLINE
    nevt = args.nevt or inputs.PROCESSES[process]["nevt"]
    opts = {}
    if args.diagrams is not None:
        opts["diagrams"] = args.diagrams           # before "schedule": streams exist for the thread kernel only
    if args.schedule:
        opts["schedule"] = args.schedule
    if args.color_sum is not None:
        opts["color_sum"] = args.color_sum
    if args.chunk_mib is not None:
        opts["jamp_chunk_mib"] = args.chunk_mib
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=f"cuda:{local}")

    peaks, peak_src = read_peaks()
    fp64_peak = B.measure_peak(0, local)        # TFLOP/s, burst, this GPU, measured now

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    r = time_process(torch, B, process, args.precision, nevt, args.steps, args.warmup, rank, world, flush, opts, dist)
    clocks = sampler.stop() if rank == 0 else None
    proc = r["proc"]

    # roofline of the dominant kernel (the diagram kernel): plain FP64 ALU bound
    diag_ms = r["stage_ms"][0]
    shared = proc.get_option("diagrams") == 1
    alg_flop = proc.diagram_flops * nevt * r["ngood"]
    if not shared and proc.get_option("color_sum") == 0:
        alg_flop += (2.0 * proc.ncolor * (proc.ncolor + 1) + 4.0 * proc.ncolor) * nevt * r["ngood"]   # fused triangular colour sum
    achieved = alg_flop / (diag_ms * 1e-3) * 1e-12
    dram_per_event, dram_src = ncu_dram_bytes_per_event(process, args.precision) if shared else (None, None)
    roofline = {"bound": "alu", "kernel": ("hsg_diagrams_kernel" if process == "gg_ttxgggg" else "hs_diagrams_kernel") if shared else "diagrams_kernel", "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s",
                "frac": achieved / fp64_peak if fp64_peak else None,
                "traffic": dram_per_event * nevt if dram_per_event else None,
                "traffic_source": (f"ncu --set full capture {dram_src} (profiles/dram_traffic.csv), scaled to this launch by the "
                                   "event count") if dram_per_event else None,
                "peak_source": "fp64 FMA probe kernel measured in this run (mg_measure_peak, burst); "
                               "MEASURED_PEAKS.json holds no fp64 figure",
                "flop_per_event_helicity": proc.diagram_flops, "kernel_ms": diag_ms,
                "hbm_peak_gbs": peaks.get("hbm_gbs"), "hbm_peak_source": peak_src}

    # second kernel of the step, the colour sum: FP64 tensor bound (DMMA, issued flop of the triangular contraction) in fp64,
    # HBM bound (it reads the jamps once) in mixed precision
    cs_roofline = None
    cs_ms = r["stage_ms"][1]
    if shared and cs_ms > 0:
        rows = nevt * r["ngood"]
        nc = proc.ncolor
        if args.precision in ("fp64", "d"):
            nt = (nc + 7) // 8
            pairs = sum(ks // 2 + 1 for ks in range(2 * nt))                   # (k-step, n-tile) pairs on or below the diagonal
            flop = rows / 8 * pairs * 2 * 512.0                                # x 2 parts, 512 flop per m8n8k4
            dmma_peak = B.measure_peak(2, local)
            ach = flop / (cs_ms * 1e-3) * 1e-12
            cs_roofline = {"bound": "tensor", "kernel": "color_sum_big_kernel" if nc > 128 else "color_sum_dmma2_kernel", "achieved": ach, "peak": dmma_peak, "unit": "TFLOP/s",
                           "frac": ach / dmma_peak, "kernel_ms": cs_ms, "flop_counted": "issued DMMA (triangular k-step x n-tile pairs)",
                           "peak_source": "mma.sync.m8n8k4.f64 probe measured in this run (mg_measure_peak kind 2)"}
        elif nc > 128:
            # 720 colours: compute bound on the TF32 tensor path; issued MMA flop = per 128-row tile and part, per (block of
            # 240 columns, 24-colour chunk on or below the block's diagonal) two products (L_hi, L_lo) of 128 x width x 24
            widths = [min(240, (24 * (c - 10 * b + 1) + 15) // 16 * 16) for b in range(3) for c in range(10 * b, 30)]
            flop = rows / 128 * 2 * sum(2 * 2.0 * 128 * w * 24 for w in widths)
            tf32_peak = B.measure_peak(3, local)
            ach = flop / (cs_ms * 1e-3) * 1e-12
            cs_roofline = {"bound": "tensor", "kernel": "color_sum_tf32_big_kernel", "achieved": ach, "peak": tf32_peak, "unit": "TFLOP/s",
                           "frac": ach / tf32_peak if tf32_peak else None, "kernel_ms": cs_ms,
                           "flop_counted": "issued tcgen05.mma kind::tf32 (J Lhi + J Llo, triangular in 24-colour chunks)",
                           "peak_source": "tcgen05 kind::tf32 probe measured in this run (mg_measure_peak kind 3)"}
        elif not proc.get_option("hs_color_alu"):
            nbytes = rows * nc * 2 * 4.0
            ach = nbytes / (cs_ms * 1e-3) * 1e-9
            cs_roofline = {"bound": "hbm", "kernel": "color_sum_tf32_kernel", "achieved": ach, "peak": peaks.get("hbm_gbs"), "unit": "GB/s",
                           "frac": ach / peaks["hbm_gbs"] if peaks.get("hbm_gbs") else None, "kernel_ms": cs_ms,
                           "bytes_counted": "the fp32 jamps, read once", "peak_source": peak_src}

    out = {"metric": METRIC, "value": r["value"], "unit": "MEs/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64" if args.precision in ("fp64", "d") else ("f64+f32" if args.precision in ("mixed", "m") else "f32"),
           "data": "synthetic",
           "config": {"workload": f"{process}: {nevt} events/batch/GPU, flat RAMBO sqrt(s)=1500 GeV seed 1 ("
                                              + ("SURVEY.md 8(f) row 3; batch size chosen here)" if process == "gg_ttxgggg" else "BASELINE.json config)"),
                      "process": process, "precision": args.precision, "nevt_per_gpu": nevt, "good_helicities": r["ngood"],
                      "diagrams": "helicity-shared (CTA = event, thread = helicity)" if shared else "thread = (event, helicity)",
                      "schedule": "helicity streams" if args.schedule else ("helicity = thread index" if shared else "helicity = grid.y"),
                      "color_sum": (("DMMA (mma.sync f64), Cholesky form" if args.precision in ("fp64", "d") else
                                     ("ALU kernel" if proc.get_option("hs_color_alu") and process != "gg_ttxgggg" else "tcgen05 kind::tf32, split, Cholesky form"))
                                    if shared else ("tensor" if proc.get_option("color_sum") == 1 else "fused ALU")),
                      "jamp_chunk_mib": proc.get_option("jamp_chunk_mib"),
                      "l2": "256 MiB device memset between timed steps (outside the per-step event pairs)"},
           "gpu_launches": r["launches"], "stage_ms": {"diagrams": r["stage_ms"][0], "color_sum": r["stage_ms"][1],
                                                         "helicity_sum": r["stage_ms"][2]},
           "roofline": roofline, "roofline_color_sum": cs_roofline, "clocks": clocks}

    if rank == 0 and (args.ramp or (world == 1 and not args.no_extras)):          # (one-GPU study: not in multi-rank runs)
        # the paper's small-grid curves (MEs/s against events per batch): plain launches, and the
        # same launch sequence replayed as a CUDA graph (option "graph")
        sizes, n = [], 32
        while n < nevt:
            sizes.append(n)
            n *= 2 if 512 <= n < 2048 else 4          # 32, 128, 512, 1024, 2048, 8192, ...: finer where the curves bend
        ramp = {"plain": {}, "graph": {}}
        for n in sizes:
            for mode in ("plain", "graph"):
                q = time_process(torch, B, process, args.precision, n, 10, 3, 0, 1, None, dict(opts, graph=1 if mode == "graph" else 0),
                                 stages=False)
                ramp[mode][str(n)] = q["value"]
                q["proc"].close()
        ramp["plain"][str(nevt)] = r["value"]
        peak = max(ramp["plain"].values())
        ramp["events_for_90pct_of_peak"] = min(int(k) for k, v in ramp["plain"].items() if v >= 0.9 * peak)
        out["ramp_MEs_per_s"] = ramp
    if rank == 0 and not args.no_extras:
        # end to end through the host-buffer entry point: pinned host momenta -> device -> me -> host, every step
        hm = torch.from_numpy(r["mom_h"]).pin_memory()
        he = torch.empty(nevt, dtype=torch.float64).pin_memory()
        proc.sigma_batch_host(hm.numpy(), he.numpy())
        t0 = time.perf_counter()
        for _ in range(args.steps):
            proc.sigma_batch_host(hm.numpy(), he.numpy())
        dt = time.perf_counter() - t0
        out["e2e"] = {"value": nevt * args.steps / dt, "unit": "MEs/s", "h2d_bytes_per_step": int(hm.numel() * 8),
                      "d2h_bytes_per_step": int(he.numel() * 8), "n_gpus_measured": 1}
        if world == 1:
            ns = ORACLE_SAMPLE[process]
            val, cores, secs = oracle_rate(process, ns)
            out["cpu_baseline"] = {"value": val, "unit": "MEs/s", "cores": cores, "kind": "oracle",
                                   "sample": f"first {ns} events of the same batch, {secs:.1f} s"}
            per = {}
            for pname in inputs.PROCESSES:
                for prec in ("fp64", "mixed"):
                    if pname == process and prec == args.precision:
                        per[f"{pname}/{prec}"] = {"MEs_per_s": r["value"], "ms_per_batch": r["ms_per_step"]}
                        continue
                    try:
                        q = time_process(torch, B, pname, prec, inputs.PROCESSES[pname]["nevt"], 3, 3, 0, 1, flush, opts)
                        per[f"{pname}/{prec}"] = {"MEs_per_s": q["value"], "ms_per_batch": q["ms_per_step"],
                                                  "stage_ms": {"diagrams": q["stage_ms"][0], "color_sum": q["stage_ms"][1]},
                                                  "diagram_tflops": q["proc"].diagram_flops * inputs.PROCESSES[pname]["nevt"]
                                                  * q["ngood"] / (q["stage_ms"][0] * 1e-3) * 1e-12}
                        q["proc"].close()
                    except Exception as ex:  # keep the headline line even if a side measurement fails
                        per[f"{pname}/{prec}"] = {"error": str(ex)[:200]}
            out["per_process"] = per
    elif rank == 0:
        out["e2e"] = None
    if rank == 0:
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
