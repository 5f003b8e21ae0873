#!/usr/bin/env python
"""bench.py — throughput of the B200-native closed-shell (T) energy path.

    python bench.py --gpus N --steps K --warmup W [--config 5] [--window 10] [--full]
    python bench.py --impl reference ...        # the CPU oracle on the same workload (bounded sample)

A "step" is one pass of the whole hot path (DF slab former -> W builder -> fused V -> energy
contraction -> fixed-order sums) over one batch of occupied-triplet
blocks of the workload.  Default workload: BASELINE.json configs[4] (nocc=100 nvir=380 naux=1680,
the configuration the >= 60 % target is quoted on), one triplet block per GPU = all triplets
i<=j<=k inside an occupied window of `--window` orbitals (rank r takes window [r*w, (r+1)*w)):
weak scaling, no data-path collective (triplets are independent; the only exchange is one scalar
sum).  `--full` evaluates the complete E(T) of the config in one step instead.

value = algorithmic W-builder FP64 flops of the step (bqc_t_flops: #triplets * 12 v^3 (v+o); slab
forming and the energy contraction are NOT credited) / max-over-ranks device time, in TFLOP/s.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

METRIC = "(T) FP64 TFLOP/s (W-builder algorithmic flops / whole-path time)"
UNIT = "TFLOP/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5,
                    help="BASELINE.json configs[n-1], n = 1..5; 6-8 = cc-pVTZ/QZ-shaped inputs (SURVEY NEXT-2); "
                         "9 = the paper's largest CCSD(T) size, 1 380 orbitals (use --schedule abc)")
    ap.add_argument("--schedule", default="ijk", choices=["ijk", "abc"],
                    help="ijk: occupied triplets outside, v^3 inside (default); abc: the paper's loop order, "
                         "virtual triples outside, o^3 inside (BQC_T_FLAG_ABC_DRIVEN)")
    ap.add_argument("--abc-window", type=int, default=38, help="virtual orbitals per triple block (--schedule abc)")
    ap.add_argument("--window", type=int, default=10, help="occupied orbitals per triplet block (per GPU)")
    ap.add_argument("--full", action="store_true", help="whole E(T) of the config in one step")
    ap.add_argument("--occ-block", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=1)
    ap.add_argument("--peak-seconds", type=float, default=2.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-profile", action="store_true",
                    help="time the calls without BQC_T_FLAG_PROFILE (the library then replays a CUDA graph for short "
                         "schedules); the per-kernel split comes from one extra profiled call after the timed region")
    ap.add_argument("--cpu-triplets", type=int, default=3, help="triplets the oracle evaluates (cpu_baseline)")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="torch.distributed backend of the N>1 plumbing (barrier, max-over-ranks, the scalar exchange)")
    ap.add_argument("--share-gpu", action="store_true",
                    help="TEST ONLY: every rank uses cuda:0 (implies --backend gloo); exercises the N>1 code path on a "
                         "1-GPU box, its timings mean nothing and the line says so")
    ap.add_argument("--shard-sweep", type=int, default=0, metavar="N",
                    help="ONE GPU: evaluate the N block-triple shards of a full E(T) one after another and report "
                         "each shard's time, flops and slab blocks formed, plus the strong-scaling efficiency they "
                         "imply (T_1 / (N max_r T_r)); a projection from measured per-shard times, not an N-GPU run")
    ap.add_argument("--path", default="t", choices=["t", "mp2"],
                    help="t: the (T) energy (the headline); mp2: the DF-MP2 energy of PAPER.md Eq. (1) (SURVEY NEXT-4)")
    return ap.parse_args()


def workload_name(cfg, c, lo, hi, full, ntrip, abc=False):
    base = f"config{cfg} nocc={c['nocc']} nvir={c['nvir']} naux={c['naux']} (synthetic water-cluster shape)"
    if abc:
        if full:
            return base + f", abc-driven schedule, full E(T): all {ntrip} virtual triples a<=b<=c"
        return base + f", abc-driven schedule, one triple block per GPU: virtual window [{lo},{hi}) = {ntrip} triples"
    if full:
        return base + f", full E(T): all {ntrip} triplets i<=j<=k"
    return base + f", one triplet block per GPU: occupied window [{lo},{hi}) = {ntrip} triplets"


# ----------------------------------------------------------------------------- one process per GPU
def ensure_ranks(args):
    """`python bench.py --gpus N` (no torchrun) starts the N ranks itself: it re-executes under
    `python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1`, rank r bound to
    GPU r.  Under torchrun (WORLD_SIZE set) it only checks that WORLD_SIZE matches --gpus."""
    if args.gpus < 1:
        raise SystemExit(f"bench.py: --gpus {args.gpus} must be >= 1")
    if args.share_gpu:
        args.backend = "gloo"
    world_env = os.environ.get("WORLD_SIZE")
    if args.impl == "reference":
        return                                  # the oracle arm runs on rank 0's host cores only
    if world_env is not None:
        if int(world_env) != args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world_env}; launch with "
                             f"--nproc-per-node {args.gpus} or drop torchrun and let bench.py start the ranks")
        return
    if args.gpus == 1:
        return
    if args.path == "mp2":
        raise SystemExit("bench.py --path mp2 is a single-GPU measurement (--gpus 1)")
    ndev = torch.cuda.device_count()
    if ndev < args.gpus and not args.share_gpu:
        raise SystemExit(f"bench.py --gpus {args.gpus}: only {ndev} CUDA device(s) visible; one rank per GPU is "
                         "required (no rank shares a GPU in a measurement)")
    import socket
    sock = socket.socket()
    sock.bind(("127.0.0.1", 0))
    port = sock.getsockname()[1]
    sock.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    sys.stdout.flush()
    os.execv(sys.executable, cmd)


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.gpu)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
            # nvidia-smi's own start-up briefly holds driver locks: let it reach its first sample before the
            # timed region begins, so that short steps are not perturbed by it
            t0 = time.perf_counter()
            while not self.lines and time.perf_counter() - t0 < 3.0:
                time.sleep(0.05)
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()        # the exact PID we started
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for n, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------- reference arm (oracle)
def oracle_sample(inp, triplet, abc=False):
    """Time the oracle as it stands on one triplet (one virtual triple for the abc-driven schedule) of the
    workload; returns (seconds, e_ijk)."""
    from oracle import t_oracle as orc      # bench.py's cpu_baseline / --impl reference leg only
    t0 = time.perf_counter()
    e = orc.e_virtual_triple(inp, *triplet) if abc else orc.e_triplet(inp, *triplet)
    return time.perf_counter() - t0, e


def cpu_threads():
    try:
        from threadpoolctl import threadpool_info
        n = max((p.get("num_threads", 1) for p in threadpool_info()), default=1)
        return int(n)
    except Exception:
        return os.cpu_count() or 1


def run_reference(args, rank, world):
    if rank != 0:
        return
    from bqc_inputs import CONFIGS, make_config
    c = CONFIGS[args.config]
    o, v = c["nocc"], c["nvir"]
    inp = make_config(args.config)
    lo, hi = (0, o) if args.full else (0, min(args.window, o))
    trip = (lo, (lo + hi - 1) // 2, hi - 1)
    flops = 12.0 * v ** 3 * (v + o)
    for _ in range(min(args.warmup, 1)):
        oracle_sample(inp, trip)
    times = []
    for _ in range(args.steps):
        dt, _e = oracle_sample(inp, trip)
        times.append(dt)
    dt = float(np.mean(times))
    val = flops / dt * 1e-12
    ntrip = (hi - lo) * (hi - lo + 1) * (hi - lo + 2) // 6 - (hi - lo)      # i=j=k contributes exactly 0: not counted
    sample = (f"one triplet {trip} of the workload per step (12 v^3 (v+o) = {flops:.3e} flops; our arm's step is all "
              f"{ntrip} of them, the TFLOP/s normalisation makes the two comparable), NumPy/OpenBLAS oracle as it stands")
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_name(args.config, c, lo, hi, args.full, ntrip), "sample": sample},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def pipe_peak_tflops(gpu=0):
    """SMs x maximum SM clock x 128 FP64 flop/clk: the DMMA pipe's full rate (the floor of the roofline denominator)."""
    props = torch.cuda.get_device_properties(gpu)
    return props.multi_processor_count * getattr(props, "clock_rate", 0) * 1e3 * 128 * 1e-12


# ----------------------------------------------------------------------------- DF-MP2
def run_mp2(args):
    """One step = one whole E_MP2 evaluation of the config (single GPU).  value = algorithmic (ov|ov) flops
    o(o+1)/2 * 2 v^2 X / device time."""
    import paper_2502_17963_b200 as bqc
    from bqc_inputs import CONFIGS, make_config
    torch.cuda.set_device(0)
    c = CONFIGS[args.config]
    o, v, X = c["nocc"], c["nvir"], c["naux"]
    inp = make_config(args.config)
    host = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (inp.eps_occ, inp.eps_vir, inp.B_ov)]
    dev = [t.cuda() for t in host]
    opts = bqc.make_mp2_opts(occ_block=args.occ_block, flags=bqc.BQC_T_FLAG_PROFILE)
    mp2_ws = torch.empty(bqc.bqc_mp2_workspace_bytes(o, v, X, opts), dtype=torch.uint8, device="cuda")
    opts = bqc.make_mp2_opts(occ_block=args.occ_block, flags=bqc.BQC_T_FLAG_PROFILE, workspace=mp2_ws)
    peak = max(bqc.bqc_fp64_peak_tflops(0, args.peak_seconds), pipe_peak_tflops(0))
    e_pair = torch.zeros((o, o), dtype=torch.float64, device="cuda")
    for _ in range(args.warmup):
        e_val = bqc.bqc_mp2_energy_ex(o, v, X, *dev, opts=opts, e_pair=e_pair)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = 0
    ev0.record()
    for _ in range(args.steps):
        e_val = bqc.bqc_mp2_energy_ex(o, v, X, *dev, opts=opts, e_pair=e_pair)
        prof = bqc.bqc_mp2_last_profile()
        launches += int(prof["kernel_launches"])
    ev1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1) / max(args.steps, 1)
    flops = bqc.bqc_mp2_flops(o, v, X)
    t0 = time.perf_counter()
    for _ in range(max(args.e2e_steps, 1)):
        e_host, h2d, d2h = bqc.bqc_mp2_energy_host(o, v, X, *host)
    e2e_ms = (time.perf_counter() - t0) * 1e3 / max(args.e2e_steps, 1)
    assert e_host == e_val
    gemm_tf = flops / (prof["gemm_ms"] * 1e-3) * 1e-12
    out = {"metric": "DF-MP2 FP64 TFLOP/s ((ov|ov) algorithmic flops / whole-path time)", "value": flops / (ms * 1e-3) * 1e-12,
           "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"DF-MP2 energy, config{args.config} nocc={o} nvir={v} naux={X}, all {o * (o + 1) // 2} pairs i<=j",
                      "occ_block": bqc.bqc_mp2_plan_occ_block(o, v, X, opts)},
           "e_mp2_hartree": e_val, "fp64_tensor_peak_tflops_measured": peak,
           "kernel_ms_per_step": {"ovov_gemm": prof["gemm_ms"], "pair_energy": prof["energy_ms"], "call_total": prof["total_ms"]},
           "roofline": {"bound": "tensor", "kernel": "gemm_nt_kernel ((ov|ov) former)", "achieved": gemm_tf, "peak": peak,
                        "unit": UNIT, "frac": gemm_tf / peak, "traffic": None},
           "clocks": clocks,
           "e2e": {"value": flops / (e2e_ms * 1e-3) * 1e-12, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                   "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms},
           "gpu_launches": launches}
    if not args.no_cpu_baseline:
        from oracle import mp2_oracle as orc_mp2        # bench.py's cpu_baseline leg only
        npairs = min(o * o, 64)
        t0 = time.perf_counter()
        worst = 0.0
        e_gpu = e_pair.cpu().numpy()
        for n in range(npairs):
            i, j = n % o, (n * 7) % o
            ref = orc_mp2.pair_energy(inp, i, j)
            worst = max(worst, abs(e_gpu[i, j] - ref) / (1e-10 * abs(ref) + 1e-12 * abs(e_val) / (o * o)))
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": npairs * 2.0 * v * v * X / dt * 1e-12, "unit": UNIT, "cores": cpu_threads(),
                               "kind": "oracle", "sample": f"{npairs} pairs of the workload in {dt:.2f} s, NumPy oracle as it stands",
                               "gpu_vs_oracle_worst_err_over_tol": worst}
        assert worst <= 1.0
    print(json.dumps(out), flush=True)


# ----------------------------------------------------------------------------- per-shard times on one GPU
def run_shard_sweep(args):
    """The multi-GPU path has no data-path collective: rank r's time is the time of shard r.  This mode measures
    every shard of an N-way block-triple deal on ONE GPU, one after another (no two shards run at once), and
    reports what N GPUs would need: max over shards (+ one 8-byte all-gather).  It is labelled a projection."""
    import paper_2502_17963_b200 as bqc
    from bqc_inputs import CONFIGS, make_config
    torch.cuda.set_device(0)
    c = CONFIGS[args.config]
    o, v, X = c["nocc"], c["nvir"], c["naux"]
    n = args.shard_sweep
    inp = make_config(args.config)
    dev = [torch.from_numpy(a).cuda() for a in inp.arrays()]
    flags = bqc.BQC_T_FLAG_PROFILE | bqc.BQC_T_FLAG_SHARD_BLOCKS | (bqc.BQC_T_FLAG_ABC_DRIVEN if args.schedule == "abc" else 0)
    peak = max(bqc.bqc_fp64_peak_tflops(0, args.peak_seconds), pipe_peak_tflops(0))
    shards, partial = [], []
    for r in range(n):
        opts = bqc.make_opts(occ_block=args.occ_block, shard_rank=r, shard_count=n, flags=flags)
        ws = torch.empty(bqc.bqc_t_workspace_bytes(o, v, X, opts), dtype=torch.uint8, device="cuda")
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        ev0.record()
        e = bqc.bqc_t_energy_ex(o, v, X, *dev, opts=opts, workspace=ws)
        ev1.record()
        torch.cuda.synchronize()
        prof = bqc.bqc_t_last_profile()
        shards.append({"rank": r, "ms": ev0.elapsed_time(ev1), "flops": bqc.bqc_t_flops(o, v, opts),
                       "slab_blocks_formed": int(prof["form_blocks"]), "w_builder_ms": prof["gemm_ms"],
                       "former_ms": prof["form_ms"], "occ_block": bqc.bqc_t_plan_occ_block(o, v, X, opts)})
        partial.append(e)
        del ws
    e_total = bqc.bqc_sum_in_order(torch.tensor(partial, dtype=torch.float64))
    flops = sum(s["flops"] for s in shards)
    tmax, tsum = max(s["ms"] for s in shards), sum(s["ms"] for s in shards)
    out = {"metric": "projected " + METRIC, "value": flops / (tmax * 1e-3) * 1e-12, "unit": UNIT, "n_gpus": 1,
           "projected_for_gpus": n, "steps": 1, "warmup": 0, "ms_per_step": tmax, "higher_is_better": True,
           "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"config{args.config} nocc={o} nvir={v} naux={X}, full E(T) dealt over {n} shards by whole "
                                  "block triples; shards timed one after another on ONE GPU",
                      "note": "projection: max over per-shard times (the path's only exchange is one scalar per rank); "
                              "not a multi-GPU measurement"},
           "fp64_tensor_peak_tflops_measured": peak, "e_t_hartree": e_total, "shards": shards,
           "sum_of_shard_ms": tsum, "max_shard_ms": tmax,
           "projected_efficiency_vs_sum": tsum / (n * tmax),
           "load_imbalance_max_over_mean_flops": max(s["flops"] for s in shards) / (flops / n)}
    print(json.dumps(out), flush=True)


# ----------------------------------------------------------------------------- our arm
def ncu_traffic(config, schedule):
    """DRAM bytes per W-builder launch from the committed `ncu --set full` capture (profiles/r2_traffic.csv:
    config,schedule,kernel,src_sha,dram_read_bytes,dram_write_bytes,capture).  Returned only when the capture
    was made from the sources this build was compiled from; otherwise (None, reason)."""
    import csv
    import hashlib
    path = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    if not os.path.exists(path):
        return None, "no committed ncu capture (profiles/r2_traffic.csv absent); not measured in this run"
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2502_17963_b200", "csrc")
    for f in sorted(os.listdir(csrc)):
        with open(os.path.join(csrc, f), "rb") as fh:
            h.update(fh.read())
    sha = h.hexdigest()[:12]
    with open(path) as fh:
        for row in csv.DictReader(fh):
            if int(row["config"]) == config and row["schedule"] == schedule and row["kernel"] == "w_builder":
                if row["src_sha"] != sha:
                    return None, (f"profiles/r2_traffic.csv holds a capture of sources {row['src_sha']}, this build is "
                                  f"{sha}; not measured in this run")
                return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]), (
                    f"ncu --set full dram__bytes_read.sum + dram__bytes_write.sum per launch, {row['capture']} "
                    f"(sources {sha}); a committed capture, not measured in this run")
    return None, f"no ncu capture of config {config} / schedule {schedule}; not measured in this run"


def main():
    args = parse()
    ensure_ranks(args)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch.distributed as dist
    import paper_2502_17963_b200 as bqc
    from bqc_inputs import CONFIGS, make_config

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA library is the only implementation")
    if args.path == "mp2":
        if rank == 0:
            run_mp2(args)
        return
    if args.shard_sweep > 0:
        if rank == 0:
            run_shard_sweep(args)
        return
    gpu = 0 if args.share_gpu else local_rank
    if gpu >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} needs cuda:{gpu} but only {torch.cuda.device_count()} device(s) are visible")
    torch.cuda.set_device(gpu)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        if args.backend == "nccl":
            # NCCL's init lines (ranks, transports, NVLS) go to stderr so that stdout stays one JSON line
            os.environ.setdefault("NCCL_DEBUG", "INFO")
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
            os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
            dist.init_process_group("nccl", device_id=torch.device("cuda", gpu))
        else:
            dist.init_process_group("gloo")

    c = CONFIGS[args.config]
    o, v, X = c["nocc"], c["nvir"], c["naux"]
    abc = args.schedule == "abc"
    nidx = v if abc else o                  # the index the outer loop (window, blocks, shards) runs over
    sched_flags = bqc.BQC_T_FLAG_PROFILE | (bqc.BQC_T_FLAG_ABC_DRIVEN if abc else 0)
    w = nidx if args.full else min(args.abc_window if abc else args.window, nidx)
    nblocks = max(1, nidx // w)
    lo = 0 if args.full else (rank % nblocks) * w
    hi = nidx if args.full else lo + w
    strong = args.full and world > 1        # one E(T) dealt over the ranks by whole block triples
    if strong:
        opts = bqc.make_opts(occ_block=args.occ_block, shard_rank=rank, shard_count=world,
                             flags=sched_flags | bqc.BQC_T_FLAG_SHARD_BLOCKS)
    else:
        opts = bqc.make_opts(occ_block=args.occ_block, occ_lo=lo, occ_hi=hi, flags=sched_flags)
    flops_rank = bqc.bqc_t_flops(o, v, opts)
    f1 = 12.0 * o ** 3 * (v + o) if abc else 12.0 * v ** 3 * (v + o)      # flops of one unit of the outer loop
    ntrip = int(round(flops_rank / f1))

    t0 = time.perf_counter()
    inp = make_config(args.config)
    gen_s = time.perf_counter() - t0
    host = [torch.from_numpy(a) for a in inp.arrays()]
    pinned = False
    if inp.nbytes() < 48e9:                             # a pinned second copy of 117 GB (config 9) does not fit the host
        try:
            host = [t.pin_memory() for t in host]      # e2e copies come from pinned memory
            pinned = True
        except RuntimeError:
            pass
    dev = [t.cuda(non_blocking=True) for t in host]
    torch.cuda.synchronize()
    ws = torch.empty(bqc.bqc_t_workspace_bytes(o, v, X, opts), dtype=torch.uint8, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # FP64 tensor-core peak measured in this run: the roofline denominator
    peak_dmma = bqc.bqc_fp64_peak_tflops(0, args.peak_seconds)

    e_trip = torch.zeros(bqc.bqc_t_num_triplets(nidx), dtype=torch.float64, device="cuda")

    topts = opts
    if args.no_profile:
        topts = bqc.make_opts(occ_block=opts.occ_block, occ_lo=opts.occ_lo, occ_hi=opts.occ_hi,
                              shard_rank=opts.shard_rank, shard_count=opts.shard_count,
                              flags=opts.flags & ~bqc.BQC_T_FLAG_PROFILE)

    def step():
        return bqc.bqc_t_energy_ex(o, v, X, *dev, opts=topts, workspace=ws, e_triplet=e_trip)

    for _ in range(args.warmup):
        e_val = step()
    barrier()
    sampler = ClockSampler(gpu)
    sampler.start()
    launches = 0
    prof = None
    # Inputs larger than L2 need no flush (config 2 and up: GBs of F per launch).  A working set that fits the
    # 126 MB L2 (config 1) is timed step by step with a 512 MB write between steps, outside the event pairs.
    vin = o if abc else v
    small_ws = ntrip * 3 * (-(-vin // 8) * 8) ** 3 * 8 < 2 * 126e6
    flush = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device="cuda") if small_ws else None
    pairs = []
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if flush is None:
        ev0.record()
    for _ in range(args.steps):
        if flush is not None:
            flush.add_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
        e_val = step()
        if flush is not None:
            b.record()
            pairs.append((a, b))
        prof = bqc.bqc_t_last_profile()
        launches += int(prof["kernel_launches"])
    if flush is None:
        ev1.record()
    barrier()
    clocks = sampler.stop()
    if flush is None:
        ms = ev0.elapsed_time(ev1) / max(args.steps, 1)
    else:
        ms = sum(a.elapsed_time(b) for a, b in pairs) / max(args.steps, 1)
        del flush
    if args.no_profile:        # kernel split from one profiled call outside the timed region
        assert bqc.bqc_t_energy_ex(o, v, X, *dev, opts=opts, workspace=ws, e_triplet=e_trip) == e_val
        prof = dict(bqc.bqc_t_last_profile(), kernel_launches=prof["kernel_launches"])
    peak_after = bqc.bqc_fp64_peak_tflops(0, min(args.peak_seconds, 1.0))
    # Denominator: the DMMA rate measured in this run, but never less than the pipe's full rate at the maximum SM
    # clock (SMs x clock x 128 flop/clk: what the microbenchmark reaches when nothing caps it) — a power-capped or
    # otherwise slow peak measurement must not inflate the fractions.
    peak_pipe = pipe_peak_tflops(gpu)
    peak_measured = max(peak_dmma, peak_after)
    peak = max(peak_measured, peak_pipe)

    # end to end through the C ABI with HOST buffers (H2D of all inputs + D2H of the scalar inside)
    e2e_ms, h2d, d2h = None, 0, 0
    if args.e2e_steps > 0:
        del ws, dev                                     # the host-pointer call makes its own device copies
        bqc.bqc_release_cached()
        torch.cuda.empty_cache()
        eopts = bqc.make_opts(occ_block=args.occ_block, occ_lo=opts.occ_lo, occ_hi=opts.occ_hi,
                              shard_rank=opts.shard_rank, shard_count=opts.shard_count,
                              flags=opts.flags & ~bqc.BQC_T_FLAG_PROFILE)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            e_host, h2d, d2h = bqc.bqc_t_energy_host(o, v, X, *host, opts=eopts)
        torch.cuda.synchronize()
        e2e_ms = (time.perf_counter() - t0) * 1e3 / args.e2e_steps
        assert e_host == e_val, "e2e result differs from the device-resident result"

    # max over ranks, whole-job aggregate; per-rank record for the scaling / load-balance report
    mine = {"rank": rank, "ms_per_step": ms, "e2e_ms_per_step": e2e_ms or 0.0, "flops": float(flops_rank),
            "triplets": ntrip, "slab_blocks_formed": int(prof["form_blocks"]) if prof else 0,
            "w_builder_ms": prof["gemm_ms"] if prof else 0.0, "launches": launches}
    if world > 1:
        per_rank = [None] * world
        dist.all_gather_object(per_rank, mine)
        e_total = bqc.combine_partials(e_val)              # the path's one exchange: a scalar per rank
    else:
        per_rank, e_total = [mine], e_val
    ms = max(r["ms_per_step"] for r in per_rank)
    e2e_ms_max = max(r["e2e_ms_per_step"] for r in per_rank)
    flops_total = sum(r["flops"] for r in per_rank)
    launches_total = sum(r["launches"] for r in per_rank)

    if rank == 0:
        # working set of one W-builder launch vs the 126 MB L2: slabs of the outer index + the F arrays it writes
        vin, oin = (o, v) if abc else (v, o)                   # inner ("virtual") / outer extents of the schedule
        slab_mb = vin * vin * ((v + o + 15) // 16 * 16) * 8 / 1e6
        f_mb = 3 * (-(-vin // 8) * 8) ** 3 * 8 / 1e6
        batch = max(1, int(round(ntrip / max(prof["gemm_launches"], 1)))) if prof else 1
        ws_mb = f_mb * batch + slab_mb * 3
        l2_note = (f"per W-builder launch: ~{batch} triplets x {f_mb:.0f} MB of F written + slabs of {slab_mb:.0f} MB "
                   f"each = {ws_mb:.0f} MB, " + ("larger than the 126 MB L2; no flush needed" if not small_ws else
                                                   "fits L2: 512 MB written between steps (outside the timed event pairs)"))
        value = flops_total / (ms * 1e-3) * 1e-12
        flops_full = bqc.bqc_t_flops(o, v, bqc.make_opts(flags=bqc.BQC_T_FLAG_ABC_DRIVEN) if abc else None)
        gemm_tf = flops_rank / (prof["gemm_ms"] * 1e-3) * 1e-12 if prof["gemm_ms"] > 0 else None
        traffic, traffic_src = ncu_traffic(args.config, args.schedule)
        mean_flops = flops_total / world
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "strong" if strong else "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, c, lo, hi, args.full, ntrip, abc),
                       "sample": f"all {ntrip} triplets of the workload per step and GPU (the reference arm's step is one "
                                 "triplet of the same workload; TFLOP/s normalises both)",
                       "schedule": args.schedule, "triplets_per_gpu": ntrip, "occ_block": bqc.bqc_t_plan_occ_block(o, v, X, opts),
                       "parallelism": (f"one E(T) dealt over {world} ranks by whole block triples (BQC_T_FLAG_SHARD_BLOCKS), "
                                       "inputs replicated, one scalar exchange" if strong else
                                       f"{world} rank(s), one occupied window each, inputs replicated, one scalar exchange"),
                       "l2": l2_note,
                       "timing": "CUDA events on the launch stream around K bqc_t_energy_ex calls, max over ranks"
                                 + ("; timed without BQC_T_FLAG_PROFILE (CUDA-graph replay for short schedules), "
                                    "kernel_ms_per_step / roofline from one profiled call after the timed region"
                                    if args.no_profile else ""),
                       "pinned_host": pinned, "input_gen_s": round(gen_s, 1)},
            "pct_of_fp64_tensor_peak": 100.0 * value / (peak * world),
            "fp64_tensor_peak_tflops_measured": peak_measured,
            "fp64_tensor_peak_tflops_used": peak,
            "seconds_per_step": ms * 1e-3,
            "seconds_per_full_E_T_extrapolated": flops_full / (value * 1e12),
            "e_t_of_step_hartree": e_total,
            "kernel_ms_per_step": {"w_builder": prof["gemm_ms"], "energy": prof["energy_ms"],
                                   "slab_former": prof["form_ms"], "prepare": prof["prepare_ms"],
                                   "call_total": prof["total_ms"]},
            "roofline": {"bound": "tensor", "kernel": "gemm_nt_kernel (W builder, row a2)",
                         "achieved": gemm_tf, "peak": peak, "unit": UNIT,
                         "frac": (gemm_tf / peak) if gemm_tf else None,
                         "peak_source": "max(FP64 DMMA peak measured in this run by bqc_fp64_peak_tflops — a register-"
                                        "resident mma.sync m8n8k4 loop on all SMs —, SMs x max SM clock x 128 flop/clk); "
                                        "MEASURED_PEAKS.json has no FP64 entry",
                         "launches": int(prof["gemm_launches"]),
                         "flops_per_launch": flops_rank / max(prof["gemm_launches"], 1),
                         "traffic": traffic, "traffic_source": traffic_src},
            "clocks": clocks,
            "e2e": {"value": (flops_total / (e2e_ms_max * 1e-3) * 1e-12) if e2e_ms_max else None, "unit": UNIT,
                    "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": e2e_ms_max, "steps": args.e2e_steps},
            "gpu_launches": launches_total,
        }
        if world > 1:
            out["ranks"] = {"per_rank": per_rank,
                            "load_imbalance_max_over_mean_flops": max(r["flops"] for r in per_rank) / mean_flops,
                            "time_imbalance_max_over_mean": ms / (sum(r["ms_per_step"] for r in per_rank) / world),
                            "backend": args.backend}
            if args.share_gpu:
                out["config"]["shared_gpu"] = ("TEST MODE: all ranks ran on cuda:0, so the timings are not a "
                                               "multi-GPU measurement")
        if world == 1 and not args.no_cpu_baseline:
            # the oracle as it stands on three triplets of the workload (one per class i<j<k, i=j<k, i<j=k); its
            # per-triplet values are compared with the e_ijk the timed GPU steps produced (north_star tolerance)
            mid = (lo + hi - 1) // 2
            trips = [(lo, mid, hi - 1), (lo, lo, hi - 1), (lo, hi - 1, hi - 1)][:max(1, args.cpu_triplets)]
            e_gpu = e_trip.cpu().numpy()
            dts, worst = [], 0.0
            for trip in trips:
                dt, e_ref = oracle_sample(inp, trip, abc)
                dts.append(dt)
                d = abs(e_gpu[bqc.bqc_t_triplet_index(nidx, *trip)] - e_ref)
                worst = max(worst, d / (1e-10 * abs(e_ref) + 1e-12 * abs(e_total) / max(ntrip, 1)))
            dt = float(np.sum(dts))
            out["cpu_baseline"] = {"value": len(trips) * f1 / dt * 1e-12, "unit": UNIT, "cores": cpu_threads(),
                                   "kind": "oracle",
                                   "sample": f"triplets {trips} of the workload ({f1:.3e} flops each) in {dt:.1f} s, "
                                             "NumPy/OpenBLAS oracle as it stands",
                                   "seconds_per_full_E_T_extrapolated": dt / len(trips) * flops_full / f1,
                                   "gpu_vs_oracle_worst_err_over_tol": worst}
            assert worst <= 1.0, f"GPU per-triplet energies differ from the oracle: {worst:.3g} x tolerance"
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
