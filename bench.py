#!/usr/bin/env python
"""bench.py -- ns per spin flip of the full Swendsen-Wang sweep (BASELINE.json metric) on B200.

    python bench.py --gpus 1 --steps K --warmup W            # the CUDA path (libsw.so)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, as it stands, on the host cores
    torchrun ... bench.py --gpus N ...                       # N independent replicas ("replicas only", weak scaling)

A step = one full SW sweep (bonds -> labels -> cluster decisions -> spin update) of the
workload BASELINE.json's metric is quoted on: q=2 Potts, L=4096, T=Tc (config 2), at an equilibrated state.
Prints ONE JSON line (rank 0).  See DESIGN.md section 8 for what every key means and how it is measured.
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
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "ns per spin flip (full SW sweep) at L=4096, T_c"
UNIT = "ns/spin-flip"
B_ALG = 10.0            # algorithmic HBM bytes per spin per sweep: 1+4 (label) + 4+1 (flip)
B_ALG_KERNEL = {"k_tile_label": 5.0, "k_tile_flip": 5.0, "k_flip": 5.0}   # per spin, per launch


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.samples = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            f = [x.strip() for x in s.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_ns_per_spin(L, q, model, T, seed, sweeps, warm):
    from oracle import sw_oracle as o
    s = o.init_spins(L, q, seed)
    s = o.run(L, q, model, T, seed, 0, warm, s)
    t0 = time.perf_counter()
    o.run(L, q, model, T, seed, warm, sweeps, s)
    dt = time.perf_counter() - t0
    return dt * 1e9 / (sweeps * L * L), dt


def run_reference(args):
    """Base-contract reference arm for this tier: the oracle, as it stands, one thread on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1202_0635_b200.workloads import CONFIGS, HEADLINE
    w = CONFIGS[HEADLINE]
    # bounded sample: one step = one oracle sweep of an L_s x L_s lattice of the same model at the same T,
    # L_s sized so that steps+warmup sweeps take about two minutes at ~200 ns per spin on one core
    budget_s, per_spin = 120.0, 200e-9
    n_steps = args.steps + args.warmup
    Ls = 64
    while Ls < w.L and (2 * Ls) ** 2 * n_steps * per_spin <= budget_s:
        Ls *= 2
    from oracle import sw_oracle as o
    s = o.init_spins(Ls, w.q, w.seed)
    s = o.run(Ls, w.q, w.model, w.T, w.seed, 0, args.warmup, s)
    t0 = time.perf_counter()
    o.run(Ls, w.q, w.model, w.T, w.seed, args.warmup, args.steps, s)
    dt = time.perf_counter() - t0
    ns = dt * 1e9 / (args.steps * Ls * Ls)
    sample = f"{args.steps} oracle sweeps of an L={Ls} lattice (q={w.q}, T=Tc), 1 thread, after {args.warmup} warm-up sweeps"
    line = {
        "impl": "reference", "metric": METRIC, "value": ns, "unit": UNIT, "n_gpus": 0, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt * 1e3 / args.steps, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "u8 spins / int32 labels / u32 Philox", "data": "synthetic",
        "config": {"workload": f"config 2 shape: q=2 Potts, T=Tc, bounded sample L={Ls} (metric workload L={w.L})", "sample_L": Ls},
        "cpu_baseline": {"value": ns, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": ns, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def load_capture(kernel: str, workload: str):
    """Per-launch counts of `kernel` from the committed ncu capture (profiles/traffic.json, written by
    `python -m paper_1202_0635_b200.ncu_summary --record`), or None if there is none for this workload or if the kernel
    sources changed since it was taken (the hash of csrc/ is stored with it)."""
    tr = ROOT / "profiles" / "traffic.json"
    if not tr.exists():
        return None
    try:
        from paper_1202_0635_b200.ncu_summary import csrc_sha256
        cap = json.loads(tr.read_text()).get(f"{kernel}@{workload}")
        if cap is None or cap.get("csrc_sha256") != csrc_sha256():
            return None
        return cap
    except Exception:
        return None


def run_batch(args, w, seed):
    """NEXT-2: B lattices of the workload's (L, q, model, T), own seeds, advanced together (sw_create_batch).  One JSON line."""
    import torch
    from paper_1202_0635_b200 import binding as sw
    B, N = args.batch, w.L * w.L
    bt = sw.Batch(w.L, w.q, w.model, [w.T] * B, [seed + 7919 * b for b in range(B)])
    bt.sweep(args.equil)
    sampler = ClockSampler(int(os.environ.get("LOCAL_RANK", "0")))
    sampler.start()
    for _ in range(3):
        bt.sweep(max(1, args.warmup // 3))
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    bt.sweep(args.steps)                              # synchronous at return
    dt = time.perf_counter() - t0
    clocks = sampler.stop()
    print(json.dumps({
        "metric": "ns per spin flip (full SW sweep), batch of lattices", "value": dt * 1e9 / (args.steps * B * N), "unit": UNIT, "n_gpus": 1,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "u8 spins / int32 labels / u32 Philox", "data": "synthetic",
        "config": {"workload": f"batch of {B} x {w.name}", "B": B, "L": w.L, "q": w.q, "model": "potts" if w.model == 0 else "clock", "T": w.T,
                   "equil_sweeps": args.equil, "timing": "host clock around one synchronous sw_batch_sweep(steps)",
                   "backend": "tiles of all lattices in one grid" if w.L % 128 == 0 else "one CTA per lattice"},
        "clocks": clocks}), flush=True)
    bt.close()


def run_microbench(args):
    """Issue-rate probes (sw_microbench): warp-instructions per SM cycle per sub-partition, per opcode and mix.
    Prints one JSON line per probe and a markdown table (the table is what profiles/ keeps)."""
    import ctypes
    import torch
    from paper_1202_0635_b200 import binding as sw
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --microbench needs a CUDA device")
    torch.cuda.init()
    torch.zeros(1, device="cuda")
    lib = sw.load()
    warps = [1, 2, 4, 8, 16]
    rows = []
    k = 0
    while True:
        name = lib.sw_microbench_name(k)
        if name is None:
            break
        rates = []
        for w in warps:
            out = (ctypes.c_double * 4)()
            rc = lib.sw_microbench(k, w, args.mb_iters, out)
            if rc != 0:
                raise SystemExit(f"sw_microbench({k}, {w}) failed: {rc}")
            rates.append(out[0])
        rows.append((k, name.decode(), rates))
        print(json.dumps({"probe": k, "name": name.decode(), "warps_per_smsp": warps, "units_per_cycle_per_smsp": rates}), flush=True)
        k += 1
    print()
    print("| probe | " + " | ".join(f"{w} warps/SMSP" for w in warps) + " |")
    print("|---|" + "---|" * len(warps))
    for k, name, rates in rows:
        print(f"| {name} | " + " | ".join(f"{r:.3f}" for r in rates) + " |")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--microbench", action="store_true", help="run the instruction-issue probes instead of the sweep bench")
    ap.add_argument("--mb-iters", type=int, default=4000)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default=None, help="a key of workloads.CONFIGS (default: the headline config)")
    ap.add_argument("--L", type=int, default=0, help="override the workload's lattice size (the L-scan of PAPER.md:75, Table 1)")
    ap.add_argument("--equil", type=int, default=300, help="untimed sweeps from the random start before warm-up")
    ap.add_argument("--algo", default="auto", choices=["auto", "generic", "tiled", "small", "hawick", "kalentev"],
                    help="labeling back-end (sw_set_algorithm); hawick / kalentev are the paper's own labellers (A/B reference)")
    ap.add_argument("--batch", type=int, default=0, help="B > 0: time a batch of B lattices of the workload's (L, q, model, T) (sw_create_batch)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup

    if args.microbench:
        run_microbench(args)
        return
    if args.impl == "reference":
        run_reference(args)
        return

    import numpy as np
    import torch
    from paper_1202_0635_b200 import binding as sw
    from paper_1202_0635_b200.workloads import CONFIGS, HEADLINE

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl cuda needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    w = CONFIGS[args.workload or HEADLINE]
    if args.L > 0:
        import dataclasses
        w = dataclasses.replace(w, L=args.L, name=f"{w.name}@L={args.L}")
    L, q, N = w.L, w.q, w.L * w.L
    from paper_1202_0635_b200 import replicas
    seed = replicas.replica_seed(w.seed, rank)       # replicas only: every rank its own lattice
    if args.batch > 0:
        run_batch(args, w, seed)
        return
    ALGOS = {"auto": 0, "generic": 1, "tiled": 2, "small": 3, "hawick": 4, "kalentev": 5}
    lat = sw.Lattice(L, q, w.model, w.T, seed, algo=ALGOS[args.algo])
    stream = torch.cuda.current_stream()
    l2_flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    lat.sweep(args.equil)                             # reach the equilibrium cluster structure (untimed)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: K steps, each bracketed by events, L2 flushed between steps -------------------
    for _ in range(args.warmup):
        l2_flush.zero_()
        lat.sweep_async(1)
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    launches0 = lat.launch_count
    wall0 = time.perf_counter()
    for k in range(args.steps):
        l2_flush.zero_()                              # not timed: between ev1[k-1] and ev0[k]
        ev0[k].record(stream)
        lat.sweep_async(1)
        ev1[k].record(stream)
    barrier()
    wall = time.perf_counter() - wall0
    launches = lat.launch_count - launches0
    step_ms = [a.elapsed_time(b) for a, b in zip(ev0, ev1)]
    total_ms = float(sum(step_ms))

    # back-to-back (warm L2) run of the same K steps, for context
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    lat.sweep_async(args.steps)
    e1.record(stream)
    barrier()
    b2b_ms = e0.elapsed_time(e1)
    # the paper's second column: update + measurement of energy and magnetisation every sweep
    barrier()
    m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    m0.record(stream)
    lat.sweep_record(args.steps)
    m1.record(stream)
    barrier()
    meas_ms = m0.elapsed_time(m1)
    clocks = sampler.stop()
    st = lat.stats()
    iters_per_sweep = float(st[5] / st[6]) if st[6] > 0 else None     # the paper's labellers only (6.6-8.6 at Tc)

    # ---- per-kernel device time (events between kernels), L2 flushed before each sweep ----------------------
    prof = {}
    nprof = min(args.steps, 50)
    for _ in range(nprof):
        l2_flush.zero_()
        for name, ms in lat.sweep_profile(1).items():
            prof[name] = prof.get(name, 0.0) + ms
    prof = {k: v / nprof for k, v in prof.items()}    # ms per launch
    dom = max(prof, key=prof.get)
    peak, peak_src = peaks()
    dom_bytes = B_ALG_KERNEL.get(dom, 5.0) * N
    t_dom = prof[dom] * 1e-3                                          # seconds per launch of the dominant kernel
    hbm_nominal = {"bytes_per_launch": dom_bytes, "achieved": dom_bytes / t_dom / 1e9, "peak": peak, "unit": "GB/s",
                   "frac": dom_bytes / t_dom / 1e9 / peak, "peak_source": peak_src,
                   "note": "SURVEY 8(d) accounting (int32 labels: 1 + 4 B/site); this kernel moves 1 + 2 B/site"}
    roofline = dict(hbm_nominal, bound="hbm", kernel=dom, traffic=None, ms_per_launch=prof[dom])
    cap = load_capture(dom, w.name)
    if cap is not None:
        # The dominant kernel is bound by the integer ALU pipe, not by HBM: achieved = ALU-pipe busy
        # cycles per launch (2 per ALU-class warp-instruction and 2 per IMAD.WIDE, rates measured by `bench.py --microbench`,
        # counts from the committed ncu capture of this very source) / live kernel time; peak = sub-partitions x SM clock.
        sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
        clk_hz = (clocks["sm_mhz"] or 1965.0) * 1e6
        apeak = sms * 4 * clk_hz
        roofline = {"bound": "alu", "kernel": dom, "achieved": cap["alu_pipe_cycles"] / t_dom, "peak": apeak, "unit": "ALU-pipe busy cycles/s",
                    "frac": cap["alu_pipe_cycles"] / t_dom / apeak, "traffic": cap["dram_bytes"], "ms_per_launch": prof[dom],
                    "peak_source": f"{sms} SMs x 4 sub-partitions x {clk_hz / 1e6:.0f} MHz (one ALU-pipe cycle per sub-partition and clock)",
                    "warp_instructions_per_launch": cap["warp_instructions"],
                    "other_pipes": {k: cap[k + "_pipe_cycles"] / t_dom / apeak for k in ("fma", "xu", "lsu")},
                    "issue_slots": cap["warp_instructions"] / t_dom / apeak,
                    "model": "profiles/r2_microbench.md (measured issue rates) applied to the opcode histogram of profiles/" + cap["report"],
                    "hbm_nominal": hbm_nominal,
                    "hbm_measured": {"bytes_per_launch": cap["dram_bytes"], "achieved": cap["dram_bytes"] / t_dom / 1e9, "peak": peak,
                                     "unit": "GB/s", "frac": cap["dram_bytes"] / t_dom / 1e9 / peak}}

    # ---- end to end through the C ABI with host buffers -------------------------------------------------------
    host_in = torch.empty((L, L), dtype=torch.uint8).pin_memory()
    host_out = torch.empty((L, L), dtype=torch.uint8).pin_memory()
    lat.get_spins(host_in)
    t_idx = lat.sweep_index
    e2e_steps = min(args.steps, 50)
    for _ in range(3):
        lat.set_spins(host_in, t_idx); lat.sweep(1); lat.get_spins(host_out); lat.observables()
    barrier()
    t0 = time.perf_counter()
    for k in range(e2e_steps):
        lat.set_spins(host_in, t_idx + k)             # H2D: L*L bytes
        lat.sweep(1)
        lat.get_spins(host_out)                       # D2H: L*L bytes
        bh, sh = lat.observables()                    # D2H: 32 x 8 bytes
        host_in, host_out = host_out, host_in
    barrier()
    e2e_s = time.perf_counter() - t0
    total_ms, b2b_ms, e2e_s = replicas.max_over_ranks([total_ms, b2b_ms, e2e_s], dist, device="cuda")

    flips = float(world) * args.steps * N
    value = replicas.whole_job_ns_per_flip(total_ms, args.steps, N, world)   # ns per spin flip, whole job
    e2e_value = e2e_s * 1e9 / (float(world) * e2e_steps * N)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        Ls, ns_sw = min(L, 4096), 12     # ~15 s of one host core at ~70 ns per spin
        ns, dt = oracle_ns_per_spin(Ls, q, w.model, w.T, w.seed, ns_sw, 1)
        cpu = {"value": ns, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{ns_sw} oracle sweeps of an L={Ls} lattice of the same model and T after 1 warm-up sweep ({dt:.1f} s)",
               "note": "the test oracle as it stands: single thread, never tuned (a checker, not a CPU Swendsen-Wang implementation to beat)"}

    if rank == 0:
        sweep_gbs = B_ALG * N / (total_ms / args.steps * 1e-3) / 1e9
        line = {
            "metric": METRIC if w.name == HEADLINE else "ns per spin flip (full SW sweep)", "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "u8 spins / int32 labels / u32 Philox", "data": "synthetic",
            "config": {"workload": w.name, "L": L, "q": q, "model": "potts" if w.model == 0 else "clock", "T": w.T,
                       "equil_sweeps": args.equil, "l2": "flushed between steps (256 MiB memset, untimed)",
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "backend": {1: "generic", 2: "tiled", 3: "one CTA", 4: "hawick (paper)", 5: "kalentev (paper)"}[lat.algorithm]},
            "spin_flips_per_s": flips / (total_ms * 1e-3),
            "back_to_back": {"ns_per_spin_flip": b2b_ms * 1e6 / flips, "ms_per_step": b2b_ms / args.steps, "note": "same K sweeps in one enqueue, warm L2"},
            "with_measurement": {"ns_per_spin_flip": meas_ms * 1e6 / (args.steps * N), "ms_per_step": meas_ms / args.steps,
                                 "note": "rank 0: same K sweeps with the integer energy / magnetisation histograms of every configuration (sw_sweep_record)"},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": N, "d2h_bytes_per_step": N + 2 * 16 * 8, "steps": e2e_steps},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "sweep_roofline": {"bytes_per_spin": B_ALG, "achieved_gbs": sweep_gbs, "frac": sweep_gbs / peak,
                               "note": "whole sweep at the contract's 10 B per spin (SURVEY 8(d)) against the measured HBM copy peak"},
            "kernels_ms": prof,
            "cpu_baseline": cpu,
            "labeling_iterations_per_sweep": iters_per_sweep,
            "paper_context": {"gtx580_ns_per_spin_flip": 2.51, "source": "PAPER.md:83 Table 1 (another machine: context, not the target)"},
            "wall_s": wall,
        }
        print(json.dumps(line), flush=True)
    lat.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
