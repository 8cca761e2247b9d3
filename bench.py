#!/usr/bin/env python
"""bench.py — accepted hops/s and proposals/s of the PR-KMC hot path (BASELINE.json metric).

A "step" is one cg_run(hops_per_step) of the whole hot path (propose, select, apply, update)
on the headline workload, config 5 of BASELINE.json (L=512, T=0.05, E=0.01, M=65536, seed 8).
N GPUs run N independent replicas (seeds 8, 9, ...),
no data-path collective; value = hops of all ranks / max-over-ranks device time.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
"""
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

import workloads  # noqa: E402

METRIC, UNIT = "accepted_hops_per_s", "hops/s"


def rank_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def reduce_over_ranks(ms, units, dist=None):
    """(device ms of this rank, units it processed) -> (max ms over ranks, sum of units)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms), int(units)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(ms)], dtype=torch.float64, device=dev)
    u = torch.tensor([int(units)], dtype=torch.int64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), int(u.item())


def replica_config(rank):
    """Rank r runs config 5 with seed 8 + r: independent samples, the paper's own
    recommendation for using more hardware."""
    cfg = dict(workloads.CONFIGS[workloads.HEADLINE][0])
    cfg["seed"] += rank
    return cfg


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=lambda: self.rows.extend(self.proc.stdout), daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            reasons.update(n for n, v in zip(names, f[3:7]) if v.lower() == "active")
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def time_oracle(cfg, seconds, chunk):
    """The oracle as it stands, one core, on a bounded sample of the workload."""
    from oracle import cgo
    kw = workloads.init_args(cfg)
    t0 = time.perf_counter()
    o = cgo.Oracle(hop_log=False, **kw)
    t_init = time.perf_counter() - t0
    hops, t0 = 0, time.perf_counter()
    while True:
        o.run(chunk)
        hops += chunk
        el = time.perf_counter() - t0
        if el >= seconds:
            break
    c = o.counters()
    return {"hops": hops, "seconds": el, "init_seconds": t_init, "attempts": c["attempts"],
            "update_seconds": o.update_seconds(), "near_ties": o.near_ties()}


def run_reference(args):
    """--impl reference: the CPU oracle (serial mixed algorithm) on host cores."""
    rank, world = rank_world()
    if rank != 0:
        return
    from oracle import cgo
    cfg = replica_config(0)
    kw = workloads.init_args(cfg)
    hops_per_step = args.ref_hops_per_step
    o = cgo.Oracle(hop_log=False, **kw)
    for _ in range(args.warmup):
        o.run(hops_per_step)
    a0 = o.counters()["attempts"]
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.run(hops_per_step)
    el = time.perf_counter() - t0
    hops = args.steps * hops_per_step
    c = o.counters()
    value = hops / el
    sample = "%d steps x %d hops of config 5 after %d warm-up hops from the random start" % (
        args.steps, hops_per_step, args.warmup * hops_per_step)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "cfg5_L512 (L=512, T=0.05, E=0.01, xi=1, W=1, seed=8); M only enters "
                               "the oracle's iteration bookkeeping", "hops_per_step": hops_per_step},
        "attempts_per_s": (c["attempts"] - a0) / el,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "host_cores": os.cpu_count()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


CTL_BYTES = 128  # sizeof(CgCtl) in csrc/cg.cu: the control block cg_set_state / cg_get_state move


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    rank, world = rank_world()
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_1407_5026_b200 as pkg

    sms = torch.cuda.get_device_properties(local).multi_processor_count
    cfg = replica_config(rank)
    kw = workloads.init_args(cfg, sms * 2048)
    N, H, K, W = kw["L"] ** 2, args.hops_per_step, args.steps, args.warmup
    warm_kw = dict(kw, seed=kw["seed"] + 1000)
    warm = pkg.CoulombGlass(device=local, **warm_kw)     # warm-up replica: same shape, other seed
    g = pkg.CoulombGlass(device=local, **kw)             # the timed workload starts at hop 0
    if args.ctas or args.threads:
        warm.set_launch(args.ctas, args.threads)
        g.set_launch(args.ctas, args.threads)
    flush = torch.zeros(512 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(W):
        warm.run(H)
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    with ClockSampler(local) as clk:
        for e0, e1 in ev:
            flush.add_(1)                 # L2 flush between timed steps (not timed)
            e0.record()
            g.run(H)                      # ONE persistent kernel launch = one step
            e1.record()
        barrier()
    ms_rank = sum(e0.elapsed_time(e1) for e0, e1 in ev)
    ms, hops_all = reduce_over_ranks(ms_rank, K * H, dist if world > 1 else None)
    c = g.counters()
    assert c["hops"] == K * H

    # ---- end to end through the C ABI with pinned HOST buffers (restore -> run -> read back)
    n_host = torch.empty(N, dtype=torch.int8).pin_memory().numpy()
    eps_host = torch.empty(N, dtype=torch.float64).pin_memory().numpy()
    t_e2e, dP = warm.state_into(n_host, eps_host)
    wc = warm.counters()
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        warm.set_state(n_host, eps_host, wc["attempts"], wc["hops"], dP)      # H2D
        warm.run(H)
        _, dP = warm.state_into(n_host, eps_host)                             # D2H, syncs
        wc = warm.counters()
    barrier()
    e2e_ms, e2e_hops = reduce_over_ranks(1e3 * (time.perf_counter() - t0), K * H, dist if world > 1 else None)
    bitmap = 4 * ((N + 31) // 32)
    e2e = {"value": e2e_hops / (e2e_ms * 1e-3), "unit": UNIT,
           "h2d_bytes_per_step": 8 * N + bitmap + CTL_BYTES,
           "d2h_bytes_per_step": 8 * N + bitmap + 3 * CTL_BYTES,
           "what": "cg_set_state(host n, eps) + cg_run + cg_get_state(host n, eps) + cg_get_counters per step"}

    if rank != 0:
        return
    sec = ms * 1e-3
    out = {
        "metric": METRIC, "value": hops_all / sec, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg5_L512: L=512 N=262144 T=0.05 E=0.01 xi=1 W=1 M=65536 seed=8(+rank), "
                               "hops 1..steps*hops_per_step from the random start",
                   "hops_per_step": H, "launch": g.launch(), "replicas": world,
                   "l2": "flushed between timed steps (512 MiB write); within a step the state is "
                         "L2-resident by construction"},
        "proposals_per_s": world * c["proposals_evaluated"] / sec if world == 1 else None,
        "attempts_per_s": c["attempts"] / sec if world == 1 else None,
        "rank0": {"attempts": c["attempts"], "iterations": c["iterations"],
                  "proposals_evaluated": c["proposals_evaluated"],
                  "mean_p": c["iterations"] / c["hops"], "acceptance": c["hops"] / c["attempts"],
                  "proposals_per_s": c["proposals_evaluated"] / (ms_rank * 1e-3),
                  "us_per_hop": 1e3 * ms_rank / c["hops"]},
        "gpu_launches": K,
        "e2e": e2e,
        "clocks": clk.summary(),
    }

    # ---- roofline of the eps update (16 N algorithmic bytes per hop, L2-resident)
    l2_peak = pkg.bench_l2_rmw(16 * N, reps=2000, trials=10)      # 4 MiB = both eps buffers
    achieved = 16.0 * N * c["hops"] / (ms_rank * 1e-3) / 1e9
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    out["roofline"] = {
        "bound": "l2", "kernel": "cg_pr_persistent (the whole hop: propose, select, apply, update; one launch per step)",
        "achieved": achieved, "peak": l2_peak, "unit": "GB/s", "frac": achieved / l2_peak,
        # ncu --set full (profiles/r1l_ncu_pr_persistent.txt, 20 000 hops): 4.37 MB of DRAM traffic per launch =
        # 0.22 KB per hop and 6.95 MB of L2 sectors (4.84 read + 2.11 written) per hop - the state is L2-resident,
        # so DRAM bytes are not the bound
        "traffic": 219.0 * c["hops"] / K, "traffic_source": "ncu dram__bytes per hop x hops per launch",
        "l2_bytes_per_hop_ncu": 6.95e6,
        "peak_source": "measured live: cg_bench_l2_rmw, 16-byte ld.cg/st.cg RMW over a resident %d-byte "
                       "buffer, 2000 passes per launch, best of 10 (MEASURED_PEAKS.json has no L2 figure)" % (16 * N),
        "algorithmic_bytes_per_hop": 16 * N,
        "hbm_peak_gbs": peaks.get("hbm_gbs"), "frac_of_hbm_peak": achieved / peaks["hbm_gbs"] if peaks.get("hbm_gbs") else None,
    }
    # the update kernel alone on scripted hops (forward log + its reversal = back to the start state)
    u = pkg.CoulombGlass(device=local, hop_log=2000, **warm_kw)
    u.run(2000)
    _, hi, hj = u.hops()
    v = pkg.CoulombGlass(device=local, **warm_kw)
    si = np.concatenate([hi, hj[::-1]]); sj = np.concatenate([hj, hi[::-1]])
    best = min(v.apply_hops(si, sj) for _ in range(5))
    upd = 16.0 * N * si.size / (best * 1e-3) / 1e9
    out["roofline_update_kernel"] = {
        "bound": "l2", "kernel": "cg_update_scripted (step a6 alone, %d scripted hops per launch)" % si.size,
        "achieved": upd, "peak": l2_peak, "unit": "GB/s", "frac": upd / l2_peak, "us_per_hop": 1e3 * best / si.size}

    if world == 1 and not args.no_cpu_baseline:
        r = time_oracle(cfg, args.cpu_seconds, 250)
        out["cpu_baseline"] = {
            "value": r["hops"] / r["seconds"], "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "first %d hops of config 5 from the random start (%.1f s; init %.1f s not timed)" % (
                r["hops"], r["seconds"], r["init_seconds"]),
            "attempts_per_s": r["attempts"] / r["seconds"], "host_cores": os.cpu_count(),
            "W_U_us_per_hop": 1e6 * r["update_seconds"] / r["hops"],
            "update_gbs": 16.0 * N * r["hops"] / r["update_seconds"] / 1e9, "near_ties": r["near_ties"]}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--hops-per-step", type=int, default=100_000)
    ap.add_argument("--ref-hops-per-step", type=int, default=2_000)
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ctas", type=int, default=0)
    ap.add_argument("--threads", type=int, default=0)
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
