"""Per-config throughput report and replica packing (§8f-2), through the Python binding.

    python -m paper_1407_5026_b200.report --configs [--hops 200000] [--warm 2000]
    python -m paper_1407_5026_b200.report --replicas [--hops 100000]
    python -m paper_1407_5026_b200.report --observables [--hops 200000]

--configs: every workload of BASELINE.json (workloads.CONFIGS), a bounded prefix of its chain, one line each:
accepted hops/s, window proposals evaluated/s (M per PR iteration), attempts consumed/s
(m = (p-1)M + q per hop), mean p and mean q (0-based label of the executed proposal),
acceptance A = hops/attempts over the run and over its last 10 %, the paper's split of the time per hop
 W_U = the eps update alone (`cg_apply_hops` on the hops just executed and their reversal) and
W_R = time per hop - W_U (in the persistent kernel the two overlap, so W_R is what the update does not
explain), the update's algorithmic GB/s (16 N bytes per hop) and the drift of the incremental eps against a
full-sum recomputation.

--replicas: independent sims side by side on one GPU: packed into ONE persistent launch (`cg_run_many`), and
as separate persistent kernels on separate CUDA streams.

--observables: the read-only device passes of include/cg.h "Observables" on a chain with its hop log: the
deterministic clock t = attempts/Gamma next to the stochastic one of step 3c ("does not produce any
appreciable difference"), sigma0 = dP/(N E t), the density of states around the
Coulomb gap, the length of the P(t) series, and what each call costs (wall time of the whole call,
device-to-host copy included).

Needs a CUDA device; nothing here computes on the host.
"""
import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np      # noqa: E402
import torch            # noqa: E402

import workloads        # noqa: E402
from . import binding   # noqa: E402


def _timed(fn):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def update_alone_us(kw, n_script=1000):
    """W_U: microseconds per hop of step a6 alone at this lattice, on hops of its own chain."""
    u = binding.CoulombGlass(hop_log=n_script, **kw)
    u.run(n_script)
    _, hi, hj = u.hops()
    v = binding.CoulombGlass(**kw)
    si = np.concatenate([hi, hj[::-1]])
    sj = np.concatenate([hj, hi[::-1]])
    best = min(v.apply_hops(si, sj) for _ in range(3))
    return 1e3 * best / si.size


def report_configs(hops, warm):
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    print("# %s, %d SMs; %d warm-up hops, then min(config's hops, %d) timed in 10 chunks" % (
        torch.cuda.get_device_name(0), sms, warm, hops))
    for name, cfgs in workloads.CONFIGS.items():
        for cfg in cfgs:
            kw = workloads.init_args(cfg, sms * 2048)
            N, M = kw["L"] ** 2, kw["M"]
            g = binding.CoulombGlass(**kw)
            H = min(cfg["hops"], hops)
            chunk = H // 10
            g.run(warm)
            torch.cuda.synchronize()
            c0 = g.counters()
            ms, cs = 0.0, [c0]
            for _ in range(10):
                ms += _timed(lambda: g.run(chunk))
                cs.append(g.counters())
            c, c9 = cs[-1], cs[-2]
            Hd = c["hops"] - c0["hops"]
            it = c["iterations"] - c0["iterations"]
            at = c["attempts"] - c0["attempts"]
            mean_q = (at - (it - Hd) * M) / Hd - 1.0
            A_all = Hd / at
            A_last = (c["hops"] - c9["hops"]) / (c["attempts"] - c9["attempts"])
            us_hop = 1e3 * ms / Hd
            w_u = update_alone_us(kw)
            ln = g.launch()
            print("%-9s T=%-5g M=%-6d %3d CTAs x %d: %7.0f hops/s  %.2e proposals/s  %.2e attempts/s  "
                  "p=%.3f q=%8.1f  A=%.2e (last 10%%: %.2e)  %5.2f us/hop = W_U %.3f + W_R %.2f  "
                  "update alone %6.0f GB/s  drift %.1e" % (
                      name, kw["T"], M, ln["n_ctas"], ln["threads"], Hd / ms * 1e3, M * it / ms * 1e3,
                      at / ms * 1e3, it / Hd, mean_q, A_all, A_last, us_hop, w_u, us_hop - w_u,
                      16.0 * N / w_u / 1e3, g.recompute_eps()))
            sys.stdout.flush()


def report_replicas(hops):
    def run(name, idxs, copies):
        sims = []
        for r in range(copies):
            for i in idxs:
                kw = workloads.init_args(workloads.CONFIGS[name][i])
                kw["seed"] += 100 * r
                sims.append(binding.CoulombGlass(stream=torch.cuda.Stream(), **kw))
        for g in sims:
            g.run(1000)
        torch.cuda.synchronize()

        def go():
            for g in sims:
                g.run(hops)
            for g in sims:
                torch.cuda.current_stream().wait_stream(g._stream)
        ms = _timed(go)
        print("%s x%d replicas (%d CTAs each): %.0f hops/s aggregate, %.0f per replica" % (
            name, len(sims), sims[0].launch()["n_ctas"], len(sims) * hops / ms * 1e3, hops / ms * 1e3))
        sys.stdout.flush()

    def packed(name, idxs, copies, n_ctas=0):
        """The same replica sets through cg_run_many: one launch, every sim on its own CTAs."""
        sims = []
        for r in range(copies):
            for i in idxs:
                kw = workloads.init_args(workloads.CONFIGS[name][i])
                kw["seed"] += 100 * r
                g = binding.CoulombGlass(**kw)
                if n_ctas:
                    g.set_launch(n_ctas, 512)
                sims.append(g)
        binding.run_many(sims, 1000)
        torch.cuda.synchronize()
        ms = _timed(lambda: binding.run_many(sims, hops))
        print("%s x%d replicas packed into one launch (%d CTAs each): %.0f hops/s aggregate, %.0f per replica" % (
            name, len(sims), sims[0].launch()["n_ctas"], len(sims) * hops / ms * 1e3, hops / ms * 1e3))
        sys.stdout.flush()

    sms = torch.cuda.get_device_properties(0).multi_processor_count
    packed("cfg3_L128", [0, 1, 2, 3], 1)
    packed("cfg3_L128", [0, 1, 2, 3], 2, n_ctas=sms // 8)
    packed("cfg1_L16", [0], 32)
    packed("cfg1_L16", [0], sms)
    packed("cfg2_L64", [0], sms // 5)
    run("cfg3_L128", [0, 1, 2, 3], 1)     # the temperature sweep of config 3 as one replica set
    run("cfg3_L128", [0, 1, 2, 3], 2)
    run("cfg1_L16", [0], 1)
    run("cfg1_L16", [0], 32)
    run("cfg1_L16", [0], 148)
    run("cfg2_L64", [0], 29)


def report_observables(hops):
    import time
    print("# %s; %d hops from the random start, hop log on" % (torch.cuda.get_device_name(0), hops))

    def wall(fn):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        r = fn()
        return r, 1e3 * (time.perf_counter() - t0)

    for name, idx in (("cfg3_L128", 1), ("cfg5_L512", 0)):
        cfg = workloads.CONFIGS[name][idx]
        kw = workloads.init_args(cfg)
        g = binding.CoulombGlass(hop_log=hops, **kw)
        g.run(hops)
        t_det = g.state()[2]
        g.time_stochastic()                                  # first call: context warm-up
        t_st, ms_t = wall(g.time_stochastic)
        (hist, outside), ms_d = wall(lambda: g.dos(-4.0, 2.0**-4, 128))
        (t, P), ms_s = wall(g.series)
        sig, _ = wall(g.sigma0)
        gdos = hist / (g.N * 2.0**-4)
        mid = 64                                             # bin [0, 1/16)
        print("%s T=%-5g: t_det %.6e  t_stoch %.6e (rel. diff %+.2e)  sigma0 %.4e  dP %d" % (
            name, kw["T"], t_det, t_st, t_st / t_det - 1, sig, P[-1]))
        print("    g(eps) at eps = -2, -1, -0.5, -0.25, 0, 0.25, 0.5, 1, 2: %s  (outside [-4,4): %d)" % (
            " ".join("%.3f" % gdos[mid + int(e * 16)] for e in (-2, -1, -0.5, -0.25, 0, 0.25, 0.5, 1, 2)), outside))
        print("    cost: time_stochastic %.2f ms (%d logged hops), dos %.2f ms (N = %d), series %.2f ms (%d points)" % (
            ms_t, hops, ms_d, g.N, ms_s, t.size))
        sys.stdout.flush()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", action="store_true")
    ap.add_argument("--replicas", action="store_true")
    ap.add_argument("--observables", action="store_true")
    ap.add_argument("--hops", type=int, default=0)
    ap.add_argument("--warm", type=int, default=2000)
    a = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("report needs a CUDA device: the hot path has no CPU fallback")
    if a.configs:
        report_configs(a.hops or 200_000, a.warm)
    if a.replicas:
        report_replicas(a.hops or 100_000)
    if a.observables:
        report_observables(a.hops or 200_000)


if __name__ == "__main__":
    main()
