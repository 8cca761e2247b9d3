"""The five synthetic workloads of BASELINE.json, as cg_init arguments.

Pure data shared by the tests, bench.py and both implementations' harnesses; holds none of
the method's arithmetic.  The paper's own workloads are self-generated random lattices
(2D L x L torus, nu = 1/2, xi = 1, W = 1, random start PAPER.md:84), so the
inputs ARE the recipe: (L, W, xi, T, E, seed, M) plus the number of executed hops.
"""

CONFIGS = {
    "cfg1_L16": [dict(L=16, W=1.0, xi=1.0, T=0.1, E=0.0, seed=1, M=256, hops=100_000)],
    "cfg2_L64": [dict(L=64, W=1.0, xi=1.0, T=0.05, E=0.0, seed=2, M=1024, hops=1_000_000)],
    "cfg3_L128": [dict(L=128, W=1.0, xi=1.0, T=T, E=0.01, seed=s, M=4096, hops=1_000_000)
                  for T, s in ((0.2, 3), (0.1, 4), (0.05, 5), (0.03, 6))],
    # "max resident threads" (SMs x 2048) is resolved at run time: M=None
    "cfg4_L256": [dict(L=256, W=1.0, xi=1.0, T=0.02, E=0.01, seed=7, M=M, hops=1_000_000)
                  for M in (1024, 8192, 65536, None)],
    "cfg5_L512": [dict(L=512, W=1.0, xi=1.0, T=0.05, E=0.01, seed=8, M=65536, hops=1_000_000)],
}

HEADLINE = "cfg5_L512"


def init_args(cfg, max_resident_threads=148 * 2048):
    """dict -> keyword arguments of cg_init / cgo_init."""
    kw = {k: cfg[k] for k in ("L", "W", "xi", "T", "E", "seed", "M")}
    if kw["M"] is None:
        kw["M"] = int(max_resident_threads)
    return kw
