"""Pins for the Markov chain itself: PR bookkeeping, acceptance probabilities, stationarity.

PAPER.md:29-41 (rejection / parallel rejection), 54-57 (rates), 71-78 (mixed PR algorithm).
"""
import math
import os

import numpy as np
import pytest
from scipy import stats

from physics_bruteforce import distance_matrix, hamiltonian, min_image

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_fig1a_worked_example(oracle_lib):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "fig1a_pr_example.txt")) if l[0] != "#"]
    M, p, q, m = (int(x) for x in rows[0])
    assert oracle_lib.pr_split(m, M) == (p, q)
    # neighbours of the example: label q=M closes an iteration, q=1 opens the next
    assert oracle_lib.pr_split(12, 12) == (1, 12)
    assert oracle_lib.pr_split(13, 12) == (2, 1)
    assert oracle_lib.pr_split(1, 12) == (1, 1)


@pytest.mark.parametrize("A,M", [(0.05, 12), (0.01, 64), (0.2, 4), (0.002, 1024)])
def test_fixed_acceptance_chain(oracle_lib, A, M):
    """<m> = 1/A and <p> = 1/[1-(1-A)^M] for constant acceptance A."""
    hops = 60000
    o = oracle_lib.Oracle(16, T=0.1, seed=1234, M=M)
    o.set_fixed_A(A)
    o.run(hops)
    a, _, _ = o.hops()
    ends = a.astype(np.int64) + 1
    m = np.diff(np.concatenate([[0], ends]))
    p = (m - 1) // M + 1
    # m is geometric(A): mean 1/A, variance (1-A)/A^2
    assert abs(m.mean() - 1 / A) < 5 * math.sqrt((1 - A) / A**2 / hops)
    B = 1 - (1 - A) ** M                       # probability an iteration contains an accept
    assert abs(p.mean() - 1 / B) < 5 * math.sqrt((1 - B) / B**2 / hops) + 1e-12
    c = o.counters()
    assert c["hops"] == hops and c["attempts"] == ends[-1]
    assert c["iterations"] == p.sum() and c["proposals_evaluated"] == M * p.sum()
    # distribution, not only the mean: P(m > x) = (1-A)^x
    for x in (int(0.5 / A), int(2 / A)):
        want = (1 - A) ** x
        assert abs((m > x).mean() - want) < 5 * math.sqrt(want * (1 - want) / hops)


def _enumerate_first_hop(o, L, T, E):
    """Exact law of the first executed hop from a fixed state on a tiny lattice:
    P_prop(i,k) = (1/N) w_k/S, acc = theta_ij min[1, exp(-dH/T)] (Eq.(2)),
    dH by brute-force H(after)-H(before) from Eq.(1) plus the field term -E dx."""
    n, _, _, _ = o.state()
    phi = o.phi()
    N = L * L
    h = L // 2
    disc = sorted((dy * dy + dx * dx, dy, dx) for dy in range(-h + 1, h + 1)
                  for dx in range(-h + 1, h + 1) if 0 < dy * dy + dx * dx <= h * h)
    w = np.array([math.exp(-2.0 * math.sqrt(r2)) for r2, _, _ in disc])
    S = w.sum()
    H0 = hamiltonian(n, phi, L)
    prob = {}
    for i in range(N):
        yi, xi = divmod(i, L)
        for k, (_, dy, dx) in enumerate(disc):
            j = ((yi + dy) % L) * L + (xi + dx) % L
            if n[i] != 1 or n[j] != 0:
                continue
            m = n.copy(); m[i] = 0; m[j] = 1
            dH = hamiltonian(m, phi, L) - H0 - E * dx
            prob[(i, j)] = (1.0 / N) * (w[k] / S) * min(1.0, math.exp(-dH / T))
    return prob


@pytest.mark.parametrize("T,E,seed", [(0.5, 0.0, 7), (0.3, 0.3, 8)])
def test_4x4_exact_acceptance_probabilities(oracle_lib, T, E, seed):
    L, R = 4, 20000
    o = oracle_lib.Oracle(L, T=T, E=E, seed=seed, M=4)
    n0 = o.state()[0].copy()
    prob = _enumerate_first_hop(o, L, T, E)
    A = sum(prob.values())
    counts = {}
    ms = np.empty(R)
    for r in range(R):
        start = r * 1000003
        o.set_state(n0, start)
        before = o.counters()["hops"]
        o.run(1)
        a, i, j = o.hops(before, 1)
        key = (int(i[0]), int(j[0]))
        assert key in prob, "executed a hop of zero probability"
        counts[key] = counts.get(key, 0) + 1
        ms[r] = int(a[0]) + 1 - start
    keys = sorted(prob)
    exp = np.array([prob[k] / A * R for k in keys])
    obs = np.array([counts.get(k, 0) for k in keys], float)
    big = exp >= 5
    obs_b = np.append(obs[big], obs[~big].sum()); exp_b = np.append(exp[big], exp[~big].sum())
    if exp_b[-1] == 0:
        obs_b, exp_b = obs_b[:-1], exp_b[:-1]
    assert stats.chisquare(obs_b, exp_b).pvalue > 1e-4
    assert abs(ms.mean() - 1 / A) < 5 * math.sqrt((1 - A) / A**2 / R)


def test_4x4_stationary_distribution_is_boltzmann(oracle_lib):
    """Eq.(2) with a symmetric proposal satisfies detailed balance w.r.t. exp(-H/T) at E=0
    (PAPER.md:54-57, 71).  Attempt-weighted histogram over the C(16,8)=12870 states."""
    L, T = 4, 0.5
    o = oracle_lib.Oracle(L, T=T, E=0.0, seed=2024, M=4)
    phi = o.phi()
    n = o.state()[0].astype(np.int64).copy()
    hops = 1500000
    o.run(hops)
    a, i, j = o.hops()
    ends = a.astype(np.int64) + 1
    hold = np.diff(np.concatenate([[0], ends]))          # attempts spent in the state before hop h
    pw = 1 << np.arange(16)
    code = int((n * pw).sum())
    delta = (1 << j.astype(np.int64)) - (1 << i.astype(np.int64))
    codes = code + np.concatenate([[0], np.cumsum(delta)[:-1]])   # state held before hop h
    weight = np.bincount(codes, weights=hold, minlength=1 << 16)
    # exact Boltzmann weights by dense algebra over all half-filled states
    states = np.array([c for c in range(1 << 16) if bin(c).count("1") == 8])
    bits = ((states[:, None] >> np.arange(16)) & 1).astype(float)
    r = distance_matrix(L)
    with np.errstate(divide="ignore"):
        v = np.where(r > 0, 1.0 / r, 0.0)
    qv = bits - 0.5
    H = bits @ phi + 0.5 * np.einsum("si,ij,sj->s", qv, v, qv)
    assert H[5] == pytest.approx(hamiltonian(bits[5], phi, L))
    emp = weight[states] / weight.sum()
    assert weight.sum() == ends[-1] and weight[states].sum() == weight.sum()
    order = np.argsort(H)

    def binned_tv(temp):
        pi = np.exp(-(H - H.min()) / temp); pi /= pi.sum()
        b = np.minimum((np.cumsum(pi[order]) * 20).astype(int), 19)   # 20 energy bins of equal mass
        return 0.5 * np.abs(np.bincount(b, weights=emp[order], minlength=20)
                            - np.bincount(b, weights=pi[order], minlength=20)).sum(), pi

    tv, pi = binned_tv(T)
    assert tv < 0.01
    assert abs((emp * H).sum() - (pi * H).sum()) < 0.01  # mean energy
    top = np.argsort(pi)[-30:]                           # the 30 most probable states individually
    assert np.allclose(emp[top], pi[top], rtol=0.15)
    # power of the test: a 10 % error in the temperature is rejected by the same statistic
    assert binned_tv(1.1 * T)[0] > 0.03 and binned_tv(0.9 * T)[0] > 0.03


def test_chain_invariants(oracle_lib):
    """cg_run(a); cg_run(b) == cg_run(a+b); M only changes the iteration count (G8);
    t = attempts/Gamma; near-tie certificate O10 stays at zero."""
    kw = dict(T=0.05, E=0.01, seed=5)
    o1 = oracle_lib.Oracle(32, M=64, **kw); o1.run(700); o1.run(1300)
    o2 = oracle_lib.Oracle(32, M=4096, **kw); o2.run(2000)
    for x, y in zip(o1.hops(), o2.hops()):
        assert np.array_equal(x, y)
    n1, e1, t1, p1 = o1.state(); n2, e2, t2, p2 = o2.state()
    assert np.array_equal(n1, n2) and np.array_equal(e1, e2) and t1 == t2 and p1 == p2
    c1, c2 = o1.counters(), o2.counters()
    assert c1["attempts"] == c2["attempts"] and c1["iterations"] > c2["iterations"]
    assert t1 == c1["attempts"] / o1.tables()["Gamma"]
    a, i, j = o1.hops()
    assert np.all(np.diff(a.astype(np.int64)) > 0) and a[-1] + 1 == c1["attempts"]
    L = 32
    dx = [min_image(int(jj) % L - int(ii) % L, L) for ii, jj in zip(i, j)]
    assert p1 == sum(dx)
    assert o1.near_ties() == 0 and o1.exp_evaluations() > 0
    assert n1.sum() == 512


def test_apply_hops_reproduces_run(oracle_lib):
    o = oracle_lib.Oracle(16, T=0.1, seed=1, M=8); o.run(500)
    _, i, j = o.hops()
    s = oracle_lib.Oracle(16, T=0.1, seed=1, M=8); s.apply_hops(i, j)
    assert np.array_equal(o.state()[0], s.state()[0]) and np.array_equal(o.state()[1], s.state()[1])
    assert o.state()[3] == s.state()[3]


def test_near_tie_certificate_fires_inside_its_band_only(oracle_lib):
    """O10 / reading G10: an attempt that reaches the Metropolis factor with |u_a - exp(-dH/T)| <=
    2^-50 exp(-dH/T) must be counted, one a few times further away must not (a certificate with a
    wrong scale would be a silent no-op).  dH of a fixed uphill attempt on the 4x4 lattice comes from
    Eq.(1) by brute force; T is then tuned, ulp by ulp, so that exp(-dH/T) lands next to that
    attempt's own u_a (T only enters through this one division)."""
    L = 4
    base = oracle_lib.Oracle(L, T=0.5, E=0.0, seed=4242, M=4)
    n0, eps0, _, _ = base.state()
    phi = base.phi()
    inv = base.tables()["invr_k"]
    H0 = hamiltonian(n0, phi, L)
    found = None
    for a in range(200000):                      # an attempt with theta_ij = 1, dH > 0 and a mid-range u_a
        i, j, k, ud, ua = base.decode_attempt(a)
        if n0[i] != 1 or n0[j] != 0 or not 0.05 < ua < 0.6:
            continue
        m = n0.copy(); m[i] = 0; m[j] = 1
        if hamiltonian(m, phi, L) - H0 > 0.2:
            found = (a, i, j, k, ua)
            break
    assert found
    a, i, j, k, ua = found
    dE = (eps0[j] - eps0[i]) - inv[k]            # the oracle's operands (O7), E = 0; pinned against Eq.(1) below
    assert dE == pytest.approx(hamiltonian(m, phi, L) - H0, abs=1e-12)

    def p_of(T):
        return math.exp((-dE) / T)

    T = -dE / math.log(ua)                       # exp(-dE/T) = u_a up to rounding; walk T to the nearest ulp
    while p_of(T) < ua:
        T = np.nextafter(T, np.inf)
    while p_of(T) > ua:
        T = np.nextafter(T, -np.inf)
    cand = [np.nextafter(T, -np.inf), T, np.nextafter(T, np.inf), np.nextafter(np.nextafter(T, np.inf), np.inf)]
    T_in = min(cand, key=lambda t: abs(p_of(t) - ua))
    assert abs(p_of(T_in) - ua) <= 2.0 ** -52 * ua          # well inside the 2^-50 band
    T_out = T_in
    while abs(p_of(T_out) - ua) <= 2.0 ** -48 * ua:         # walk out of the band, but stay close
        T_out = np.nextafter(T_out, np.inf)
    assert 2.0 ** -48 * ua < abs(p_of(T_out) - ua) < 2.0 ** -44 * ua

    def ties_at(T):
        o = oracle_lib.Oracle(L, T=float(T), E=0.0, seed=4242, M=4)
        o.set_state(n0, a)                       # the next attempt evaluated is a
        o.run(1)
        first = int(o.hops(0, 1)[0][0])
        # count only what attempt a itself contributed: replay from a + 1 and subtract
        rest = 0
        if first != a:
            o2 = oracle_lib.Oracle(L, T=float(T), E=0.0, seed=4242, M=4)
            o2.set_state(n0, a + 1)
            o2.run(1)
            rest = o2.near_ties()
        return o.near_ties() - rest, o.exp_evaluations()

    inside, evals = ties_at(T_in)
    assert evals >= 1 and inside == 1
    outside, evals = ties_at(T_out)
    assert evals >= 1 and outside == 0
