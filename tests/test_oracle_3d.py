"""Pins for the cubic 3D lattice ("significantly more advantageous in 3D
than in 2D", "easily extended to higher dimensions"; reading G22 in DESIGN.md).

Same Hamiltonian (Eq.(1)), rates (Eq.(2)) and mixed algorithm
on N = L^3 sites, s = (z L + y) L + x.  Everything here is brute force in numpy / Python from those
definitions; nothing comes from the oracle's own tables.
"""
import math

import numpy as np
import pytest
from scipy import stats


def _coords(L):
    s = np.arange(L ** 3)
    return s // (L * L), (s // L) % L, s % L


def _dist3(L):
    """Euclidean minimum-image distances on the L^3 torus."""
    z, y, x = _coords(L)
    r2 = 0
    for c in (z, y, x):
        d = np.abs(c[:, None] - c[None, :])
        d = np.minimum(d, L - d)
        r2 = r2 + d * d
    return np.sqrt(r2.astype(float))


def _invr3(L):
    r = _dist3(L)
    with np.errstate(divide="ignore"):
        return np.where(r > 0, 1.0 / r, 0.0)


def _hamiltonian3(n, phi, v):
    """Eq.(1), E = 0: H = sum phi_i n_i + 1/2 sum_{i != j} (n_i - 1/2)(n_j - 1/2)/r_ij."""
    q = np.asarray(n, float) - 0.5
    return float(np.dot(phi, n) + 0.5 * q @ v @ q)


def _disc3(L):
    h = L // 2
    rng = range(-h + 1, h + 1)
    return sorted((dz * dz + dy * dy + dx * dx, dz, dy, dx) for dz in rng for dy in rng for dx in rng
                  if 0 < dz * dz + dy * dy + dx * dx <= h * h)


def _target(i, d, L):
    z, y, x = i // (L * L), (i // L) % L, i % L
    return (((z + d[1]) % L) * L + (y + d[2]) % L) * L + (x + d[3]) % L


def test_L4_cubic_tower_closed_form(oracle_lib):
    """PAPER.md:80 on the 4^3 torus with hops r <= L/2 = 2: 6 neighbours at r = 1, 12 at
    sqrt 2, 8 at sqrt 3 and 3 at r = 2 (the +-L/2 images coincide, tie -> +L/2, G3):
    S = 6 e^-2 + 12 e^-2sqrt2 + 8 e^-2sqrt3 + 3 e^-4, K = 29."""
    o = oracle_lib.Oracle(4, xi=1.0, T=0.5, seed=1, dim=3)
    t = o.tables()
    S = 6 * math.exp(-2.0) + 12 * math.exp(-2 * math.sqrt(2)) + 8 * math.exp(-2 * math.sqrt(3)) + 3 * math.exp(-4.0)
    assert t["K"] == 29 and o.N == 64
    assert t["S"] == pytest.approx(S, rel=1e-15)
    assert t["Gamma"] == pytest.approx(64 * S, rel=1e-15)
    assert t["cdf"][5] == pytest.approx(6 * math.exp(-2.0) / S, rel=1e-14)
    assert t["cdf"][17] == pytest.approx((6 * math.exp(-2.0) + 12 * math.exp(-2 * math.sqrt(2))) / S, rel=1e-14)
    assert t["cdf"][28] == 1.0
    d = list(zip(t["dz"], t["dy"], t["dx"]))
    # order (r2, dz, dy, dx); the r = L/2 entries once each, positive component
    assert d[:6] == [(-1, 0, 0), (0, -1, 0), (0, 0, -1), (0, 0, 1), (0, 1, 0), (1, 0, 0)]
    assert d[26:] == [(0, 0, 2), (0, 2, 0), (2, 0, 0)]


@pytest.mark.parametrize("L", [4, 6, 8])
def test_cubic_tables_against_definition(oracle_lib, L):
    o = oracle_lib.Oracle(L, xi=1.0, T=0.1, seed=3, dim=3)
    t = o.tables()
    disc = _disc3(L)
    assert t["K"] == len(disc)
    assert [tuple(int(v) for v in d) for d in zip(t["dz"], t["dy"], t["dx"])] == [d[1:] for d in disc]
    r = np.sqrt(np.array([d[0] for d in disc], float))
    assert np.array_equal(t["invr_k"], 1.0 / r)
    S = math.fsum(math.exp(-2.0 * x) for x in r)
    assert t["S"] == pytest.approx(S, rel=1e-13) and t["Gamma"] == pytest.approx(L ** 3 * S, rel=1e-13)
    cdf = t["cdf"]
    assert np.all(np.diff(cdf) >= 0) and cdf[-1] == 1.0
    assert np.allclose(np.diff(np.concatenate([[0.0], cdf])), np.exp(-2.0 * r) / S, rtol=0, atol=2e-15)
    # each ordered pair within range exactly once, its reverse exactly once
    i = (1 * L + 2) * L + 3
    js = [_target(i, d, L) for d in disc]
    assert len(set(js)) == len(js) and i not in js
    for j in js[:40]:
        assert [_target(j, d, L) for d in disc].count(i) == 1
    # minimum-image 1/r between arbitrary sites, also beyond L/2 (corners: r up to L sqrt3 / 2)
    v = _invr3(L)
    rng = np.random.default_rng(L)
    for a, b in rng.integers(0, L ** 3, (200, 2)):
        assert o.invr_sites(a, b) == v[a, b]
    assert o.invr_sites(0, ((L // 2) * L + L // 2) * L + L // 2) == 1.0 / math.sqrt(3 * (L // 2) ** 2)


@pytest.mark.parametrize("L,seed", [(4, 5), (6, 6)])
def test_cubic_local_energies_and_update(oracle_lib, L, seed):
    """eps_i = phi_i + sum_{j != i}(n_j - 1/2)/r_ij; sum eps = sum phi at half filling;
    after every executed hop the incremental update (G1) equals the definition."""
    o = oracle_lib.Oracle(L, T=0.3, E=0.05, seed=seed, M=8, dim=3)
    v = _invr3(L)
    phi = o.phi()
    n, eps, _, _ = o.state()
    assert n.sum() == L ** 3 // 2
    assert abs(phi.mean()) < 0.1 and np.all(np.abs(phi) <= 0.5)
    want = phi + v @ (n.astype(float) - 0.5)
    assert np.allclose(eps, want, rtol=0, atol=1e-12)
    assert abs(eps.sum() - phi.sum()) < 1e-10
    for _ in range(150):
        o.run(1)
        n, eps, _, _ = o.state()
        assert n.sum() == L ** 3 // 2
        assert np.allclose(eps, phi + v @ (n.astype(float) - 0.5), rtol=0, atol=1e-11)
    assert o.recompute_eps()[1] < 1e-11


def test_cubic_dH_equals_energy_difference(oracle_lib):
    """dH_ij = eps_j - eps_i - 1/r_ij - E dx_ij against H(after) - H(before) from
    Eq.(1) by brute force, for every allowed hop of a 4^3 state: the exact first-hop law
    P(i,j) = (1/N)(w_k/S) theta_ij min[1, exp(-dH/T)] / A (Eq.(2)) and <m> = 1/A."""
    L, T, E, R = 4, 0.4, 0.2, 12000
    o = oracle_lib.Oracle(L, T=T, E=E, seed=17, M=4, dim=3)
    n0 = o.state()[0].copy()
    phi, v = o.phi(), _invr3(L)
    disc = _disc3(L)
    w = np.array([math.exp(-2.0 * math.sqrt(d[0])) for d in disc])
    S = w.sum()
    H0 = _hamiltonian3(n0, phi, v)
    prob = {}
    for i in range(L ** 3):
        for k, d in enumerate(disc):
            j = _target(i, d, L)
            if n0[i] != 1 or n0[j] != 0:
                continue
            m = n0.copy(); m[i] = 0; m[j] = 1
            dH = _hamiltonian3(m, phi, v) - H0 - E * d[3]
            prob[(i, j)] = (1.0 / L ** 3) * (w[k] / S) * min(1.0, math.exp(-dH / T))
    A = sum(prob.values())
    counts, ms = {}, np.empty(R)
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
    assert stats.chisquare(obs_b, exp_b).pvalue > 1e-4
    assert abs(ms.mean() - 1 / A) < 5 * math.sqrt((1 - A) / A ** 2 / R)


def test_2x2x2_stationary_distribution_is_boltzmann(oracle_lib):
    """Detailed balance of Eq.(2) with the symmetric proposal on the smallest cubic
    lattice: L = 2, N = 8, the C(8,4) = 70 half-filled states, E = 0.  Attempt-weighted histogram
    against exp(-H/T)/Z with H from Eq.(1)."""
    L, T = 2, 0.35
    o = oracle_lib.Oracle(L, T=T, E=0.0, seed=77, M=4, dim=3)
    assert o.tables()["K"] == 3                      # (0,0,1), (0,1,0), (1,0,0): +-1 coincide, tie -> +1
    phi, v = o.phi(), _invr3(L)
    n = o.state()[0].astype(np.int64).copy()
    hops = 400000
    o.run(hops)
    a, i, j = o.hops()
    ends = a.astype(np.int64) + 1
    hold = np.diff(np.concatenate([[0], ends]))
    code = int((n * (1 << np.arange(8))).sum())
    delta = (1 << j.astype(np.int64)) - (1 << i.astype(np.int64))
    codes = code + np.concatenate([[0], np.cumsum(delta)[:-1]])
    weight = np.bincount(codes, weights=hold, minlength=256)
    states = np.array([c for c in range(256) if bin(c).count("1") == 4])
    bits = ((states[:, None] >> np.arange(8)) & 1).astype(float)
    H = np.array([_hamiltonian3(b, phi, v) for b in bits])
    emp = weight[states] / weight.sum()
    assert weight[states].sum() == weight.sum() == ends[-1]

    def tv(temp):
        pi = np.exp(-(H - H.min()) / temp); pi /= pi.sum()
        return 0.5 * np.abs(emp - pi).sum()

    assert tv(T) < 0.01
    assert tv(1.1 * T) > 0.03 and tv(0.9 * T) > 0.03     # power: a 10 % error in T is rejected


def test_cubic_proposal_frequencies_and_invariants(oracle_lib):
    """Proposal law Gamma^T_ij / Gamma: site uniform, displacement ~ w_k / S;
    run(a); run(b) == run(a+b); dP = sum of minimum-image dx along the field direction x."""
    L = 4
    o = oracle_lib.Oracle(L, T=0.2, E=0.1, seed=9, M=16, dim=3)
    disc = _disc3(L)
    w = np.array([math.exp(-2.0 * math.sqrt(d[0])) for d in disc]); w /= w.sum()
    R = 60000
    ks = np.zeros(len(disc)); sites = np.zeros(L ** 3)
    for a in range(R):
        i, j, k, ud, ua = o.decode_attempt(a)
        assert j == _target(i, disc[k], L) and 0 <= ud < 1 and 0 <= ua < 1
        ks[k] += 1; sites[i] += 1
    assert stats.chisquare(ks, w * R).pvalue > 1e-4
    assert stats.chisquare(sites, np.full(L ** 3, R / L ** 3)).pvalue > 1e-4
    o1 = oracle_lib.Oracle(6, T=0.1, E=0.05, seed=4, M=8, dim=3); o1.run(300); o1.run(500)
    o2 = oracle_lib.Oracle(6, T=0.1, E=0.05, seed=4, M=999, dim=3); o2.run(800)
    for x, y in zip(o1.hops(), o2.hops()):
        assert np.array_equal(x, y)
    assert np.array_equal(o1.state()[1], o2.state()[1]) and o1.state()[2:] == o2.state()[2:]
    _, i, j = o1.hops()
    dx = (j.astype(np.int64) % 6 - i.astype(np.int64) % 6) % 6
    dx = np.where(dx > 3, dx - 6, dx)
    assert o1.state()[3] == dx.sum()
    assert o1.near_ties() == 0


def test_2d_is_the_Lz_1_case(oracle_lib):
    """The 2D oracle is the Lz = 1 case of the same loops: dz = 0 everywhere and the 2D pins
    (tests/test_oracle_*.py) still hold; here only that the 3D entry point is a different lattice."""
    o2 = oracle_lib.Oracle(4, T=0.5, seed=1)
    assert np.all(o2.tables()["dz"] == 0) and o2.tables()["K"] == 10
    with pytest.raises(ValueError):
        oracle_lib.Oracle(5, dim=3)
