"""Pins for oracle steps O2-O5 (disorder, occupations, displacement list, tower, Gamma)."""
import math

import numpy as np
import pytest


def _disc(L):
    h = L // 2
    return sorted((dy * dy + dx * dx, dy, dx) for dy in range(-h + 1, h + 1)
                  for dx in range(-h + 1, h + 1) if 0 < dy * dy + dx * dx <= h * h)


def test_L4_tower_closed_form(oracle_lib):
    """Gamma = N sum_j Gamma^T_ij, Gamma^T = exp(-2r/xi).
    On the 4x4 torus with hops r <= L/2 a site has 4 neighbours at r=1,
    4 at sqrt(2) and 2 at r=2 (the +-L/2 images coincide): S = 4e^-2 + 4e^-2sqrt2 + 2e^-4."""
    o = oracle_lib.Oracle(4, xi=1.0, T=0.5, seed=1)
    t = o.tables()
    S = 4 * math.exp(-2.0) + 4 * math.exp(-2.0 * math.sqrt(2.0)) + 2 * math.exp(-4.0)
    assert t["K"] == 10
    assert t["S"] == pytest.approx(S, rel=1e-15)
    assert t["Gamma"] == pytest.approx(16 * S, rel=1e-15)
    c = [4 * math.exp(-2.0) / S, (4 * math.exp(-2.0) + 4 * math.exp(-2 * math.sqrt(2))) / S, 1.0]
    assert t["cdf"][3] == pytest.approx(c[0], rel=1e-14)
    assert t["cdf"][7] == pytest.approx(c[1], rel=1e-14)
    assert t["cdf"][9] == 1.0
    # list order (r2, dy, dx), r = L/2 entries once each with the positive component
    assert list(zip(t["dy"], t["dx"])) == [(-1, 0), (0, -1), (0, 1), (1, 0), (-1, -1), (-1, 1),
                                           (1, -1), (1, 1), (0, 2), (2, 0)]
    xi2 = oracle_lib.Oracle(4, xi=2.0, T=0.5, seed=1).tables()
    assert xi2["S"] == pytest.approx(4 * math.exp(-1.0) + 4 * math.exp(-math.sqrt(2.0)) + 2 * math.exp(-2.0),
                                     rel=1e-15)


@pytest.mark.parametrize("L", [4, 6, 16, 64])
def test_tables_against_definition(oracle_lib, L):
    o = oracle_lib.Oracle(L, xi=1.0, T=0.1, seed=3)
    t = o.tables()
    disc = _disc(L)
    assert t["K"] == len(disc)
    assert [(int(a), int(b)) for a, b in zip(t["dy"], t["dx"])] == [(dy, dx) for _, dy, dx in disc]
    r = np.sqrt(np.array([r2 for r2, _, _ in disc], float))
    assert np.array_equal(t["invr_k"], 1.0 / r)
    S = math.fsum(math.exp(-2.0 * x) for x in r)
    assert t["S"] == pytest.approx(S, rel=1e-13)
    assert t["Gamma"] == pytest.approx(L * L * S, rel=1e-13)
    cdf = t["cdf"]
    assert np.all(np.diff(cdf) >= 0) and cdf[-1] == 1.0 and cdf[0] > 0
    assert np.allclose(np.diff(np.concatenate([[0.0], cdf])), np.exp(-2.0 * r) / S, rtol=0, atol=2e-15)
    # every ordered pair (i, j) within range exactly once, and its reverse exactly once
    i = 1 * L + 2
    yi, xi = divmod(i, L)
    js = [((yi + dy) % L) * L + (xi + dx) % L for _, dy, dx in disc]
    assert len(set(js)) == len(js) and i not in js
    for j in js[:50]:
        yj, xj = divmod(j, L)
        back = [((yj + dy) % L) * L + (xj + dx) % L for _, dy, dx in disc]
        assert back.count(i) == 1


def test_K_values_of_the_configs(oracle_lib):
    # lattice points with 0 < r <= L/2 counted independently
    for L in (16, 64):
        h = L // 2
        yy, xx = np.mgrid[-h + 1:h + 1, -h + 1:h + 1]
        r2 = yy * yy + xx * xx
        assert oracle_lib.Oracle(L, seed=1).tables()["K"] == int(((r2 > 0) & (r2 <= h * h)).sum())


def test_invr_is_minimum_image_coulomb(oracle_lib):
    """r_ij = Euclidean minimum-image distance."""
    L = 8
    o = oracle_lib.Oracle(L, seed=5)
    for a in range(0, L * L, 5):
        for b in range(L * L):
            ya, xa = divmod(a, L); yb, xb = divmod(b, L)
            dy = min(abs(ya - yb), L - abs(ya - yb)); dx = min(abs(xa - xb), L - abs(xa - xb))
            want = 0.0 if a == b else 1.0 / math.sqrt(dy * dy + dx * dx)
            assert o.invr_sites(a, b) == want
            assert o.invr_sites(a, b) == o.invr_sites(b, a)


@pytest.mark.parametrize("L,W", [(16, 1.0), (64, 1.0), (32, 2.0)])
def test_disorder_and_half_filling(oracle_lib, L, W):
    """phi ~ U[-W/2, W/2) iid (PAPER.md:52 with reading G2), sum_i n_i = N/2."""
    o = oracle_lib.Oracle(L, W=W, seed=11)
    phi = o.phi()
    n, _, t, dP = o.state()
    N = L * L
    assert n.sum() == N // 2 and set(np.unique(n)) <= {0, 1}
    assert phi.min() >= -W / 2 and phi.max() < W / 2
    assert abs(phi.mean()) < 5 * W / math.sqrt(12 * N)
    assert abs(phi.var() - W * W / 12) < 5 * W * W * math.sqrt(1 / 180 / N)
    assert t == 0.0 and dP == 0
    # different seeds give different realisations, same seed the same one
    o2 = oracle_lib.Oracle(L, W=W, seed=11)
    o3 = oracle_lib.Oracle(L, W=W, seed=12)
    assert np.array_equal(o2.phi(), phi) and np.array_equal(o2.state()[0], n)
    assert not np.array_equal(o3.phi(), phi) and not np.array_equal(o3.state()[0], n)
    # occupation is not correlated with the potential (random initial configuration)
    assert abs(np.corrcoef(phi, n)[0, 1]) < 5 / math.sqrt(N)


def test_rejects_bad_arguments(oracle_lib):
    for kw in (dict(L=5), dict(L=0), dict(L=16, T=0.0), dict(L=16, xi=0.0), dict(L=16, M=0)):
        args = dict(L=16, T=0.1, xi=1.0, M=4)
        args.update(kw)
        with pytest.raises(ValueError):
            oracle_lib.Oracle(args.pop("L"), **args)
