"""Pins for oracle steps O6-O8: local energies, dH_ij, the O(N) update."""
import numpy as np
import pytest

from physics_bruteforce import distance_matrix, hamiltonian, min_image


@pytest.mark.parametrize("L", [4, 6, 8, 16])
def test_eps_matches_its_definition(oracle_lib, L):
    """eps_i = phi_i + sum_{j != i} (n_j - nu)/r_ij, by dense numpy."""
    o = oracle_lib.Oracle(L, seed=21 + L)
    n, eps, _, _ = o.state()
    r = distance_matrix(L)
    with np.errstate(divide="ignore"):
        v = np.where(r > 0, 1.0 / r, 0.0)
    want = o.phi() + v @ (n.astype(float) - 0.5)
    assert np.allclose(eps, want, rtol=0, atol=1e-12)


@pytest.mark.parametrize("L", [8, 16, 32])
def test_sum_of_eps_equals_sum_of_phi_at_half_filling(oracle_lib, L):
    """sum_i eps_i = sum_i phi_i + sum_j (n_j - 1/2) sum_i 1/r_ij, and sum_i 1/r_ij is the same
    for every j on the torus, so the second term vanishes when sum_j n_j = N/2."""
    o = oracle_lib.Oracle(L, seed=5)
    _, eps, _, _ = o.state()
    assert abs(eps.sum() - o.phi().sum()) < 1e-9
    o.run(500)
    assert abs(o.state()[1].sum() - o.phi().sum()) < 1e-9


def test_H_from_eps(oracle_lib):
    """Eq.(1) at E=0: H = sum phi_i n_i + 1/2 sum_i (n_i - 1/2)(eps_i - phi_i)."""
    L = 8
    o = oracle_lib.Oracle(L, seed=8)
    n, eps, _, _ = o.state()
    phi = o.phi()
    H = hamiltonian(n, phi, L)
    assert H == pytest.approx(np.dot(phi, n) + 0.5 * np.dot(n - 0.5, eps - phi), abs=1e-11)


def test_checkerboard_is_antisymmetric(oracle_lib):
    """phi = 0 and a checkerboard: the lattice maps onto itself with n -> 1-n under a unit shift,
    so eps on occupied sites is minus eps on empty sites, and all occupied sites are equal."""
    L = 8
    o = oracle_lib.Oracle(L, W=0.0, seed=1)
    s = np.arange(L * L)
    n = (((s // L) + (s % L)) % 2).astype(np.int8)
    o.set_state(n)
    _, eps, _, _ = o.state()
    assert np.allclose(eps[n == 1], -eps[n == 0][0], atol=1e-13)
    assert np.ptp(eps[n == 1]) < 1e-13 and eps[n == 1][0] < 0    # occupied sites sit in a well


@pytest.mark.parametrize("L", [4, 6, 8])
def test_dH_from_eps_equals_H_difference_for_every_allowed_hop(oracle_lib, L):
    """dH_ij = eps_j - eps_i - 1/r_ij (E=0) against H(after) - H(before), Eq.(1)."""
    o = oracle_lib.Oracle(L, seed=31 + L)
    n, eps, _, _ = o.state()
    phi = o.phi()
    t = o.tables()
    H0 = hamiltonian(n, phi, L)
    checked = 0
    for i in np.flatnonzero(n == 1):
        yi, xi = divmod(int(i), L)
        for k in range(t["K"]):
            j = ((yi + int(t["dy"][k])) % L) * L + (xi + int(t["dx"][k])) % L
            if n[j] != 0:
                continue
            m = n.copy(); m[i] = 0; m[j] = 1
            dH = eps[j] - eps[i] - t["invr_k"][k]
            assert dH == pytest.approx(hamiltonian(m, phi, L) - H0, abs=5e-13)
            checked += 1
    assert checked > 30


def test_update_rule_after_every_hop(oracle_lib):
    """Step 3b (reading G1): the incremental eps equals the definition after
    every executed hop; n keeps sum N/2; dP accumulates the minimum-image dx."""
    L = 8
    o = oracle_lib.Oracle(L, T=0.3, E=0.2, seed=77, M=4)
    r = distance_matrix(L)
    with np.errstate(divide="ignore"):
        v = np.where(r > 0, 1.0 / r, 0.0)
    phi = o.phi()
    n_prev, _, _, dP_prev = o.state()
    for h in range(300):
        o.run(1)
        n, eps, _, dP = o.state()
        a, i, j = o.hops(h, 1)
        i, j = int(i[0]), int(j[0])
        assert n_prev[i] == 1 and n_prev[j] == 0 and n[i] == 0 and n[j] == 1
        changed = np.flatnonzero(n != n_prev)
        assert sorted(changed) == sorted([i, j]) and n.sum() == L * L // 2
        assert np.allclose(eps, phi + v @ (n - 0.5), rtol=0, atol=1e-12)
        assert dP - dP_prev == min_image(j % L - i % L, L)
        n_prev, dP_prev = n, dP
    _, dev = o.recompute_eps()
    assert dev < 1e-12


def test_drift_of_incremental_eps_stays_small_on_long_runs(oracle_lib):
    o = oracle_lib.Oracle(32, T=0.1, E=0.01, seed=4, M=64)
    o.run(20000)
    _, dev = o.recompute_eps()
    assert dev < 1e-10
    assert o.state()[0].sum() == 512


def test_field_term_sign_and_size(oracle_lib):
    """dH = ... - E dx: with E > 0 hops with dx > 0 are favoured, so dP drifts
    positive (reading G14); the accept decision of single attempts is reproduced from eps."""
    L = 16
    o = oracle_lib.Oracle(L, T=0.2, E=0.5, seed=3, M=8)
    t = o.tables()
    T, E = 0.2, 0.5
    # replay the first 3000 attempts by hand from the oracle's own eps/n but independent arithmetic
    n, eps, _, _ = o.state()
    n = n.copy(); eps = eps.copy()
    o.run(40)
    a_log, i_log, j_log = o.hops()
    hop_at = {int(a): (int(i), int(j)) for a, i, j in zip(a_log, i_log, j_log)}
    r = distance_matrix(L)
    with np.errstate(divide="ignore"):
        v = np.where(r > 0, 1.0 / r, 0.0)
    for a in range(int(a_log[-1]) + 1):
        i, j, k, ud, ua = o.decode_attempt(a)
        acc = False
        if n[i] == 1 and n[j] == 0:
            dx = int(t["dx"][k])
            assert dx == min_image(j % L - i % L, L)
            dE = eps[j] - eps[i] - v[i, j] - E * dx
            acc = dE <= 0 or ua < np.exp(-dE / T)
        assert acc == (a in hop_at), a
        if acc:
            assert hop_at[a] == (i, j)
            n[i], n[j] = 0, 1
            eps += v[:, j] - v[:, i]
    o2 = oracle_lib.Oracle(L, T=0.2, E=0.5, seed=3, M=8)
    o2.run(5000)
    assert o2.state()[3] > 500          # strong field: clear positive drift


def test_half_lattice_hops_count_as_plus_half_L(oracle_lib):
    """Reading G3: a hop of exactly L/2 along x has dx = +L/2 (components in (-L/2, L/2]);
    on the 4x4 lattice such hops are frequent enough to pin the dP bookkeeping."""
    L = 4
    o = oracle_lib.Oracle(L, T=5.0, E=0.0, seed=12, M=2)
    o.run(3000)
    _, i, j = o.hops()
    dx = np.array([min_image(int(b) % L - int(a) % L, L) for a, b in zip(i, j)])
    assert (dx == 2).sum() > 10 and (dx == -2).sum() == 0
    assert o.state()[3] == dx.sum()
