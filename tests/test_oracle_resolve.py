"""Pins for the oracle's close-encounter resolution (the paper's mdt_hkce, PAPER.md:104
fn. 14, 126, 297-315; readings X-1..X-5) - no GPU.  Independent references: the pinned Kepler drift (no
interaction left => pure two-body motion), scipy's DOP853 on the same equations of motion written with the
pinned changeover function, time reversal, and the energy budget of the whole hybrid step."""
import math

import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle
from paper_2601_19654_b200 import workloads as W

G = W.G_AU_DAY_MSUN


def _relv(got, ref):
    return float((np.max(np.abs(got - ref), axis=0) / np.linalg.norm(ref, axis=0)).max())


def _encounter_system(sep=0.01, m=1e-5, extra=3, seed=5):
    """star + two bodies of mass m on neighbouring orbits at 1 AU, `sep` apart, + `extra` bystanders"""
    M = 1.0
    a = np.array([1.0, 1.0 + 0.6 * sep] + [1.7 + 0.4 * k for k in range(extra)])
    n = len(a)
    e = np.array([0.01, 0.012] + [0.05] * extra)
    inc = np.array([0.001, 0.002] + [0.01] * extra)
    Om = np.zeros(n); om = np.zeros(n)
    Man = np.array([0.3, 0.3 + 0.8 * sep] + [1.0 + k for k in range(extra)])
    mass = np.array([m, m] + [1e-7] * extra)
    x, vh = W.elements_to_state(G * (M + mass), a, e, inc, Om, om, Man)
    v = oracle.h2dh(M, mass, vh)
    rh, rc = oracle.hill(G, M, mass, x, v, n_hill=3.0)
    return M, mass, x, v, rc


def test_X1_without_interaction_it_is_the_kepler_drift():
    w = W.make_config(0)
    mu, gm = G * w.m_star, G * w.mass
    x1, v1, fl = oracle.drift(mu, w.dt, w.x, w.v)
    enc = oracle.encounters(w.dt, w.x, w.v, x1, v1, w.rcrit)
    assert enc["count"] >= 4
    idx = np.unique(enc["pairs"])
    # massless bodies: nothing but the star's Kepler term is left
    r = oracle.resolve(mu, gm * 0.0, w.rcrit, w.dt, w.x, w.v, x1, v1, enc["pairs"])
    assert r["fail"] == 0 and r["n"] == len(idx)
    assert _relv(r["x"][:, idx], x1[:, idx]) <= 1e-12 and _relv(r["v"][:, idx], v1[:, idx]) <= 1e-12
    # rcrit -> 0: every listed pair is outside its shell, 1 - K = 0
    r = oracle.resolve(mu, gm, w.rcrit * 1e-9, w.dt, w.x, w.v, x1, v1, enc["pairs"])
    assert _relv(r["x"][:, idx], x1[:, idx]) <= 1e-12 and _relv(r["v"][:, idx], v1[:, idx]) <= 1e-12
    # bodies outside the list keep the drift result bit for bit; empty list: nothing changes
    r = oracle.resolve(mu, gm, w.rcrit, w.dt, w.x, w.v, x1, v1, enc["pairs"])
    rest = np.setdiff1d(np.arange(w.nb), idx)
    assert np.array_equal(r["x"][:, rest], x1[:, rest]) and np.array_equal(r["v"][:, rest], v1[:, rest])
    assert not np.array_equal(r["x"][:, idx], x1[:, idx])
    r = oracle.resolve(mu, gm, w.rcrit, w.dt, w.x, w.v, x1, v1, np.zeros((0, 2), dtype=np.int32))
    assert np.array_equal(r["x"], x1) and r["n"] == 0


@pytest.mark.parametrize("sep,h", [(0.01, 2.0), (0.003, 1.0), (0.02, -3.0), (0.0009, 0.5)])
def test_X2_against_dop853_on_the_same_equations(sep, h):
    """sep = 0.01, 0.02: inside the changeover shell (0 < K < 1); 0.003, 0.0009: partly / wholly inside 0.1 rc"""
    M, mass, x, v, rc = _encounter_system(sep)
    mu, gm = G * M, G * mass
    pairs = np.array([[0, 1], [0, 3], [1, 4]], dtype=np.int32)       # the close pair + two distant listed pairs
    idx = np.unique(pairs)
    loc = {b: k for k, b in enumerate(idx)}
    n = len(idx)

    def rhs(t, y):
        X = y[:3 * n].reshape(n, 3); V = y[3 * n:].reshape(n, 3)
        A = -mu * X / np.linalg.norm(X, axis=1)[:, None] ** 3
        for i, j in pairs:
            d = X[loc[j]] - X[loc[i]]
            r = np.linalg.norm(d)
            u = (1.0 - oracle.changeover(r, max(rc[i], rc[j]))) / r**3
            A[loc[i]] += gm[j] * u * d
            A[loc[j]] -= gm[i] * u * d
        return np.concatenate([V.ravel(), A.ravel()])

    y0 = np.concatenate([x[:, idx].T.ravel(), v[:, idx].T.ravel()])
    sol = solve_ivp(rhs, (0.0, h), y0, method="DOP853", rtol=1e-13, atol=1e-18)
    assert sol.success
    xr = sol.y[:3 * n, -1].reshape(n, 3).T; vr = sol.y[3 * n:, -1].reshape(n, 3).T
    x1, v1, _ = oracle.drift(mu, h, x, v)
    r = oracle.resolve(mu, gm, rc, h, x, v, x1, v1, pairs, tol=1e-13)
    assert r["fail"] == 0 and r["n"] == n
    assert _relv(r["x"][:, idx], xr) <= 2e-11 and _relv(r["v"][:, idx], vr) <= 2e-11
    # and the encounter matters: the close pair does not follow its Kepler drift
    assert _relv(r["v"][:, :2], v1[:, :2]) > 1e-7


def test_X3_time_reversal_and_pair_order():
    M, mass, x, v, rc = _encounter_system(0.008)
    mu, gm = G * M, G * mass
    pairs = np.array([[0, 1], [1, 2]], dtype=np.int32)
    x1, v1, _ = oracle.drift(mu, 2.0, x, v)
    f = oracle.resolve(mu, gm, rc, 2.0, x, v, x1, v1, pairs)
    b = oracle.resolve(mu, gm, rc, -2.0, f["x"], f["v"], f["x"], f["v"], pairs)
    idx = np.unique(pairs)
    assert _relv(b["x"][:, idx], x[:, idx]) <= 1e-11 and _relv(b["v"][:, idx], v[:, idx]) <= 1e-11
    g = oracle.resolve(mu, gm, rc, 2.0, x, v, x1, v1, pairs[::-1].copy())
    assert _relv(g["x"][:, idx], f["x"][:, idx]) <= 1e-15


def _hybrid_steps(M, mass, x, v, rc, dt, nsteps, resolve):
    """the hybrid step composed from the oracle's pinned parts (S-1), with or without X-1..X-5"""
    mu, gm = G * M, G * mass
    a, _ = oracle.accel(gm, x, rc)
    nres = 0
    for _ in range(nsteps):
        v = oracle.kick(0.5 * dt, v, a)
        x, _ = oracle.jump(0.5 * dt, mu, gm, x, v)
        x0, v0 = x.copy(), v.copy()
        x, v, _ = oracle.drift(mu, dt, x, v)
        enc = oracle.encounters(dt, x0, v0, x, v, rc)
        if resolve and enc["count"] > 0:
            r = oracle.resolve(mu, gm, rc, dt, x0, v0, x, v, enc["pairs"])
            assert r["fail"] == 0
            x, v = r["x"], r["v"]
            nres += 1
        x, _ = oracle.jump(0.5 * dt, mu, gm, x, v)
        a, _ = oracle.accel(gm, x, rc)
        v = oracle.kick(0.5 * dt, v, a)
    return x, v, nres


def test_X4_the_resolved_hybrid_step_keeps_the_energy_through_a_close_encounter():
    """inside the shell the kick carries only K of the pair force; the encounter solve must supply the rest"""
    M, mass, x, v, rc = _encounter_system(sep=0.004, m=3e-5, extra=2)
    E0 = oracle.energy(G, M, mass, x, v)["E"]
    xa, va, nres = _hybrid_steps(M, mass, x, v, rc, 1.0, 30, resolve=True)
    xb, vb, _ = _hybrid_steps(M, mass, x, v, rc, 1.0, 30, resolve=False)
    ea = abs(oracle.energy(G, M, mass, xa, va)["E"] - E0) / abs(E0)
    eb = abs(oracle.energy(G, M, mass, xb, vb)["E"] - E0) / abs(E0)
    assert nres >= 20
    assert ea < 1e-7 and eb > 100 * ea, (ea, eb)


def _multi_component_system():
    """star + seven massive bodies forming THREE encounter components whose members interleave in body order:
    pair A = (0, 3) at 1 AU, pair B = (1, 5) at 1.6 AU, chain C = (2, 4), (4, 6) at 2.3 AU; + 2 bystanders.
    The sorted list (0,3), (1,5), (2,4), (4,6) alternates between the components."""
    M = 1.0
    sepA, sepB, sepC = 0.006, 0.004, 0.005
    a = np.empty(9); Man = np.empty(9)
    a[[0, 3]] = [1.0, 1.0 + 0.6 * sepA]; Man[[0, 3]] = [0.3, 0.3 + 0.8 * sepA]
    a[[1, 5]] = [1.6, 1.6 + 0.6 * sepB]; Man[[1, 5]] = [2.1, 2.1 + 0.8 * sepB / 1.6]
    a[[2, 4, 6]] = [2.3, 2.3 + 0.6 * sepC, 2.3 + 1.2 * sepC]; Man[[2, 4, 6]] = [4.0, 4.0 + 0.8 * sepC / 2.3, 4.0 + 1.7 * sepC / 2.3]
    a[7:] = [3.1, 3.7]; Man[7:] = [1.0, 5.0]
    e = np.array([0.01, 0.02, 0.015, 0.012, 0.018, 0.022, 0.013, 0.05, 0.05])
    inc = np.array([0.001, 0.003, 0.002, 0.002, 0.001, 0.004, 0.003, 0.01, 0.01])
    z = np.zeros(9)
    mass = np.array([1e-5, 2e-5, 1.5e-5, 1.2e-5, 0.8e-5, 1e-5, 2.5e-5, 1e-7, 1e-7])
    x, vh = W.elements_to_state(G * (M + mass), a, e, inc, z, z, Man)
    v = oracle.h2dh(M, mass, vh)
    _, rc = oracle.hill(G, M, mass, x, v, n_hill=3.0)
    pairs = np.array([[0, 3], [1, 5], [2, 4], [4, 6]], dtype=np.int32)
    return M, mass, x, v, rc, pairs


@pytest.mark.parametrize("h", [2.0, -1.5])
def test_X1_several_interacting_components_against_dop853_on_the_union_system(h):
    """Pins the union-find split of oracle_resolve (reading X-1): three components with non-zero masses, interleaved
    in the list, against ONE DOP853 integration of all listed bodies under all listed pairs (the paper's single call
    for 'the bodies involved in the close encounter', PAPER.md:104 fn. 14).  A pair put into the wrong component, or
    dropped, changes the states by ~1e-6, nine orders above the tolerance."""
    M, mass, x, v, rc, pairs = _multi_component_system()
    mu, gm = G * M, G * mass
    idx = np.unique(pairs)
    loc = {b: k for k, b in enumerate(idx)}
    n = len(idx)
    # every listed pair is inside its changeover shell: the encounter terms are really there
    for i, j in pairs:
        r = np.linalg.norm(x[:, j] - x[:, i])
        assert oracle.changeover(r, max(rc[i], rc[j])) < 0.9

    def rhs(t, y):
        X = y[:3 * n].reshape(n, 3); V = y[3 * n:].reshape(n, 3)
        A = -mu * X / np.linalg.norm(X, axis=1)[:, None] ** 3
        for i, j in pairs:
            d = X[loc[j]] - X[loc[i]]
            r = np.linalg.norm(d)
            u = (1.0 - oracle.changeover(r, max(rc[i], rc[j]))) / r**3
            A[loc[i]] += gm[j] * u * d
            A[loc[j]] -= gm[i] * u * d
        return np.concatenate([V.ravel(), A.ravel()])

    y0 = np.concatenate([x[:, idx].T.ravel(), v[:, idx].T.ravel()])
    sol = solve_ivp(rhs, (0.0, h), y0, method="DOP853", rtol=1e-13, atol=1e-18)
    assert sol.success
    xr = sol.y[:3 * n, -1].reshape(n, 3).T; vr = sol.y[3 * n:, -1].reshape(n, 3).T
    x1, v1, _ = oracle.drift(mu, h, x, v)
    r = oracle.resolve(mu, gm, rc, h, x, v, x1, v1, pairs, tol=1e-13)
    assert r["fail"] == 0 and r["n"] == n
    assert _relv(r["x"][:, idx], xr) <= 2e-11 and _relv(r["v"][:, idx], vr) <= 2e-11
    # every one of the seven bodies felt its encounter (none was left to the drift by a wrong split) ...
    for b in idx:
        assert np.linalg.norm(r["v"][:, b] - v1[:, b]) / np.linalg.norm(v1[:, b]) > 1e-8, b
    # ... the bystanders did not move off the drift, and the list order does not matter
    assert np.array_equal(r["x"][:, 7:], x1[:, 7:]) and np.array_equal(r["v"][:, 7:], v1[:, 7:])
    g = oracle.resolve(mu, gm, rc, h, x, v, x1, v1, pairs[[2, 0, 3, 1]].copy(), tol=1e-13)
    assert _relv(g["x"][:, idx], r["x"][:, idx]) <= 1e-13 and _relv(g["v"][:, idx], r["v"][:, idx]) <= 1e-13
    # dropping the chain's second pair (what a wrong split would amount to for body 6) is far outside the tolerance
    bad = oracle.resolve(mu, gm, rc, h, x, v, x1, v1, pairs[:3].copy(), tol=1e-13)
    assert np.linalg.norm(bad["v"][:, 4] - r["v"][:, 4]) / np.linalg.norm(r["v"][:, 4]) > 1e-9


def test_X6_massless_bodies_can_be_integrated_apart():
    """Reading X-6 (the kernel detaches massless bodies): a massless body exerts no force, so integrating every test
    particle in a system of its own with its massive partners gives the states of integrating the whole component
    together - shown here on the ORACLE alone (joint call vs one call per test particle), to the tolerance."""
    M = 1.0
    K = 6
    rng = np.random.default_rng(7)
    xg = np.array([5.2, 0.0, 0.0])
    rad = rng.uniform(0.05, 0.6, K); ang = rng.uniform(0, 2 * np.pi, K)
    X = np.empty((3, K + 2)); X[:, 0] = xg; X[:, 1] = xg + np.array([0.25, 0.1, 0.0])
    X[0, 2:] = xg[0] + rad * np.cos(ang); X[1, 2:] = xg[1] + rad * np.sin(ang); X[2, 2:] = rng.uniform(-0.01, 0.01, K)
    r = np.linalg.norm(X, axis=0)
    vc = np.sqrt(G * M / r)
    Vh = np.stack([-vc * X[1] / r, vc * X[0] / r, np.zeros(K + 2)])
    mass = np.concatenate([[1e-3, 3e-6], np.zeros(K)])            # a giant, an embryo next to it, K test particles
    V = oracle.h2dh(M, mass, Vh)
    _, rc = oracle.hill(G, M, mass, X, V, n_hill=3.0)
    mu, gm, h = G * M, G * mass, 6.0
    x1, v1, _ = oracle.drift(mu, h, X, V)
    pairs = np.array([[0, 1]] + [[0, k] for k in range(2, K + 2)] + [[1, 2], [1, 3]], dtype=np.int32)
    pairs = pairs[np.lexsort((pairs[:, 1], pairs[:, 0]))]
    joint = oracle.resolve(mu, gm, rc, h, X, V, x1, v1, pairs, tol=1e-13)
    assert joint["fail"] == 0 and joint["n"] == K + 2
    core = np.array([[0, 1]], dtype=np.int32)
    alone = oracle.resolve(mu, gm, rc, h, X, V, x1, v1, core, tol=1e-13)          # the massive bodies by themselves
    assert _relv(alone["x"][:, :2], joint["x"][:, :2]) <= 1e-12 and _relv(alone["v"][:, :2], joint["v"][:, :2]) <= 1e-12
    for k in range(2, K + 2):                                                    # every test particle with the core
        own = pairs[(pairs[:, 1] == k)]
        sub = np.concatenate([core, own]); sub = sub[np.lexsort((sub[:, 1], sub[:, 0]))]
        one = oracle.resolve(mu, gm, rc, h, X, V, x1, v1, sub, tol=1e-13)
        assert _relv(one["x"][:, [k]], joint["x"][:, [k]]) <= 1e-11 and _relv(one["v"][:, [k]], joint["v"][:, [k]]) <= 1e-11, k
        assert np.linalg.norm(one["v"][:, k] - v1[:, k]) / np.linalg.norm(v1[:, k]) > 1e-8       # the encounter matters
