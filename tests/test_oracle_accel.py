"""Pins for the oracle's acceleration (O-A) - no GPU.  Each pin is something the
definitions fix independently of oracle/mopal_oracle.c."""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2601_19654_b200 import workloads as W
from tests import mp_reference as R

G = W.G_AU_DAY_MSUN


@pytest.mark.parametrize("nb,seed", [(2, 11), (3, 12), (5, 13), (8, 14), (8, 15)])
def test_PA1_bruteforce_mpmath(nb, seed):
    w = W.random_cluster(nb, seed)
    gm = G * w.mass
    a, S = oracle.accel(gm, w.x, w.rcrit)
    a_mp, S_mp = R.accel_mp(gm, w.x, w.rcrit)
    shells = 0
    for i in range(nb):
        for c in range(3):
            err = abs(mp.mpf(float(a[c, i])) - a_mp[i][c])
            assert err <= mp.mpf(2e-16) * S_mp[i][c] + mp.mpf(1e-300), (i, c, err)
            assert abs(mp.mpf(float(S[c, i])) - S_mp[i][c]) <= mp.mpf(1e-15) * S_mp[i][c] + mp.mpf(1e-300)
    # the sample really covers inside / across / outside the changeover shell
    d = np.linalg.norm(w.x[:, :, None] - w.x[:, None, :], axis=0)
    rc = np.maximum(w.rcrit[:, None], w.rcrit[None, :])
    iu = np.triu_indices(nb, 1)
    if nb == 8:
        assert (d[iu] >= rc[iu]).any() and ((d[iu] < rc[iu]) & (d[iu] > 0.1 * rc[iu])).any()


def test_PA1_inside_inner_shell_is_zero():
    x = np.array([[0.0, 0.05], [0.0, 0.0], [0.0, 0.0]])
    a, S = oracle.accel(np.array([1e-3, 2e-3]) * G, x, np.array([1.0, 0.2]))
    assert np.all(a == 0.0) and np.all(S == 0.0)


@pytest.mark.parametrize("cfg,N", [(0, 256), (2, 300), (4, 257)])
def test_PA2_newton_third_law(cfg, N):
    w = W.shrink(cfg, N)
    # make some pairs fall in the changeover shell so that K_ij symmetry is exercised
    rcrit = w.rcrit * 40.0
    gm = G * w.mass
    a, S = oracle.accel(gm, w.x, rcrit)
    for c in range(3):
        tot = math.fsum(w.mass * a[c])
        ref = math.fsum(w.mass * S[c])
        assert abs(tot) <= 1e-14 * ref
    d = np.linalg.norm(w.x[:, :, None] - w.x[:, None, :], axis=0) + np.eye(w.nb) * 1e9
    rc = np.maximum(rcrit[:, None], rcrit[None, :])
    assert ((d < rc) & (d > 0.1 * rc)).sum() > 0


@pytest.mark.parametrize("n", [3, 7, 64])
def test_PA3_ring_closed_form(n):
    Rr, m = 2.5, 3.0e-7
    th = 2 * np.pi * np.arange(n) / n + 0.3
    x = np.stack([Rr * np.cos(th), Rr * np.sin(th), np.zeros(n)])
    a, _ = oracle.accel(np.full(n, G * m), x, np.zeros(n))
    mag = (G * m / (4 * Rr * Rr)) * sum(1.0 / math.sin(math.pi * k / n) for k in range(1, n))
    for b in range(n):
        want = -mag * x[:, b] / Rr
        # vertex coordinates are rounded to double: the nearest-neighbour terms amplify that
        # input rounding by ~R/d_min, hence the looser bound at n=64
        assert np.allclose(a[:, b], want, rtol=0, atol=(2e-15 if n <= 7 else 1e-13) * mag)
    if n == 7:  # unit-radius variant
        x1 = np.stack([np.cos(th), np.sin(th), np.zeros(n)])
        a1, _ = oracle.accel(np.full(n, G * 1.0e-6), x1, np.zeros(n))
        want = (G * 1.0e-6 / 4) * sum(1.0 / math.sin(math.pi * k / 7) for k in range(1, 7))
        assert abs(np.linalg.norm(a1[:, 0]) - want) <= 1e-15 * want


def test_PA4_K_is_the_unique_C2_quintic():
    """K(0.1rc)=0, K(rc)=1, K'=K''=0 at both ends and degree<=5 fix all six
    coefficients of the quintic smoothstep - checked by finite differences."""
    rc = 0.37
    K = lambda q: oracle.changeover((0.1 + 0.9 * q) * rc, rc)
    assert K(0.0) == 0.0 and K(1.0) == 1.0
    assert oracle.changeover(0.05 * rc, rc) == 0.0 and oracle.changeover(1.2 * rc, rc) == 1.0
    assert abs(K(0.5) - 0.5) < 1e-15
    h = 1e-3
    # one-sided first and second derivatives at the ends (K = O(q^3) there)
    assert abs(K(h)) < 11 * h**3 and abs(1 - K(1 - h)) < 11 * h**3
    # value of the third derivative pins the leading coefficient: K ~ 10 q^3
    assert abs(K(h) / h**3 - 10) < 0.02
    # degree <= 5: the 6th finite difference vanishes anywhere inside
    q0, s = 0.2, 0.1
    d6 = sum((-1) ** k * math.comb(6, k) * K(q0 + k * s) for k in range(7))
    assert abs(d6) < 1e-13
    # monotone and symmetric about (1/2, 1/2)
    qs = np.linspace(0, 1, 401)
    ks = np.array([K(q) for q in qs])
    assert np.all(np.diff(ks) >= 0)
    assert np.allclose(ks + ks[::-1], 1.0, atol=2e-16)


def test_PA4_limits_newtonian_and_zero():
    w = W.shrink(0, 64)
    gm = G * w.mass
    a0, _ = oracle.accel(gm, w.x, np.zeros(w.nb))
    # plain Newtonian direct sum in numpy (textbook definition)
    d = w.x[:, None, :] - w.x[:, :, None]            # d[:, i, j] = x_j - x_i
    r2 = (d**2).sum(0) + np.eye(w.nb)
    wgt = gm[None, :] / r2**1.5 * (1 - np.eye(w.nb))
    ref = (d * wgt[None]).sum(2)
    assert np.allclose(a0, ref, rtol=0, atol=1e-13 * np.abs(ref).max())
    sep = np.sqrt(r2).max()
    a1, _ = oracle.accel(gm, w.x, np.full(w.nb, 10.0 * sep + 1.0))
    assert np.all(a1 == 0.0)


def test_PA5_two_bodies_unequal_masses():
    x = np.array([[1.0, 1.3], [2.0, 2.4], [-0.5, -0.1]])
    gm = np.array([G * 1e-3, G * 5e-6])
    d = x[:, 1] - x[:, 0]
    r = np.linalg.norm(d)
    for rc, Kexp in [(0.0, 1.0), (2.0 * r, None)]:
        a, _ = oracle.accel(gm, x, np.array([rc, 0.0]))
        K = 1.0 if Kexp else oracle.changeover(r, rc)
        if Kexp is None:
            q = (r - 0.1 * rc) / (0.9 * rc)
            assert abs(K - (10 * q**3 - 15 * q**4 + 6 * q**5)) < 1e-15
        assert np.allclose(a[:, 0], gm[1] * K * d / r**3, rtol=4e-16, atol=0)
        assert np.allclose(a[:, 1], -gm[0] * K * d / r**3, rtol=4e-16, atol=0)


def test_coincident_bodies_contribute_nothing():
    x = np.array([[1.0, 1.0, 2.0], [0.0, 0.0, 0.0], [0.0, 0.0, 0.0]])
    gm = np.array([1e-7, 1e-7, 1e-7])
    a, _ = oracle.accel(gm, x, np.zeros(3))
    assert np.all(np.isfinite(a))
    assert a[0, 0] == pytest.approx(1e-7, rel=1e-15) and a[0, 2] == pytest.approx(-2e-7, rel=1e-15)
