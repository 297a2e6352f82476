"""Pins for the oracle's Kepler drift (O-C) - no GPU."""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2601_19654_b200 import workloads as W
from tests import mp_reference as R

MU = W.G_AU_DAY_MSUN * 1.0


def _orbit(a, e, inc=0.3, Om=0.7, om=1.1, M=0.4, mu=MU):
    x, v = W.elements_to_state(np.array([mu]), np.array([a]), np.array([e]), np.array([inc]),
                               np.array([Om]), np.array([om]), np.array([M]))
    return x, v


def _energy(x, v, mu=MU):
    return 0.5 * (v**2).sum(0) - mu / np.sqrt((x**2).sum(0))


@pytest.mark.parametrize("e", [0.0, 0.22, 0.7, 0.95])
@pytest.mark.parametrize("n", [1, 7, 500])
def test_PC1_period_return_energy_angmom(e, n):
    a = 5.2
    x0, v0 = _orbit(a, e)
    P = 2 * math.pi * math.sqrt(a**3 / MU)
    x, v = x0.copy(), v0.copy()
    E0 = _energy(x0, v0)
    L0 = np.cross(x0[:, 0], v0[:, 0])
    for _ in range(n):
        x, v, fl = oracle.drift(MU, P / n, x, v)
        assert fl[0] == 0
    # conditioning: an error d(period) shifts the body along the orbit by ~v dP; near
    # pericentre of e=0.95 that is amplified by (1+e)/(1-e)
    amp = (1 + e) / (1 - e)
    assert np.linalg.norm(x - x0) <= 1e-12 * amp * np.linalg.norm(x0) * max(1, n / 50)
    assert np.linalg.norm(v - v0) <= 1e-12 * amp**2 * np.linalg.norm(v0) * max(1, n / 50)
    assert abs(_energy(x, v)[0] - E0[0]) <= 1e-12 * abs(E0[0])
    L1 = np.cross(x[:, 0], v[:, 0])
    assert np.linalg.norm(L1 - L0) <= 1e-14 * np.linalg.norm(L0) * max(1, n / 50)


@pytest.mark.parametrize("dt", [8.0, -8.0, 1234.5, 1.0e5])
def test_PC2_circular_closed_form(dt):
    a = 2.0
    n = math.sqrt(MU / a**3)
    x0 = np.array([[a], [0.0], [0.0]])
    v0 = np.array([[0.0], [a * n], [0.0]])
    x, v, _ = oracle.drift(MU, dt, x0, v0)
    th = n * dt
    # v0 = a*n is rounded, so the orbit is circular only to ~1e-16: allow the phase error n*dt*eps
    tol = 4e-16 * (1 + abs(th))
    assert abs(x[0, 0] - a * math.cos(th)) <= tol * a and abs(x[1, 0] - a * math.sin(th)) <= tol * a
    assert abs(v[0, 0] + a * n * math.sin(th)) <= tol * a * n
    assert abs(v[1, 0] - a * n * math.cos(th)) <= tol * a * n
    assert x[2, 0] == 0.0 and v[2, 0] == 0.0


def test_PC3_fg_determinant_is_one():
    # x' x v' = (f gdot - fdot g) x0 x v0 : the determinant is |L'|/|L| and L' || L
    w = W.shrink(3, 200)
    x1, v1, fl = oracle.drift(MU, 8.0, w.x, w.v)
    assert not fl.any()
    L0 = np.cross(w.x.T, w.v.T)
    L1 = np.cross(x1.T, v1.T)
    det = (L1 * L0).sum(1) / (L0 * L0).sum(1)
    assert np.max(np.abs(det - 1)) <= 1e-15
    assert np.max(np.linalg.norm(L1 - L0, axis=1) / np.linalg.norm(L0, axis=1)) <= 2e-15


def test_PC4_reverse_is_identity_and_PC5_group_property():
    w = W.shrink(2, 300)
    x1, v1, _ = oracle.drift(MU, 4.0, w.x, w.v)
    xb, vb, _ = oracle.drift(MU, -4.0, x1, v1)
    nx = np.linalg.norm(w.x, axis=0); nv = np.linalg.norm(w.v, axis=0)
    assert np.max(np.linalg.norm(xb - w.x, axis=0) / nx) <= 1e-14
    assert np.max(np.linalg.norm(vb - w.v, axis=0) / nv) <= 1e-14
    xa, va, _ = oracle.drift(MU, 1.5, w.x, w.v)
    xa, va, _ = oracle.drift(MU, 2.5, xa, va)
    assert np.max(np.linalg.norm(xa - x1, axis=0) / nx) <= 1e-13
    assert np.max(np.linalg.norm(va - v1, axis=0) / nv) <= 1e-13


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_PC6_mpmath_elements_propagation(seed):
    """independent formulation: classical elements + Kepler's equation at 50 digits,
    including dt >> P and negative dt."""
    rng = np.random.default_rng(seed)
    nb = 8
    a = rng.uniform(0.5, 30, nb); e = rng.uniform(0, 0.9, nb)
    x, v = W.elements_to_state(np.full(nb, MU), a, e, rng.uniform(0, 0.5, nb), rng.uniform(0, 6.28, nb),
                               rng.uniform(0, 6.28, nb), rng.uniform(0, 6.28, nb))
    for dt in (8.0, -3.0, 4000.0, 3.0e5):
        x1, v1, fl = oracle.drift(MU, dt, x, v)
        assert not fl.any()
        for b in range(nb):
            xm, vm = R.kepler_elements_propagate_mp(MU, dt, x[:, b], v[:, b])
            P = 2 * math.pi * math.sqrt(a[b] ** 3 / MU)
            # inputs are doubles: an eps-level change of the state changes the mean motion by
            # ~eps and so the answer by ~eps * (#orbits) * 2pi * amplification
            tol = 2e-16 * (3 + 30 * abs(dt) / P / (1 - e[b]) ** 2)
            nx = float(mp.sqrt(sum(t * t for t in xm))); nv = float(mp.sqrt(sum(t * t for t in vm)))
            ex = max(abs(float(mp.mpf(float(x1[c, b])) - xm[c])) for c in range(3))
            ev = max(abs(float(mp.mpf(float(v1[c, b])) - vm[c])) for c in range(3))
            assert ex <= tol * nx * (1 + e[b]) / (1 - e[b]), (dt, b, ex / nx)
            assert ev <= tol * nv * ((1 + e[b]) / (1 - e[b])) ** 2, (dt, b, ev / nv)


def test_hyperbolic_and_failure_flag():
    # unbound orbit (beta < 0): energy and angular momentum still conserved (reading C-e)
    x0 = np.array([[1.0], [0.0], [0.0]]); v0 = np.array([[0.0], [0.04], [0.001]])
    assert _energy(x0, v0)[0] > 0
    x1, v1, fl = oracle.drift(MU, 50.0, x0, v0)
    assert fl[0] == 0
    assert abs(_energy(x1, v1)[0] - _energy(x0, v0)[0]) <= 1e-14 * abs(_energy(x0, v0)[0])
    assert np.allclose(np.cross(x1[:, 0], v1[:, 0]), np.cross(x0[:, 0], v0[:, 0]), rtol=1e-14, atol=1e-17)
    # r0 = 0 -> flagged, state untouched (reading C-f)
    xz = np.zeros((3, 2)); xz[:, 1] = [1, 0, 0]
    vz = np.array([[0.01, 0.0], [0.0, 0.017], [0.0, 0.0]])
    x2, v2, fl = oracle.drift(MU, 1.0, xz, vz)
    assert fl[0] == 1 and fl[1] == 0
    assert np.all(x2[:, 0] == 0) and np.all(v2[:, 0] == vz[:, 0])
    # dt = 0 is the identity
    x3, v3, _ = oracle.drift(MU, 0.0, x0, v0)
    assert np.array_equal(x3, x0) and np.array_equal(v3, v0)
