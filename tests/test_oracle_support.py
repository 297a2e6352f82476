"""Pins for the oracle's per-step support routines (readings H-1..H-4,
E-1..E-3): coordinate conversions (mco_h2dh / mce_dh2h, PAPER.md:84 item 1, fn. 12), Hill and
critical radii (mce_hill / mce_init), energy and angular momentum (mxx_en,
PAPER.md:90) - no GPU.  Every pin comes from the inertial-frame definitions (centre of mass,
kinetic + potential energy, sum of r x p of ALL N+1 bodies, star included) or from two-body closed
forms, not from the oracle's own formulas."""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2601_19654_b200 import workloads as W

G = W.G_AU_DAY_MSUN
mp.mp.dps = 40


def _inertial_system(nb, seed):
    """random star + nb bodies in an arbitrary inertial frame: masses, positions q, velocities u"""
    rng = np.random.default_rng(seed)
    m = np.concatenate([[1.3], np.exp(rng.uniform(math.log(1e-7), math.log(3e-2), nb))])
    q = rng.uniform(-5, 5, (nb + 1, 3))
    u = rng.normal(0, 0.02, (nb + 1, 3))
    return m, q, u


def _mpv(a):
    return [mp.mpf(float(t)) for t in a]


def _bary_mp(m, q, u):
    """barycentric positions and velocities of all N+1 bodies, mpmath"""
    M = sum(_mpv(m))
    qc = [sum(mp.mpf(float(m[k])) * mp.mpf(float(q[k, c])) for k in range(len(m))) / M for c in range(3)]
    uc = [sum(mp.mpf(float(m[k])) * mp.mpf(float(u[k, c])) for k in range(len(m))) / M for c in range(3)]
    qb = [[mp.mpf(float(q[k, c])) - qc[c] for c in range(3)] for k in range(len(m))]
    ub = [[mp.mpf(float(u[k, c])) - uc[c] for c in range(3)] for k in range(len(m))]
    return qb, ub


def _helio(q, u):
    return (q[1:] - q[0]).T.copy(), (u[1:] - u[0]).T.copy()


# ---- H-1 / H-2 conversions ------------------------------------------------------------------
@pytest.mark.parametrize("nb,seed", [(1, 11), (3, 12), (6, 13)])
def test_H1_h2dh_is_the_barycentric_velocity_of_the_inertial_definition(nb, seed):
    m, q, u = _inertial_system(nb, seed)
    xh, vh = _helio(q, u)
    _, ub = _bary_mp(m, q, u)
    vdh = oracle.h2dh(m[0], m[1:], vh)
    # barycentric velocity from the (rounded) heliocentric inputs: v_h - sum m v_h / M_tot, mpmath
    M = sum(_mpv(m))
    for c in range(3):
        vc = sum(mp.mpf(float(m[1 + k])) * mp.mpf(float(vh[c, k])) for k in range(nb)) / M
        for b in range(nb):
            ref = mp.mpf(float(vh[c, b])) - vc
            assert abs(mp.mpf(float(vdh[c, b])) - ref) <= mp.mpf(2.3e-16) * abs(ref) + mp.mpf(1e-30)
            # and that IS the inertial barycentric velocity (up to the rounding of u - u_star)
            assert abs(ref - ub[1 + b][c]) <= mp.mpf(1e-15)


def test_H1_two_body_closed_form_and_H2_inverse():
    # star M + planet m moving at v_h relative to the star: barycentric planet velocity = v_h M/(M+m)
    M, m = 1.0, 0.25
    vh = np.array([[0.3], [-0.1], [0.05]])
    vdh = oracle.h2dh(M, [m], vh)
    assert np.allclose(vdh, vh * M / (M + m), rtol=3e-16, atol=0)
    w = W.make_config(1)
    vh = oracle.dh2h(w.m_star, w.mass, w.v)
    back = oracle.h2dh(w.m_star, w.mass, vh)
    assert np.max(np.abs(back - w.v)) <= 4e-16 * np.max(np.abs(w.v))
    # velocity differences are frame independent
    assert np.allclose(vh[:, 1:] - vh[:, :-1], w.v[:, 1:] - w.v[:, :-1], rtol=0, atol=1e-17)
    # the generator's velocities are barycentric: total momentum with the star's (H-2) vanishes
    S = (w.mass * w.v).sum(1)
    v_star = -S / w.m_star
    assert np.allclose(vh.T - w.v.T, -v_star, rtol=0, atol=1e-17)


# ---- H-3 / H-4 Hill and critical radii ---------------------------------------------------------
def test_H3_closed_forms():
    # |x| = 13 exactly, m/(3 M) = 1/8 exactly -> r_H = 6.5, rcrit = 3 r_H = 19.5
    x = np.array([[3.0], [4.0], [12.0]]); v = np.zeros((3, 1))
    rh, rc = oracle.hill(G, 1.0, [0.375], x, v, n_hill=3.0)
    assert rh[0] == 6.5 and rc[0] == 19.5
    # Jupiter at 5.2 AU: the textbook 0.355 AU
    rh, _ = oracle.hill(G, 1.0, [9.5479e-4], np.array([[5.2], [0.0], [0.0]]), v)
    assert abs(rh[0] - 0.3551) < 2e-4
    assert abs(rh[0] - 5.2 * (9.5479e-4 / 3.0) ** (1.0 / 3.0)) <= 1e-15
    # massless body: 0
    assert oracle.hill(G, 1.0, [0.0], x, v)[1][0] == 0.0


def test_H4_osculating_variant_recovers_the_generators_semi_major_axes():
    """workloads builds the state from elements (a -> x, v) and rcrit = 3 a (m/3M)^(1/3); mode 1 goes
    back state -> a by vis-viva: two independent routes to the same number."""
    for cfg in (0, 1):
        w = W.make_config(cfg)
        _, rc = oracle.hill(G, w.m_star, w.mass, w.x, w.v, n_hill=3.0, mode=1)
        assert np.max(np.abs(rc - w.rcrit) / w.rcrit) <= 2e-12
    # mode 0 at perihelion of an e = 0.3 orbit is (1 - e) times mode 1
    e, a, m = 0.3, 2.0, 1e-4
    mu = G * (1.0 + m)
    x = np.array([[a * (1 - e)], [0.0], [0.0]])
    vh = np.array([[0.0], [math.sqrt(mu / a * (1 + e) / (1 - e))], [0.0]])
    vdh = oracle.h2dh(1.0, [m], vh)
    r0 = oracle.hill(G, 1.0, [m], x, vdh, mode=0)[0][0]
    r1 = oracle.hill(G, 1.0, [m], x, vdh, mode=1)[0][0]
    assert abs(r0 / r1 - (1 - e)) <= 1e-14
    # unbound body: falls back to the separation
    vfast = oracle.h2dh(1.0, [m], 3.0 * vh)
    assert oracle.hill(G, 1.0, [m], x, vfast, mode=1)[0][0] == pytest.approx(r0, rel=1e-15)


# ---- E-1..E-3 energy and angular momentum ----------------------------------------------------
@pytest.mark.parametrize("a,e,m", [(1.0, 0.0, 1e-3), (5.2, 0.3, 0.05), (0.4, 0.7, 1e-6)])
def test_E_two_body_closed_forms(a, e, m):
    M = 1.0
    inc, Om, om, Man = 0.4, 1.1, 2.3, 0.9
    x, vh = W.elements_to_state(G * (M + m), np.array([a]), np.array([e]), np.array([inc]), np.array([Om]),
                                np.array([om]), np.array([Man]))
    vdh = oracle.h2dh(M, [m], vh)
    r = oracle.energy(G, M, [m], x, vdh)
    E_ref = -G * M * m / (2 * a)
    assert abs(r["E"] - E_ref) <= 1e-14 * r["Eabs"]
    Lmag = M * m / (M + m) * math.sqrt(G * (M + m) * a * (1 - e * e))
    nrm = np.array([math.sin(inc) * math.sin(Om), -math.sin(inc) * math.cos(Om), math.cos(inc)])
    assert np.max(np.abs(r["L"] - Lmag * nrm)) <= 1e-14 * Lmag
    assert r["Up"] == 0.0 and abs(r["T"] + r["Us"] - r["E"]) <= 1e-30 + 1e-16 * r["Eabs"]


@pytest.mark.parametrize("nb,nbig,seed", [(2, None, 21), (5, None, 22), (6, 2, 23), (6, 0, 24), (4, 3, 25)])
def test_E_bruteforce_from_the_inertial_definitions(nb, nbig, seed):
    m, q, u = _inertial_system(nb, seed)
    xh, vh = _helio(q, u)
    vdh = oracle.h2dh(m[0], m[1:], vh)
    got = oracle.energy(G, m[0], m[1:], xh, vdh, nbig=nbig)
    # all N+1 bodies in the barycentric frame, built from the SAME rounded helio inputs the oracle sees
    q2 = np.vstack([np.zeros(3), xh.T]); u2 = np.vstack([np.zeros(3), vh.T])
    qb, ub = _bary_mp(m, q2, u2)
    mm = _mpv(m)
    T = sum(mm[k] * sum(t * t for t in ub[k]) for k in range(nb + 1)) / 2
    Us = -sum(mp.mpf(G) * mm[0] * mm[k] / mp.sqrt(sum((qb[k][c] - qb[0][c]) ** 2 for c in range(3))) for k in range(1, nb + 1))
    nbg = nb if nbig is None else nbig
    Up = -sum(mp.mpf(G) * mm[i] * mm[j] / mp.sqrt(sum((qb[i][c] - qb[j][c]) ** 2 for c in range(3)))
              for i in range(1, nb + 1) for j in range(i + 1, nb + 1) if i - 1 < nbg)
    L = [sum(mm[k] * (qb[k][(c + 1) % 3] * ub[k][(c + 2) % 3] - qb[k][(c + 2) % 3] * ub[k][(c + 1) % 3])
             for k in range(nb + 1)) for c in range(3)]
    tol = mp.mpf(3e-15)        # vdh is rounded to double once (relative 1.1e-16 per velocity)
    assert abs(mp.mpf(float(got["T"])) - T) <= tol * T
    assert abs(mp.mpf(float(got["Us"])) - Us) <= tol * abs(Us)
    assert abs(mp.mpf(float(got["Up"])) - Up) <= tol * abs(Up) + mp.mpf(1e-40)
    assert abs(mp.mpf(float(got["E"])) - (T + Us + Up)) <= tol * mp.mpf(float(got["Eabs"]))
    for c in range(3):
        assert abs(mp.mpf(float(got["L"][c])) - L[c]) <= tol * mp.mpf(float(got["Labs"][c]))


def test_E_energy_error_of_the_step_scales_as_dt_squared():
    """second-order symplectic step: the energy error after a fixed time span shrinks ~4x when dt halves
    (ties oracle.energy to the already pinned oracle.step through a property neither encodes)."""
    w = W.shrink(0, 40)
    gm, mu = G * w.mass, G * w.m_star
    rc0 = np.zeros(w.nb)
    E0 = oracle.energy(G, w.m_star, w.mass, w.x, w.v)["E"]
    errs = []
    for dt, n in [(8.0, 8), (4.0, 16)]:
        x, v = w.x, w.v
        a, _ = oracle.accel(gm, x, rc0)
        for _ in range(n):
            r = oracle.step(mu, gm, rc0, dt, x, v, a, with_encounters=False)
            x, v, a = r["x"], r["v"], r["a"]
        errs.append(abs(oracle.energy(G, w.m_star, w.mass, x, v)["E"] - E0) / abs(E0))
    assert errs[0] < 1e-6 and 2.5 < errs[0] / errs[1] < 6.0, errs
