"""Seeded synthetic planetesimal-disk workloads (inputs only).

This module is the ONE piece shared by the CUDA path's tests/bench and the CPU
oracle's tests: it draws the inputs.  It holds none of the method's arithmetic
(no pair sum, no changeover weight, no encounter test, no Gauss f,g drift) and
imports neither ``oracle`` nor the CUDA binding.  numpy only.

Recipe: the five BASELINE.json
configs stand in for the paper's own test systems (solar-mass star, a few
already-formed giants, many small bodies on low-e low-i orbits).
``numpy.random.Generator(PCG64(seed))``, float64, whole-array draws in the order
u_a, e, inc, Omega, omega, M, u_mass; giants first, then planetesimals in draw
order (not sorted in a).  Orbital elements -> heliocentric state with
mu_j = G (M_star + m_j); velocities are then made barycentric,
v_j <- v_j - sum_k m_k v_k / (M_star + sum_k m_k), positions stay heliocentric
("democratic heliocentric", PAPER.md:84, 100 fn. 12).
rcrit_j = n_hill * a_j * (m_j / (3 M_star))**(1/3) with n_hill = 3 from the
initial a_j, held fixed (PAPER.md:94, 104 fn. 13-14).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

K_GAUSS = 0.01720209895            # Gaussian gravitational constant
G_AU_DAY_MSUN = K_GAUSS * K_GAUSS  # G = k^2, AU^3 / (Msun day^2)
M_STAR = 1.0
N_HILL = 3.0


@dataclass
class Workload:
    name: str
    N: int                    # objects including the star
    nb: int                   # bodies = N - 1
    seed: int
    m_star: float
    G: float
    mass: np.ndarray          # [nb]   Msun
    x: np.ndarray             # [3,nb] AU, heliocentric
    v: np.ndarray             # [3,nb] AU/day, barycentric
    rcrit: np.ndarray         # [nb]   AU
    dt: float                 # days
    steps: int
    a0: np.ndarray = field(repr=False, default=None)  # initial semi-major axes


# (mass, a, e, inc, mean longitude)
_GIANTS_2 = [(1.0e-3, 5.2, 0.0, 0.0, 0.0), (3.0e-4, 9.5, 0.0, 0.0, 0.5 * math.pi)]
_GIANTS_4 = [(9.5479e-4, 5.2, 0.005, 0.0, 0.0),
             (2.8589e-4, 9.5, 0.005, 0.0, 0.5 * math.pi),
             (4.3662e-5, 19.2, 0.005, 0.0, math.pi),
             (5.1514e-5, 30.1, 0.005, 0.0, 1.5 * math.pi)]

CONFIGS = [
    dict(name="cfg0_N256", N=256, seed=1, giants=_GIANTS_2, a=("uniform", 2.0, 10.0),
         sig_e=0.01, sig_i=0.005, mass=("equal", 1.0e-10), dt=8.0, steps=100),
    dict(name="cfg1_N4096", N=4096, seed=2, giants=_GIANTS_2, a=("uniform", 1.0, 10.0),
         sig_e=0.01, sig_i=0.005, mass=("equal", 1.0e-9), dt=8.0, steps=1000),
    dict(name="cfg2_N16384", N=16384, seed=3, giants=[], a=("sigma", 0.5, 12.0),
         sig_e=0.02, sig_i=0.01, mass=("powerlaw", 1.0e-11, 1.0e-8), dt=4.0, steps=500),
    dict(name="cfg3_N65536", N=65536, seed=4, giants=_GIANTS_4, a=("sigma", 1.0, 30.0),
         sig_e=0.02, sig_i=0.01, mass=("powerlaw", 1.0e-11, 1.0e-8), dt=8.0, steps=200),
    dict(name="cfg4_N131072", N=131072, seed=5, giants=[], a=("uniform", 0.9, 1.1),
         sig_e=0.002, sig_i=0.001, mass=("equal", 1.0e-11), dt=1.0, steps=100),
]


def _solve_kepler(M, e):
    """Eccentric anomaly from mean anomaly (input generation only)."""
    E = M + e * np.sin(M)
    for _ in range(50):
        dE = (E - e * np.sin(E) - M) / (1.0 - e * np.cos(E))
        E = E - dE
        if np.max(np.abs(dE)) < 1e-15:
            break
    return E


def elements_to_state(mu, a, e, inc, Om, om, M):
    """Osculating elements -> Cartesian state (3-1-3 rotation).  Arrays in, [3,n] out."""
    E = _solve_kepler(M, e)
    cE, sE = np.cos(E), np.sin(E)
    b = np.sqrt(1.0 - e * e)
    # perifocal frame
    xp = a * (cE - e)
    yp = a * b * sE
    n = np.sqrt(mu / (a * a * a))
    rr = a * (1.0 - e * cE)
    vxp = -a * a * n * sE / rr
    vyp = a * a * n * b * cE / rr
    cO, sO = np.cos(Om), np.sin(Om)
    co, so = np.cos(om), np.sin(om)
    ci, si = np.cos(inc), np.sin(inc)
    r11 = cO * co - sO * so * ci
    r12 = -cO * so - sO * co * ci
    r21 = sO * co + cO * so * ci
    r22 = -sO * so + cO * co * ci
    r31 = so * si
    r32 = co * si
    x = np.stack([r11 * xp + r12 * yp, r21 * xp + r22 * yp, r31 * xp + r32 * yp])
    v = np.stack([r11 * vxp + r12 * vyp, r21 * vxp + r22 * vyp, r31 * vxp + r32 * vyp])
    return x, v


def make_disk(N, seed, giants, a, sig_e, sig_i, mass, dt, steps, name="custom",
              m_star=M_STAR, G=G_AU_DAY_MSUN, n_hill=N_HILL, nbig=None):
    nb = N - 1
    g = len(giants)
    ns = nb - g
    if ns < 0:
        raise ValueError("N too small for the giants")
    rng = np.random.Generator(np.random.PCG64(seed))
    u_a = rng.random(ns)
    e = rng.rayleigh(sig_e, ns)
    inc = rng.rayleigh(sig_i, ns)
    Om = rng.random(ns) * (2.0 * math.pi)
    om = rng.random(ns) * (2.0 * math.pi)
    Ma = rng.random(ns) * (2.0 * math.pi)
    u_m = rng.random(ns)
    e = np.minimum(e, 0.9 - 1e-12)
    kind, lo, hi = a
    if kind == "uniform":
        sma = lo + u_a * (hi - lo)
    elif kind == "sigma":      # surface density ~ a^-1.5  =>  dN/da ~ a^-1/2
        sma = (math.sqrt(lo) + u_a * (math.sqrt(hi) - math.sqrt(lo))) ** 2
    else:
        raise ValueError(kind)
    if mass[0] == "equal":
        m_s = np.full(ns, float(mass[1]))
    elif mass[0] == "powerlaw":  # dN/dm ~ m^-2.5 on [lo,hi], inverse CDF
        mlo, mhi = mass[1], mass[2]
        m_s = (mlo ** -1.5 + u_m * (mhi ** -1.5 - mlo ** -1.5)) ** (-1.0 / 1.5)
    else:
        raise ValueError(mass[0])
    if nbig is not None:         # bodies nbig.. are massless particles: m = 0, rcrit = 0
        m_s[max(int(nbig) - g, 0):] = 0.0
    gm_ = np.array([t[0] for t in giants], dtype=np.float64)
    ga = np.array([t[1] for t in giants], dtype=np.float64)
    ge = np.array([t[2] for t in giants], dtype=np.float64)
    gi = np.array([t[3] for t in giants], dtype=np.float64)
    gl = np.array([t[4] for t in giants], dtype=np.float64)
    m_all = np.concatenate([gm_, m_s])
    a_all = np.concatenate([ga, sma])
    e_all = np.concatenate([ge, e])
    i_all = np.concatenate([gi, inc])
    Om_all = np.concatenate([np.zeros(g), Om])
    om_all = np.concatenate([np.zeros(g), om])
    M_all = np.concatenate([gl, Ma])
    mu = G * (m_star + m_all)
    xh, vh = elements_to_state(mu, a_all, e_all, i_all, Om_all, om_all, M_all)
    vcm = (vh * m_all[None, :]).sum(axis=1) / (m_star + m_all.sum())
    vb = vh - vcm[:, None]
    rcrit = n_hill * a_all * np.cbrt(m_all / (3.0 * m_star))
    return Workload(name=name, N=N, nb=nb, seed=seed, m_star=m_star, G=G,
                    mass=np.ascontiguousarray(m_all), x=np.ascontiguousarray(xh),
                    v=np.ascontiguousarray(vb), rcrit=np.ascontiguousarray(rcrit),
                    dt=float(dt), steps=int(steps), a0=a_all)


def make_config(idx: int) -> Workload:
    """One of BASELINE.json's five configs (0..4)."""
    c = dict(CONFIGS[idx])
    return make_disk(**c)


def make_bigsmall(N: int, nbig: int, seed: int = 6, m_embryo: float = 3.0e-7) -> Workload:
    """The paper's production regime (N_big 1..100 massive bodies, N_small
    1e4..1e6 massless particles): the cfg3 disk recipe ([1,30] AU, sigma_e/i = 0.02/0.01, the four
    giants) whose first ``nbig`` bodies are big - the giants plus Mars-mass embryos - and the rest
    massless (rcrit = 0).  Not one of BASELINE.json's configs: the workload of SURVEY.md 8(f) row 1."""
    return make_disk(N=N, seed=seed, giants=_GIANTS_4 if nbig >= 4 else _GIANTS_4[:nbig], a=("sigma", 1.0, 30.0),
                     sig_e=0.02, sig_i=0.01, mass=("equal", m_embryo), dt=8.0, steps=100,
                     name=f"bigsmall_N{N}_nbig{nbig}", nbig=nbig)


def shrink(idx: int, N: int, seed=None) -> Workload:
    """Same recipe as config ``idx`` at a smaller N (for tests the oracle can finish)."""
    c = dict(CONFIGS[idx])
    c["N"] = N
    c["name"] = c["name"] + f"_shrunk{N}"
    if seed is not None:
        c["seed"] = seed
    return make_disk(**c)


def random_cluster(nb, seed, box=1.0, vscale=0.01, mlo=1e-9, mhi=1e-3, rc_frac=(0.0, 0.6)):
    """Small random system with bodies inside, across and outside each other's
    changeover shells - for brute-force comparisons (not a disk)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    x = rng.uniform(-box, box, (3, nb))
    v = rng.normal(0.0, vscale, (3, nb))
    mass = np.exp(rng.uniform(math.log(mlo), math.log(mhi), nb))
    rcrit = rng.uniform(rc_frac[0], rc_frac[1], nb) * box
    return Workload(name=f"cluster{nb}", N=nb + 1, nb=nb, seed=seed, m_star=M_STAR,
                    G=G_AU_DAY_MSUN, mass=mass, x=x, v=v, rcrit=rcrit, dt=1.0, steps=1)
