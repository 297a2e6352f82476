"""Pins for the oracle's big x all variant (readings R-1..R-3) - no GPU.

The paper's loops: force sum `do j = 2, nbod` x `do i = 2, nbig` (only the big
bodies are gravity sources), box padding `do j = 2, nbig`, pair
test `do i = 2, nbig` x `do j = 2, nbod`, j > i.  Each pin is fixed by those
definitions independently of oracle/mopal_oracle.c."""
import itertools

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2601_19654_b200 import workloads as W
from tests import mp_reference as R

G = W.G_AU_DAY_MSUN


# ---- acceleration (R-1) ------------------------------------------------------------------
@pytest.mark.parametrize("nb,nbig,seed", [(5, 1, 31), (8, 3, 32), (8, 7, 33), (6, 0, 34)])
def test_R1_bruteforce_mpmath(nb, nbig, seed):
    w = W.random_cluster(nb, seed)
    gm = G * w.mass
    a, S = oracle.accel(gm, w.x, w.rcrit, nbig=nbig)
    X = [[mp.mpf(float(w.x[c, b])) for c in range(3)] for b in range(nb)]
    for i in range(nb):
        acc = [mp.mpf(0)] * 3
        ab = [mp.mpf(0)] * 3
        for j in range(nbig):                          # sources: big bodies only
            if j == i:
                continue
            d = [X[j][c] - X[i][c] for c in range(3)]
            r = mp.sqrt(sum(t * t for t in d))
            rc = max(mp.mpf(float(w.rcrit[i])), mp.mpf(float(w.rcrit[j])))
            wgt = mp.mpf(float(gm[j])) * R.K_mp(r, rc) / r**3
            acc = [acc[c] + wgt * d[c] for c in range(3)]
            ab = [ab[c] + abs(wgt * d[c]) for c in range(3)]
        for c in range(3):
            assert abs(mp.mpf(float(a[c, i])) - acc[c]) <= mp.mpf(2e-16) * ab[c] + mp.mpf(1e-300)
            assert abs(mp.mpf(float(S[c, i])) - ab[c]) <= mp.mpf(1e-15) * ab[c] + mp.mpf(1e-300)


@pytest.mark.parametrize("cfg,N,nbig", [(1, 300, 2), (3, 400, 4), (2, 257, 100), (4, 200, 150)])
def test_R1_equals_full_sum_with_small_masses_zeroed(cfg, N, nbig):
    """a source of zero mass contributes exactly 0 to the (already pinned) full sum, so the
    big x all sum must reproduce it bit for bit - also inside changeover shells."""
    w = W.shrink(cfg, N)
    rcrit = w.rcrit * 30.0
    gm = G * w.mass
    gm0 = gm.copy(); gm0[nbig:] = 0.0
    a, S = oracle.accel(gm, w.x, rcrit, nbig=nbig)
    af, Sf = oracle.accel(gm0, w.x, rcrit)
    assert np.array_equal(a, af) and np.array_equal(S, Sf)
    # and it is NOT the fully interacting sum
    a_all, _ = oracle.accel(gm, w.x, rcrit)
    assert not np.array_equal(a, a_all)
    # nbig = nb is the fully interacting sum
    a_nb, S_nb = oracle.accel(gm, w.x, rcrit, nbig=w.nb)
    assert np.array_equal(a_nb, a_all)


def test_R1_test_particles_closed_form():
    """one big body: every small body feels gm_0 (x_0 - x_i)/r^3 and nothing else; the big body
    feels nothing (no back reaction) even though the small bodies carry mass."""
    rng = np.random.default_rng(41)
    nb = 50
    x = rng.normal(size=(3, nb)) * 3.0
    gm = G * rng.uniform(1e-6, 1e-3, nb)
    a, S = oracle.accel(gm, x, np.zeros(nb), nbig=1)
    assert np.all(a[:, 0] == 0.0) and np.all(S[:, 0] == 0.0)
    d = x[:, :1] - x[:, 1:]
    r = np.sqrt((d * d).sum(axis=0))
    ref = gm[0] * d / r**3
    assert np.max(np.abs(a[:, 1:] - ref) / np.abs(ref)) < 2e-15      # the numpy double formula itself carries a few ulp
    # two equal big bodies at (+-D, 0, 0), a small one on the y axis: a = -2 gm y / (D^2+y^2)^(3/2) e_y
    D, y, g = 1.5, 0.7, 3e-7
    x = np.array([[D, -D, 0.0], [0.0, 0.0, y], [0.0, 0.0, 0.0]])
    a, _ = oracle.accel(np.array([g, g, 9.9]), x, np.zeros(3), nbig=2)
    assert abs(a[1, 2] + 2 * g * y / (D * D + y * y) ** 1.5) <= 4e-16 * abs(a[1, 2])
    assert a[0, 2] == 0.0 and a[2, 2] == 0.0
    # the bigs pull each other, the (massive) small body does not pull them
    assert abs(a[0, 0] + g / (4 * D * D)) <= 4e-16 * abs(a[0, 0]) and a[1, 0] == 0.0


def test_R1_rows_variant_matches():
    w = W.shrink(1, 500)
    gm = G * w.mass
    rows = np.array([0, 1, 2, 17, 498], dtype=np.int32)
    a, S = oracle.accel(gm, w.x, w.rcrit, nbig=2)
    ar, Sr = oracle.accel_rows(gm, w.x, w.rcrit, rows, nbig=2)
    assert np.array_equal(ar, a[:, rows]) and np.array_equal(Sr, S[:, rows])


# ---- boxes and pairs (R-2, R-3) ------------------------------------------------------------
def _bent_end_state(w, h, seed):
    rng = np.random.default_rng(seed)
    v1 = w.v + rng.normal(0, 0.2, w.v.shape)
    x1 = w.x + h * 0.5 * (w.v + v1) + rng.normal(0, 0.02, w.x.shape)
    return x1, v1


def test_R2_only_big_boxes_are_padded():
    w = W.random_cluster(9, 51, box=0.5, vscale=0.3, rc_frac=(0.1, 0.9))
    h = 1.3
    x1, v1 = _bent_end_state(w, h, 51)
    lo0, hi0 = oracle.boxes(h, w.x, w.v, x1, v1, np.zeros(9))              # the bare extremes (pinned)
    lo, hi = oracle.boxes(h, w.x, w.v, x1, v1, w.rcrit, nbig=4)
    pad = np.where(np.arange(9) < 4, w.rcrit, 0.0)
    assert np.array_equal(lo, lo0 - pad) and np.array_equal(hi, hi0 + pad)
    lo_all, hi_all = oracle.boxes(h, w.x, w.v, x1, v1, w.rcrit)
    assert np.array_equal(lo_all, lo0 - w.rcrit) and np.array_equal(hi_all, hi0 + w.rcrit)


@pytest.mark.parametrize("seed,h,nbig", [(61, 1.0, 1), (62, 1.0, 3), (63, -1.0, 3), (64, 0.5, 5), (65, 2.0, 7)])
def test_R3_bruteforce_mpmath(seed, h, nbig):
    nb = 8
    w = W.random_cluster(nb, seed, box=0.5, vscale=0.3, rc_frac=(0.1, 0.9))
    x1, v1 = _bent_end_state(w, h, seed)
    res = oracle.encounters(h, w.x, w.v, x1, v1, w.rcrit, nbig=nbig)
    lo = np.empty((2, nb), dtype=object); hi = np.empty((2, nb), dtype=object)
    for b in range(nb):
        pad = mp.mpf(float(w.rcrit[b])) if b < nbig else mp.mpf(0)
        for c in range(2):
            l, u = R.hermite_extremes_mp(float(w.x[c, b]), float(x1[c, b]), float(w.v[c, b]), float(v1[c, b]), h)
            lo[c, b] = l - pad; hi[c, b] = u + pad
    inn, amb = set(), set()
    tol = mp.mpf(1e-11)
    for i, j in itertools.combinations(range(nb), 2):
        if i >= nbig:                                  # first member must be a big body
            continue
        gate = all(lo[c, i] <= hi[c, j] and lo[c, j] <= hi[c, i] for c in range(2))
        near = any(abs(lo[c, i] - hi[c, j]) <= tol * max(abs(lo[c, i]), abs(hi[c, j])) or
                   abs(lo[c, j] - hi[c, i]) <= tol * max(abs(lo[c, j]), abs(hi[c, i])) for c in range(2))
        d2, d0, d1 = R.d2min_mp(h, w.x[:, i], w.v[:, i], x1[:, i], v1[:, i], w.x[:, j], w.v[:, j], x1[:, j], v1[:, j])
        rc = max(mp.mpf(float(w.rcrit[i])), mp.mpf(float(w.rcrit[j])))
        if abs(d2 - rc * rc) <= tol * max(rc * rc, d0, d1) or near:
            amb.add((i, j))
        elif gate and d2 <= rc * rc:
            inn.add((i, j))
    got = set(map(tuple, res["pairs"].tolist()))
    assert inn - amb <= got <= inn | amb
    assert all(i < nbig and i < j for i, j in got)
    assert res["pairs"].tolist() == sorted(res["pairs"].tolist())
    fl = np.zeros(nb, dtype=np.uint8)
    for i, j in got:
        fl[i] = fl[j] = 1
    assert np.array_equal(fl, res["flag"])


def test_R3_equals_filtered_full_list_when_small_rcrit_is_zero():
    """padding a box by 0 is no padding: with rcrit = 0 on the small bodies the big x all list is
    the (already pinned) full list restricted to pairs whose first member is big."""
    w = W.shrink(4, 400)
    h = 1.0
    x1, v1, fl = oracle.drift(G * w.m_star, h, w.x, w.v)
    nbig = 37
    rcrit = w.rcrit * 400.0
    rcrit[nbig:] = 0.0
    full = oracle.encounters(h, w.x, w.v, x1, v1, rcrit)
    big = oracle.encounters(h, w.x, w.v, x1, v1, rcrit, nbig=nbig)
    keep = full["pairs"][full["pairs"][:, 0] < nbig]
    assert len(keep) > 100          # (small, small) pairs have rc = 0 and are never flagged, so keep is the full list
    assert np.array_equal(big["pairs"], keep) and big["count"] == len(keep)
    # nbig = nb is the full list
    allb = oracle.encounters(h, w.x, w.v, x1, v1, rcrit, nbig=w.nb)
    assert np.array_equal(allb["pairs"], full["pairs"])


# ---- step -----------------------------------------------------------------------------------
def test_R_step_is_the_composition_of_its_pinned_parts():
    w = W.shrink(1, 120)
    nbig = 2
    mu = G * w.m_star
    gm = G * w.mass
    h = 8.0
    a0, _ = oracle.accel(gm, w.x, w.rcrit, nbig=nbig)
    st = oracle.step(mu, gm, w.rcrit, h, w.x, w.v, a0, nbig=nbig)
    v = oracle.kick(0.5 * h, w.v, a0)
    x, _ = oracle.jump(0.5 * h, mu, gm, w.x, v)
    x0, v0 = x.copy(), v.copy()
    x, v, _ = oracle.drift(mu, h, x, v)
    enc = oracle.encounters(h, x0, v0, x, v, w.rcrit, nbig=nbig)
    x, _ = oracle.jump(0.5 * h, mu, gm, x, v)
    a, _ = oracle.accel(gm, x, w.rcrit, nbig=nbig)
    v = oracle.kick(0.5 * h, v, a)
    assert np.array_equal(st["x"], x) and np.array_equal(st["v"], v) and np.array_equal(st["a"], a)
    assert np.array_equal(st["x0"], x0) and np.array_equal(st["pairs"], enc["pairs"])


def test_R_step_massless_small_bodies_do_not_move_the_bigs():
    """with massless small bodies the big bodies' trajectory is that of the big bodies alone."""
    w = W.shrink(1, 60)
    nbig = 2
    mass = w.mass.copy(); mass[nbig:] = 0.0
    mu = G * w.m_star
    gm = G * mass
    h = 8.0
    a, _ = oracle.accel(gm, w.x, w.rcrit, nbig=nbig)
    ab, _ = oracle.accel(gm[:nbig], w.x[:, :nbig], w.rcrit[:nbig])
    x, v = w.x, w.v
    xb, vb = w.x[:, :nbig].copy(), w.v[:, :nbig].copy()
    for _ in range(3):
        st = oracle.step(mu, gm, w.rcrit, h, x, v, a, nbig=nbig)
        x, v, a = st["x"], st["v"], st["a"]
        sb = oracle.step(mu, gm[:nbig], w.rcrit[:nbig], h, xb, vb, ab)
        xb, vb, ab = sb["x"], sb["v"], sb["a"]
    assert np.array_equal(x[:, :nbig], xb) and np.array_equal(v[:, :nbig], vb)
