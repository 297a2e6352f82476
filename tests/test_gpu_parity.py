"""GPU parity: libmopal (through the C ABI binding) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are north_star's:
  accel      |a_gpu - a_ref| <= 1e-12 * sum_j |contribution_j|   per component
  encounters pair lists bit-exact except pairs within 1e-12 relative of a threshold
  drift      1e-13 relative (to the vector's 2-norm, reading C-d)
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2601_19654_b200 import workloads as W

G = W.G_AU_DAY_MSUN


@pytest.fixture(scope="module")
def M():
    from paper_2601_19654_b200 import mopal
    return mopal


def _mk(M, w, rcrit=None, cap=1 << 20):
    return M.Mopal(w.mass, w.x, w.v, w.rcrit if rcrit is None else rcrit, m_star=w.m_star, G=w.G, cap=cap)


def _check_accel(a_gpu, a_ref, S, what=""):
    err = np.abs(a_gpu - a_ref)
    tol = 1e-12 * S
    bad = err > tol + 1e-300
    worst = np.max(err / (S + 1e-300))
    assert not bad.any(), f"{what}: {bad.sum()} components out of tolerance, worst {worst:.3e} x S"
    return worst


def _rel_vec_err(got, ref):
    return np.max(np.abs(got - ref), axis=0) / np.linalg.norm(ref, axis=0)


def _pairs_ok(got, ref):
    """SURE_IN subset of GPU list subset of SURE_IN + AMBIG; returns #ambiguous."""
    S = set(map(tuple, ref["pairs"].tolist()))
    A = set(map(tuple, ref["ambig"].tolist()))
    Gs = set(map(tuple, got.tolist()))
    assert (S - A) <= Gs, f"missing {sorted((S - A) - Gs)[:5]}"
    assert Gs <= (S | A), f"extra {sorted(Gs - (S | A))[:5]}"
    return len(A)


# ------------------------------------------------------------------------------ accel
@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_accel_full_configs(M, cfg):
    w = W.make_config(cfg)
    m = _mk(M, w)
    m.accel()
    a = m.get("a")
    a_ref, S = oracle.accel(G * w.mass, w.x, w.rcrit)
    worst = _check_accel(a, a_ref, S, w.name)
    assert worst < 2e-13          # in practice ~sqrt(n) eps, far inside the bound
    m.close()


@pytest.mark.parametrize("cfg", [3, 4])
def test_accel_headline_sizes_every_row(M, cfg):
    """full-size launch configuration (the one bench.py times) against the oracle on EVERY row
    (4 s / 18 s of oracle time on the GPU box's host cores)."""
    w = W.make_config(cfg)
    m = _mk(M, w)
    assert m.pair_kernel_name() == "pair_sym_kernel"
    m.accel()
    a = m.get("a")
    a_ref, S = oracle.accel(G * w.mass, w.x, w.rcrit)
    worst = _check_accel(a, a_ref, S, w.name)
    assert worst < 2e-13
    # property at any size: Newton III with the symmetric K
    for c in range(3):
        assert abs(np.sum(w.mass * a[c])) <= 1e-11 * np.sum(w.mass * np.abs(a[c]))
    m.close()


@pytest.mark.parametrize("psm", ["1", "0"])
@pytest.mark.parametrize("nb", [1, 2, 3, 7, 8, 9, 127, 128, 129, 255, 257, 1000, 1024])
def test_accel_ragged_sizes_and_changeover_shell(M, monkeypatch, nb, psm):
    """psm = 1: pair_small_kernel (8 lanes per body); psm = 0: the tiled one-sided pair_accel_kernel"""
    monkeypatch.setenv("MO_PSM", psm)
    w = W.random_cluster(nb, 100 + nb, box=1.0, rc_frac=(0.0, 0.7)) if nb > 1 else W.random_cluster(1, 5)
    if nb > 100:   # plant one pair well inside 0.1 rc (K = 0) - random draws do not always have one
        w.x[:, 1] = w.x[:, 0] + np.array([0.03 * max(w.rcrit[0], w.rcrit[1]), 0.0, 0.0])
    m = _mk(M, w)
    assert m.pair_kernel_name() == ("pair_small_kernel" if psm == "1" else "pair_accel_kernel")
    m.accel()
    a = m.get("a")
    a_ref, S = oracle.accel(G * w.mass, w.x, w.rcrit)
    _check_accel(a, a_ref, S, f"cluster{nb}")
    if nb > 100:   # the sample really exercises K in (0,1), K = 0 and K = 1
        d = np.linalg.norm(w.x[:, :, None] - w.x[:, None, :], axis=0) + 9 * np.eye(nb)
        rc = np.maximum(w.rcrit[:, None], w.rcrit[None, :])
        assert ((d < rc) & (d > 0.1 * rc)).any() and (d <= 0.1 * rc).any() and (d >= rc).any()
    m.close()


@pytest.fixture
def force_sym(monkeypatch):
    """Select the two-sided pair kernel (pair_sym_kernel) whatever nb is; MO_SYM is read by mo_create."""
    def _set(ch=None, ipt=6):
        monkeypatch.setenv("MO_SYM", "1")
        monkeypatch.setenv("MO_PSM", "0")
        monkeypatch.setenv("MO_SYM_IPT", str(ipt))
        if ch is not None:
            monkeypatch.setenv("MO_SYM_CH", str(ch))
    return _set


@pytest.mark.parametrize("ipt", [6, 3, 2])
@pytest.mark.parametrize("nb,ch", [(1, 1), (2, 1), (33, 1), (129, 2), (257, 1), (385, 2), (511, 1), (767, 1), (768, 3), (769, 1), (1000, 2),
                                   (1537, 1), (2500, 5)])
def test_accel_sym_kernel_ragged_sizes_and_changeover_shell(M, force_sym, nb, ch, ipt):
    # several row blocks (768 / 384 / 256 rows for 6 / 3 / 2 bodies per lane), diagonal and off-diagonal tiles, ragged
    # tails, every chunking
    force_sym(ch, ipt)
    w = W.random_cluster(nb, 300 + nb, box=1.0, rc_frac=(0.0, 0.7)) if nb > 1 else W.random_cluster(1, 5)
    if nb > 100:
        w.x[:, 1] = w.x[:, 0] + np.array([0.03 * max(w.rcrit[0], w.rcrit[1]), 0.0, 0.0])
        w.x[:, nb - 1] = w.x[:, 5]          # coincident bodies in different tiles contribute nothing
    m = _mk(M, w)
    assert m.pair_geometry()["ipt"] == ipt and m.pair_kernel_name() == "pair_sym_kernel"   # the two-sided kernel really is the one running
    m.accel()
    a = m.get("a")
    a_ref, S = oracle.accel(G * w.mass, w.x, w.rcrit)
    assert np.all(np.isfinite(a))
    _check_accel(a, a_ref, S, f"sym cluster{nb}")
    m.accel()
    assert np.array_equal(a, m.get("a"))    # fixed reduction tree: bit-reproducible
    m.close()


@pytest.mark.parametrize("ipt", [6, 3, 2])
def test_accel_sym_kernel_disk_and_step(M, force_sym, ipt):
    force_sym(None, ipt)
    w = W.shrink(1, 3000)
    m = _mk(M, w)
    m.accel()
    a_ref, S = oracle.accel(G * w.mass, w.x, w.rcrit)
    _check_accel(m.get("a"), a_ref, S, "sym disk")
    st = m.step(w.dt, 2)
    x, v, acc = w.x, w.v, a_ref
    for _ in range(2):
        r = oracle.step(G * w.m_star, G * w.mass, w.rcrit, w.dt, x, v, acc)
        x, v, acc = r["x"], r["v"], r["a"]
    assert max(_rel_vec_err(m.get("x"), x).max(), _rel_vec_err(m.get("v"), v).max()) <= 3e-13
    assert st.steps_done == 2
    m.close()


def test_accel_degenerate_cases(M):
    # coincident bodies contribute nothing; rcrit = 0 is Newtonian; rcrit huge gives exactly 0
    w = W.shrink(0, 300)
    x = w.x.copy(); x[:, 7] = x[:, 3]
    gm = G * w.mass
    for rc in (np.zeros(w.nb), w.rcrit, np.full(w.nb, 1e6)):
        m = M.Mopal(w.mass, x, w.v, rc)
        m.accel()
        a = m.get("a")
        a_ref, S = oracle.accel(gm, x, rc)
        assert np.all(np.isfinite(a))
        _check_accel(a, a_ref, S)
        if rc[0] > 1e5:
            assert np.all(a == 0.0)
        m.close()


def test_accel_is_deterministic(M):
    w = W.make_config(1)
    m = _mk(M, w)
    m.accel(); a1 = m.get("a").copy()
    m.accel(); a2 = m.get("a")
    assert np.array_equal(a1, a2)
    m.close()


# ------------------------------------------------------------------------------ drift
@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_drift_all_configs(M, cfg):
    w = W.make_config(cfg)
    m = _mk(M, w)
    m.drift(w.dt)
    x, v = m.get("x"), m.get("v")
    st = m.stats()
    assert st.drift_fail == 0 and st.max_newton <= 8
    x_ref, v_ref, fl = oracle.drift(G * w.m_star, w.dt, w.x, w.v)
    assert not fl.any()
    assert _rel_vec_err(x, x_ref).max() <= 1e-13
    assert _rel_vec_err(v, v_ref).max() <= 1e-13
    m.close()


@pytest.mark.parametrize("dt", [-8.0, 0.37, 400.0, 5.0e4])
def test_drift_long_negative_and_eccentric(M, dt):
    rng = np.random.default_rng(3)
    nb = 2000
    a = rng.uniform(0.3, 40, nb); e = rng.uniform(0, 0.95, nb)
    mu = G
    x, v = W.elements_to_state(np.full(nb, mu), a, e, rng.uniform(0, 1.0, nb), rng.uniform(0, 6.28, nb),
                               rng.uniform(0, 6.28, nb), rng.uniform(0, 6.28, nb))
    m = M.Mopal(np.full(nb, 1e-12), x, v, np.zeros(nb))
    m.drift(dt)
    xg, vg = m.get("x"), m.get("v")
    assert m.stats().drift_fail == 0
    x_ref, v_ref, fl = oracle.drift(mu, dt, x, v)
    # conditioning: inputs are doubles; a relative change eps of the state moves the body by
    # ~eps * 3 pi * (#orbits) * (1+e)/(1-e) along the orbit -> scale the 1e-13 bar accordingly
    P = 2 * np.pi * np.sqrt(a**3 / mu)
    amp = 1 + 10 * np.abs(dt) / P * (1 + e) / (1 - e)
    assert np.max(_rel_vec_err(xg, x_ref) / amp) <= 1e-13
    assert np.max(_rel_vec_err(vg, v_ref) / (amp * (1 + e) / (1 - e))) <= 1e-13
    m.close()


def test_drift_failure_flag_and_hyperbolic(M):
    x = np.array([[0.0, 1.0, 1.0], [0.0, 0.0, 0.0], [0.0, 0.0, 0.0]])
    v = np.array([[0.01, 0.0, 0.0], [0.0, 0.017, 0.04], [0.0, 0.0, 0.001]])
    m = M.Mopal(np.full(3, 1e-12), x, v, np.zeros(3))
    m.drift(50.0)
    st = m.stats()
    assert st.drift_fail == 1 and st.status == M.MO_ENOCONV
    xg, vg = m.get("x"), m.get("v")
    assert np.all(xg[:, 0] == 0) and np.all(vg[:, 0] == v[:, 0])     # failed body untouched
    x_ref, v_ref, fl = oracle.drift(G, 50.0, x, v)
    assert fl.tolist() == [1, 0, 0]
    assert _rel_vec_err(xg[:, 1:], x_ref[:, 1:]).max() <= 1e-13      # bound and hyperbolic
    assert _rel_vec_err(vg[:, 1:], v_ref[:, 1:]).max() <= 1e-13
    m.close()


# ------------------------------------------------------------------------------ encounters
def _enc_inputs(w):
    x1, v1, fl = oracle.drift(G * w.m_star, w.dt, w.x, w.v)
    return x1, v1


@pytest.mark.parametrize("cfg,scale", [(0, 1.0), (1, 1.0), (2, 1.0), (2, 25.0)])
def test_encounters_full_configs(M, cfg, scale):
    """reading B-i: the harness drifts a saved copy to get (x0,v0)->(x1,v1)."""
    w = W.make_config(cfg)
    rcrit = w.rcrit * scale
    x1, v1 = _enc_inputs(w)
    ref = oracle.encounters(w.dt, w.x, w.v, x1, v1, rcrit)
    m = M.Mopal(w.mass, w.x, w.v, rcrit)
    m.snapshot()
    m.set("x", x1); m.set("v", v1)
    cnt = m.encounters(w.dt)
    got = m.pair_list(cnt)
    n_amb = _pairs_ok(got, ref)
    if n_amb == 0:
        assert cnt == ref["count"] and np.array_equal(got, ref["pairs"])
        assert np.array_equal(m.get("flag"), ref["flag"])
    assert got.tolist() == sorted(got.tolist())
    if scale > 1 or cfg < 2:
        assert cnt > 0
    m.close()


@pytest.mark.parametrize("cfg", [3, 4])
def test_encounters_headline_sizes_whole_list(M, cfg):
    """the WHOLE list at full size against the oracle's - the giants' rows 0..3 of cfg3 (thousands of hits each:
    the long-row ranking path of enc_rank_kernel) and the dense load of cfg4 included."""
    w = W.make_config(cfg)
    x1, v1 = _enc_inputs(w)
    ref = oracle.encounters(w.dt, w.x, w.v, x1, v1, w.rcrit, cap=1 << 20)
    m = _mk(M, w)
    m.snapshot()
    m.set("x", x1); m.set("v", v1)
    cnt = m.encounters(w.dt)
    got = m.pair_list(cnt)
    assert cnt == len(got) > 0
    n_amb = _pairs_ok(got, ref)
    if n_amb == 0:
        assert cnt == ref["count"] and np.array_equal(got, ref["pairs"])
        assert np.array_equal(m.get("flag"), ref["flag"])
    assert got.tolist() == sorted(got.tolist()) and np.all(got[:, 0] < got[:, 1])
    if cfg == 3:      # the giants' rows are long rows (> 64 hits: the CTA ranking path)
        assert min(np.sum(ref["pairs"][:, 0] == g) for g in range(2)) > 64
    m.close()


def _check_boxes(m, h, x0, v0, x1, v1, rcrit, nbig=None):
    """a7 directly: the library's boxes against oracle.boxes.  Both sides evaluate B-1 in the same operation
    order, so the plain-double build of the oracle must agree to the last bit and the long-double parity build to
    a few ulp of the box scale (measured between the two oracle builds: <= 7e-16)."""
    lo, hi = m.boxes()
    rl, rh = oracle.boxes(h, x0, v0, x1, v1, rcrit, nbig=nbig)
    sc = np.maximum(np.maximum(np.abs(rl), np.abs(rh)), 1e-300)
    assert np.max(np.abs(lo - rl) / sc) <= 4e-15 and np.max(np.abs(hi - rh) / sc) <= 4e-15
    dl, dh = oracle.boxes(h, x0, v0, x1, v1, rcrit, nbig=nbig, kind="f64")
    assert np.array_equal(lo, dl) and np.array_equal(hi, dh)
    return lo, hi


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_boxes_all_configs(M, cfg):
    """mce_snif LOOP 1-2 on every body of the five configs, stand-alone and inside mo_step."""
    w = W.make_config(cfg)
    x1, v1 = _enc_inputs(w)
    m = _mk(M, w)
    with pytest.raises(M.MopalError):
        m.boxes()                                  # no encounter pass yet
    m.snapshot(); m.set("x", x1); m.set("v", v1)
    m.encounters(w.dt)
    lo, hi = _check_boxes(m, w.dt, w.x, w.v, x1, v1, w.rcrit)
    turning = (w.v[:2] * v1[:2] < 0)
    assert turning.sum() >= 4                      # the interior-extremum branch is exercised
    ends_lo = np.minimum(w.x[:2], x1[:2]) - w.rcrit
    assert (lo[turning] < ends_lo[turning]).any() or (hi[turning] > (np.maximum(w.x[:2], x1[:2]) + w.rcrit)[turning]).any()
    # inside the step: the boxes are those of (x0, v0) -> drifted (x, v) of that step
    m.set("x", w.x); m.set("v", w.v)
    m.step(w.dt, 1)
    x0t, v0t = m.snapshot_tensors()
    x0, v0 = x0t[:, :w.nb].cpu().numpy(), v0t[:, :w.nb].cpu().numpy()
    xd, vd, _ = oracle.drift(G * w.m_star, w.dt, x0, v0)
    lo, hi = m.boxes()
    rl, rh = oracle.boxes(w.dt, x0, v0, xd, vd, w.rcrit)
    sc = np.maximum(np.abs(rl), np.abs(rh))
    assert np.max(np.abs(lo - rl) / sc) <= 1e-12 and np.max(np.abs(hi - rh) / sc) <= 1e-12   # drifted state to 1e-13
    m.close()


@pytest.mark.parametrize("nbig", [None, 37])
def test_boxes_planted_turning_points(M, nbig):
    """every branch of B-1 on planted (p0, w0) -> (p1, w1): one or two interior extrema, D < 0, k3 = 0 exactly,
    a root at the end of the interval, negative h; with nbig < nb only the big bodies' boxes are padded (R-2)."""
    import torch
    rng = np.random.default_rng(7)
    nb = 1200
    x0 = rng.uniform(-5, 5, (3, nb)); x1 = x0 + rng.normal(0, 0.05, (3, nb))
    v0 = rng.normal(0, 0.02, (3, nb)); v1 = v0.copy()
    v1[:2, ::2] = -v0[:2, ::2] * rng.uniform(0.2, 3.0, (2, nb // 2))          # turning points in x and y
    v1[:2, 1::4] = v0[:2, 1::4] * rng.uniform(0.2, 3.0, (2, nb // 4))          # same sign: endpoints only
    # k3 = 2 p0 + h w0 - 2 p1 + h w1 = 0 exactly: p1 = p0 + h (w0 + w1) / 2 with exactly representable numbers
    h = 4.0
    x0[0, :8] = [0.5, -1.25, 2.0, 3.5, -0.75, 1.0, 4.0, -2.5]; v0[0, :8] = 0.125; v1[0, :8] = -0.0625
    x1[0, :8] = x0[0, :8] + h * (0.125 - 0.0625) / 2
    x1[1, 8:16] = x0[1, 8:16]; v0[1, 8:16] = 0.25; v1[1, 8:16] = -0.25         # symmetric: extremum at tau = 1/2
    x1[0, 16:24] = x0[0, 16:24] + 10.0; v0[0, 16:24] = 1e-3; v1[0, 16:24] = -1e-3   # big jump: roots outside (0,1) or D < 0
    rc = rng.uniform(0.0, 0.3, nb)
    for hh in (h, -h):
        m = M.Mopal(np.full(nb, 1e-9), x1, v1, rc)
        if nbig is not None:
            m.set_nbig(nbig)
        X0 = torch.zeros_like(m.x); V0 = torch.zeros_like(m.v)
        X0[:, :nb] = torch.from_numpy(x0).cuda(); V0[:, :nb] = torch.from_numpy(v0).cuda()
        m.encounters(hh, X0, V0)
        lo, hi = _check_boxes(m, hh, x0, v0, x1, v1, rc, nbig=nbig)
        if nbig is not None:       # small bodies: no pad
            assert np.all(lo[:, nbig:] <= np.minimum(x0[:2], x1[:2])[:, nbig:])
            same = v0[:2, nbig:] * v1[:2, nbig:] >= 0
            assert np.array_equal(lo[:, nbig:][same], np.minimum(x0[:2], x1[:2])[:, nbig:][same])
        m.close()


def test_encounters_overflow_and_edges(M):
    w = W.shrink(0, 200)
    x1, v1 = _enc_inputs(w)
    huge = np.full(w.nb, 1e3)
    ref = oracle.encounters(w.dt, w.x, w.v, x1, v1, huge)
    total = w.nb * (w.nb - 1) // 2
    assert ref["count"] == total
    cap = 1000
    m = M.Mopal(w.mass, w.x, w.v, huge, cap=cap)
    m.snapshot(); m.set("x", x1); m.set("v", v1)
    cnt = m.encounters(w.dt)
    assert cnt == total                                       # true total past cap
    assert np.array_equal(m.pair_list(cnt), ref["pairs"][:cap])   # first cap pairs in sorted order
    assert m.get("flag").all()
    with pytest.raises(M.MopalError) as ei:
        m.encounters(w.dt, raise_on_overflow=True)
    assert ei.value.status == M.MO_EOVERFLOW
    m.close()
    # rcrit = 0: nothing; negative dt with start/end swapped: same list
    m = M.Mopal(w.mass, w.x, w.v, np.zeros(w.nb))
    m.snapshot(); m.set("x", x1); m.set("v", v1)
    assert m.encounters(w.dt) == 0 and not m.get("flag").any()
    m.close()
    rc = w.rcrit * 3
    ref = oracle.encounters(-w.dt, x1, v1, w.x, w.v, rc)
    m = M.Mopal(w.mass, x1, v1, rc)
    m.snapshot(); m.set("x", w.x); m.set("v", w.v)
    cnt = m.encounters(-w.dt)
    _pairs_ok(m.pair_list(cnt), ref)
    assert cnt > 0
    m.close()


def test_encounters_explicit_x0_v0_pointers(M):
    import torch
    w = W.shrink(1, 600)
    x1, v1 = _enc_inputs(w)
    ref = oracle.encounters(w.dt, w.x, w.v, x1, v1, w.rcrit)
    m = M.Mopal(w.mass, x1, v1, w.rcrit)
    x0 = torch.zeros_like(m.x); v0 = torch.zeros_like(m.v)
    x0[:, :w.nb] = torch.from_numpy(w.x).cuda(); v0[:, :w.nb] = torch.from_numpy(w.v).cuda()
    cnt = m.encounters(w.dt, x0, v0)
    _pairs_ok(m.pair_list(cnt), ref)
    m.close()


# ------------------------------------------------------------------------------ step
def _step_err(m, ref):
    return _rel_vec_err(m.get("x"), ref["x"]).max(), _rel_vec_err(m.get("v"), ref["v"]).max()


@pytest.mark.parametrize("cfg,nsteps", [(0, 10), (1, 3), (2, 1)])
def test_step_vs_oracle(M, cfg, nsteps):
    w = W.make_config(cfg)
    gm = G * w.mass
    mu = G * w.m_star
    m = _mk(M, w)
    a, _ = oracle.accel(gm, w.x, w.rcrit)
    x, v = w.x, w.v
    for k in range(nsteps):
        st = m.step(w.dt, 1)
        r = oracle.step(mu, gm, w.rcrit, w.dt, x, v, a)
        x, v, a = r["x"], r["v"], r["a"]
        ex, ev = _step_err(m, r)
        tol = 1e-13 * (1 + k)                     # graded: rounding differences grow (P-S6)
        assert ex <= tol and ev <= tol, (k, ex, ev)
        assert st.steps_done == k + 1 and st.drift_fail == 0
        got = m.pair_list(st.nce_last)
        _pairs_ok(got, r)
        if r["n_ambig"] == 0:
            assert st.nce_last == r["count"]
        # the snapshot is the oracle's x0, v0
        x0, v0 = m.snapshot_tensors()
        assert _rel_vec_err(x0[:, :w.nb].cpu().numpy(), r["x0"]).max() <= tol
        assert _rel_vec_err(v0[:, :w.nb].cpu().numpy(), r["v0"]).max() <= tol
    m.close()


def test_step_multi_equals_single_steps_and_graph_path(M):
    w = W.make_config(0)
    m1 = _mk(M, w); m2 = _mk(M, w)
    for _ in range(6):
        m1.step(w.dt, 1)
    st = m2.step(w.dt, 6)                        # CUDA-graph replay path
    assert st.steps_done == 6
    assert np.array_equal(m1.get("x"), m2.get("x")) and np.array_equal(m1.get("v"), m2.get("v"))
    assert m1.stats().nce_total == st.nce_total
    m1.close(); m2.close()


def test_step_nb1_and_reversibility(M):
    w = W.make_disk(N=2, seed=1, giants=[(1e-3, 5.2, 0.05, 0.02, 0.3)], a=("uniform", 1, 2), sig_e=0.01,
                    sig_i=0.01, mass=("equal", 1e-9), dt=8.0, steps=1)
    m = _mk(M, w)
    m.step(8.0, 1)
    r = oracle.step(G, G * w.mass, w.rcrit, 8.0, w.x, w.v, np.zeros((3, 1)))
    ex, ev = _step_err(m, r)
    assert ex <= 1e-13 and ev <= 1e-13
    m.close()
    w = W.make_config(0)
    m = _mk(M, w)
    m.step(w.dt, 5); m.step(-w.dt, 5)
    assert _rel_vec_err(m.get("x"), w.x).max() <= 1e-12 and _rel_vec_err(m.get("v"), w.v).max() <= 1e-12
    m.close()


@pytest.mark.parametrize("cfg", [3, 4])
def test_step_headline_sizes_vs_oracle(M, cfg):
    """P-S1 at full size: one mo_step against oracle.step - x, v, the snapshot x0 AND v0, the pair list and flags,
    and the closing accelerations on every row (against the oracle's sum at the stepped positions)."""
    w = W.make_config(cfg)
    gm, mu = G * w.mass, G * w.m_star
    a0, _ = oracle.accel(gm, w.x, w.rcrit)
    r = oracle.step(mu, gm, w.rcrit, w.dt, w.x, w.v, a0, cap=1 << 20)
    assert r["nfail"] == 0
    m = _mk(M, w)
    L0 = (w.mass * np.cross(w.x.T, w.v.T).T).sum(1)
    st = m.step(w.dt, 1)
    assert st.steps_done == 1 and st.drift_fail == 0
    x, v, a = m.get("x"), m.get("v"), m.get("a")
    assert _rel_vec_err(x, r["x"]).max() <= 1e-13 and _rel_vec_err(v, r["v"]).max() <= 1e-13
    x0, v0 = m.snapshot_tensors()
    assert _rel_vec_err(x0[:, :w.nb].cpu().numpy(), r["x0"]).max() <= 1e-13
    assert _rel_vec_err(v0[:, :w.nb].cpu().numpy(), r["v0"]).max() <= 1e-13
    got = m.pair_list(st.nce_last)
    n_amb = _pairs_ok(got, r)
    if n_amb == 0:
        assert st.nce_last == r["count"] and np.array_equal(got, r["pairs"]) and np.array_equal(m.get("flag"), r["flag"])
    # a is current for the GPU's x: the oracle's sum at those positions, every row
    a_ref, S = oracle.accel(gm, x, w.rcrit)
    _check_accel(a, a_ref, S, w.name + " after the step")
    L1 = (w.mass * np.cross(x.T, v.T).T).sum(1)
    assert np.linalg.norm(L1 - L0) <= 1e-13 * np.linalg.norm(L0)       # P-S2
    # two more steps through the graph path: invariants only (P-S6)
    st = m.step(w.dt, 2)
    x, v = m.get("x"), m.get("v")
    L2 = (w.mass * np.cross(x.T, v.T).T).sum(1)
    assert st.steps_done == 3 and np.linalg.norm(L2 - L0) <= 1e-13 * np.linalg.norm(L0)
    m.close()


# ------------------------------------------------------------------------------ boundary
def test_host_buffer_entry_points(M):
    import torch
    w = W.make_config(0)
    m = _mk(M, w)
    xh = torch.zeros((3, m.ld), dtype=torch.float64).pin_memory(); vh = torch.zeros_like(xh).pin_memory()
    xh[:, :w.nb] = torch.from_numpy(w.x); vh[:, :w.nb] = torch.from_numpy(w.v)
    ah = torch.zeros_like(xh).pin_memory()
    m.accel_host(xh, ah)
    a_ref, S = oracle.accel(G * w.mass, w.x, w.rcrit)
    _check_accel(ah[:, :w.nb].numpy(), a_ref, S)
    ph = torch.zeros((4096, 2), dtype=torch.int32).pin_memory()
    st = m.step_host(w.dt, 2, xh, vh, rcrit_host=torch.from_numpy(w.rcrit), a_is_current=True, pairs_host=ph)
    m2 = _mk(M, w); st2 = m2.step(w.dt, 2)
    assert np.array_equal(xh[:, :w.nb].numpy(), m2.get("x")) and np.array_equal(vh[:, :w.nb].numpy(), m2.get("v"))
    assert st.nce_last == st2.nce_last and np.array_equal(ph[:st.nce_last].numpy(), m2.pair_list(st2.nce_last))
    m.close(); m2.close()


def test_invalid_arguments_and_bookkeeping(M):
    import ctypes as C
    w = W.shrink(0, 64)
    m = _mk(M, w)
    L = M.load()
    assert L.mo_step(m._ctx, 0.0, 1, None) == M.MO_EINVAL
    assert L.mo_step(m._ctx, float("nan"), 1, None) == M.MO_EINVAL
    assert L.mo_step(m._ctx, 1.0, -1, None) == M.MO_EINVAL
    assert L.mo_encounters(m._ctx, 1.0, None, None, None) == M.MO_EINVAL   # no snapshot yet
    ctx = C.c_void_p()
    assert L.mo_create(C.byref(ctx), 0, 0, 1.0, 1.0, None, None, None, None, None, None, 0, None, None) == M.MO_EINVAL
    assert L.mo_create(C.byref(ctx), 5, 5, 1.0, 1.0, m.mass.data_ptr(), m.x.data_ptr(), m.v.data_ptr(), m.a.data_ptr(),
                       m.rcrit.data_ptr(), None, 0, m.flag.data_ptr(), None) == M.MO_EINVAL   # ld % 4
    n0 = m.launch_count()
    m.accel()
    assert m.launch_count() == n0 + (1 if m.pair_kernel_name() == "pair_small_kernel" else 3) and m.workspace_bytes() > 0
    g = m.pair_geometry()
    assert g["ctas"] >= 1 and g["ipt"] in (1, 2)
    tf, ms = M.probe_fp64_peak(2)
    assert 5.0 < tf < 80.0
    m.close()


# ------------------------------------------------------------------------------ big x all
def _mk_big(M, w, nbig, rcrit=None, cap=1 << 20):
    m = _mk(M, w, rcrit=rcrit, cap=cap)
    m.set_nbig(nbig)
    return m


@pytest.mark.parametrize("cfg,N,nbig,scale", [(1, 1500, 2, 1.0), (3, 3000, 4, 20.0), (2, 1025, 100, 30.0),
                                             (2, 2500, 129, 30.0), (4, 700, 699, 50.0), (0, 256, 1, 1.0),
                                             (2, 9000, 8999, 10.0)])
def test_bigsmall_accel(M, cfg, N, nbig, scale):
    """sources are bodies 0..nbig-1 only, every body is a sink; sizes put the
    source boundary inside a tile, on a tile edge (128 + 1) and one short of nb."""
    w = W.shrink(cfg, N)
    rcrit = w.rcrit * scale
    m = _mk_big(M, w, nbig, rcrit=rcrit)
    m.accel()
    a = m.get("a")
    a_ref, S = oracle.accel(G * w.mass, w.x, rcrit, nbig=nbig)
    _check_accel(a, a_ref, S, f"{w.name} nbig={nbig}")
    if nbig < w.nb - 1:
        a_all, _ = oracle.accel(G * w.mass, w.x, rcrit)
        assert not np.array_equal(a_ref, a_all)
    # back to fully interacting on the same context
    m.set_nbig(w.nb)
    m.accel()
    a_ref, S = oracle.accel(G * w.mass, w.x, rcrit)
    _check_accel(m.get("a"), a_ref, S, f"{w.name} back to nbig=nb")
    m.close()


@pytest.mark.parametrize("cfg,N,nbig,scale", [(1, 1500, 2, 1.0), (3, 3000, 4, 1.0), (2, 1025, 100, 40.0),
                                             (4, 2000, 150, 60.0), (4, 700, 699, 50.0), (4, 3000, 1, 500.0)])
def test_bigsmall_encounters(M, cfg, N, nbig, scale):
    """boxes of the big bodies only are padded, first pair members are big."""
    w = W.shrink(cfg, N)
    rcrit = w.rcrit * scale
    x1, v1 = _enc_inputs(w)
    ref = oracle.encounters(w.dt, w.x, w.v, x1, v1, rcrit, nbig=nbig)
    m = _mk_big(M, w, nbig, rcrit=rcrit)
    m.snapshot()
    m.set("x", x1); m.set("v", v1)
    cnt = m.encounters(w.dt)
    got = m.pair_list(cnt)
    n_amb = _pairs_ok(got, ref)
    assert cnt > 0 and np.all(got[:, 0] < nbig) and np.all(got[:, 0] < got[:, 1])
    if n_amb == 0:
        assert cnt == ref["count"] and np.array_equal(got, ref["pairs"])
        assert np.array_equal(m.get("flag"), ref["flag"])
    full = oracle.encounters(w.dt, w.x, w.v, x1, v1, rcrit)
    if nbig < w.nb - 1 and scale > 1:
        assert full["count"] != ref["count"]
    m.close()


def test_bigsmall_encounters_overflow(M):
    w = W.shrink(4, 600)
    nbig = 5
    huge = np.full(w.nb, 1e3)
    x1, v1 = _enc_inputs(w)
    ref = oracle.encounters(w.dt, w.x, w.v, x1, v1, huge, nbig=nbig)
    total = sum(w.nb - 1 - i for i in range(nbig))
    assert ref["count"] == total
    cap = 700
    m = _mk_big(M, w, nbig, rcrit=huge, cap=cap)
    m.snapshot(); m.set("x", x1); m.set("v", v1)
    cnt = m.encounters(w.dt)
    assert cnt == total and np.array_equal(m.pair_list(cnt), ref["pairs"][:cap])
    assert m.get("flag").all()
    m.close()


@pytest.mark.parametrize("cfg,N,nbig,nsteps", [(1, 1200, 2, 4), (3, 2000, 4, 3), (2, 1500, 130, 2)])
def test_bigsmall_step_vs_oracle(M, cfg, N, nbig, nsteps):
    w = W.shrink(cfg, N)
    mass = w.mass.copy()
    if cfg != 2:
        mass[nbig:] = 0.0               # massless small bodies; cfg 2 keeps them massive: P still sums all
    gm = G * mass
    mu = G * w.m_star
    m = M.Mopal(mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G)
    m.set_nbig(nbig)
    a, _ = oracle.accel(gm, w.x, w.rcrit, nbig=nbig)
    x, v = w.x, w.v
    for k in range(nsteps):
        st = m.step(w.dt, 1)
        r = oracle.step(mu, gm, w.rcrit, w.dt, x, v, a, nbig=nbig)
        x, v, a = r["x"], r["v"], r["a"]
        ex, ev = _step_err(m, r)
        tol = 1e-13 * (1 + k)
        assert ex <= tol and ev <= tol, (k, ex, ev)
        got = m.pair_list(st.nce_last)
        _pairs_ok(got, r)
        if r["n_ambig"] == 0:
            assert st.nce_last == r["count"]
        assert np.all(got[:, 0] < nbig)
    # graph-replay path with nbig set
    m2 = M.Mopal(mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G)
    m2.set_nbig(nbig)
    st2 = m2.step(w.dt, nsteps)
    assert np.array_equal(m.get("x"), m2.get("x")) and np.array_equal(m.get("v"), m2.get("v"))
    assert st2.nce_last == st.nce_last
    m.close(); m2.close()


@pytest.mark.parametrize("N,nbig", [(262_144, 100), (1_000_000, 36)])
def test_bigsmall_production_sizes(M, N, nbig):
    """the paper's production regime (N_big <= 100, N_small up to 1e6): every big row
    of the encounter list against the oracle, sampled accel rows, invariants after steps."""
    w = W.make_bigsmall(N, nbig)
    gm = G * w.mass
    m = _mk_big(M, w, nbig)
    m.accel()
    rows = np.unique(np.concatenate([np.arange(min(nbig + 3, w.nb)),
                                     np.random.default_rng(2).integers(0, w.nb, 40)])).astype(np.int32)
    a_ref, S = oracle.accel_rows(gm, w.x, w.rcrit, rows, nbig=nbig)
    _check_accel(m.get("a")[:, rows], a_ref, S, w.name)
    x1, v1 = _enc_inputs(w)
    m.snapshot(); m.set("x", x1); m.set("v", v1)
    cnt = m.encounters(w.dt)
    got = m.pair_list(cnt)
    ref = oracle.encounters(w.dt, w.x, w.v, x1, v1, w.rcrit, nbig=nbig, cap=1 << 20)
    n_amb = _pairs_ok(got, ref)
    assert cnt > 0
    if n_amb == 0:
        assert np.array_equal(got, ref["pairs"]) and np.array_equal(m.get("flag"), ref["flag"])
    m.set("x", w.x); m.set("v", w.v); m.invalidate_accel()
    st = m.step(w.dt, 2)
    assert st.steps_done == 2 and st.drift_fail == 0
    x, v = m.get("x"), m.get("v")
    a_ref, S = oracle.accel_rows(gm, x, w.rcrit, rows, nbig=nbig)
    _check_accel(m.get("a")[:, rows], a_ref, S, w.name + " after 2 steps")
    m.close()


def test_bigsmall_invalid(M):
    w = W.shrink(0, 64)
    m = _mk(M, w)
    L = M.load()
    assert L.mo_set_nbig(m._ctx, 0) == M.MO_EINVAL
    assert L.mo_set_nbig(m._ctx, w.nb + 1) == M.MO_EINVAL
    assert L.mo_set_nbig(None, 1) == M.MO_EINVAL
    assert L.mo_set_nbig(m._ctx, w.nb) == M.MO_OK
    m.close()


# ------------------------------------------------------------------------------ support routines
@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_support_h2dh_dh2h(M, cfg):
    w = W.make_config(cfg)
    m = _mk(M, w)
    m.dh2h()
    vh = m.get("v")
    ref = oracle.dh2h(w.m_star, w.mass, w.v)
    assert _rel_vec_err(vh, ref).max() <= 1e-15
    m.h2dh()
    back = oracle.h2dh(w.m_star, w.mass, ref)
    assert _rel_vec_err(m.get("v"), back).max() <= 1e-15
    assert _rel_vec_err(m.get("v"), w.v).max() <= 1e-15
    assert np.array_equal(m.get("x"), w.x)
    m.close()


@pytest.mark.parametrize("cfg,mode,n_hill", [(0, 0, 3.0), (1, 1, 3.0), (2, 0, 2.5), (3, 1, 3.0), (4, 0, 3.0)])
def test_support_hill(M, cfg, mode, n_hill):
    import torch
    w = W.make_config(cfg)
    m = _mk(M, w, rcrit=np.zeros(w.nb))
    rh_t = torch.zeros(w.nb, dtype=torch.float64, device=m.device)
    m.hill(n_hill, mode, rhill=rh_t)
    rh, rc = oracle.hill(G, w.m_star, w.mass, w.x, w.v, n_hill=n_hill, mode=mode)
    got_rc, got_rh = m.get("rcrit"), rh_t.cpu().numpy()
    tol = 2e-15 if mode == 0 else 1e-13          # mode 1: 1/a = 2/r - v^2/mu cancels ~2x, eccentric orbits more
    assert np.max(np.abs(got_rh - rh) / rh) <= tol and np.max(np.abs(got_rc - rc) / rc) <= tol
    if mode == 1 and cfg in (1, 3):
        assert np.max(np.abs(got_rc - w.rcrit) / w.rcrit) <= 1e-11     # the generator's radii
    m.close()


@pytest.mark.parametrize("cfg,N,nbig", [(0, 256, None), (1, 3000, None), (2, 5000, 300), (1, 2000, 2), (4, 1025, 1024)])
def test_support_energy(M, cfg, N, nbig):
    w = W.shrink(cfg, N) if N != W.make_config(cfg).N else W.make_config(cfg)
    m = _mk(M, w)
    if nbig is not None:
        m.set_nbig(nbig)
    got = m.energy()
    ref = oracle.energy(G, w.m_star, w.mass, w.x, w.v, nbig=nbig)
    for k in ("T", "Us", "Up"):
        assert abs(got[k] - ref[k]) <= 1e-13 * abs(ref[k]) + 1e-300, (k, got[k], ref[k])
    assert abs(got["E"] - ref["E"]) <= 1e-12 * ref["Eabs"]
    assert np.all(np.abs(got["L"] - ref["L"]) <= 1e-12 * ref["Labs"])
    g2 = m.energy()
    assert g2["E"] == got["E"] and np.array_equal(g2["L"], got["L"])      # deterministic
    m.close()


def test_support_energy_headline_size_and_conservation(M):
    """full cfg3: pair potential over 2.1e9 pairs against the oracle's (OpenMP, a few seconds); then the
    hybrid step conserves E to ~dt^2 and L to rounding."""
    w = W.make_config(3)
    m = _mk(M, w)
    e0 = m.energy()
    ref = oracle.energy(G, w.m_star, w.mass, w.x, w.v)
    assert abs(e0["Up"] - ref["Up"]) <= 1e-12 * abs(ref["Up"])
    assert abs(e0["E"] - ref["E"]) <= 1e-12 * ref["Eabs"]
    m.step(w.dt, 5)
    e1 = m.energy()
    assert abs(e1["E"] - e0["E"]) <= 1e-6 * abs(e0["E"])
    assert np.linalg.norm(e1["L"] - e0["L"]) <= 1e-12 * np.linalg.norm(e0["L"])
    m.close()


@pytest.mark.parametrize("cfg,N,mode,nbig", [(1, 1500, 0, None), (3, 2500, 1, None), (1, 1200, 0, 2)])
def test_support_hill_inside_step(M, cfg, N, mode, nbig):
    """mo_set_hill: rcrit recomputed from the state at the start of every step."""
    w = W.shrink(cfg, N)
    gm, mu = G * w.mass, G * w.m_star
    m = _mk(M, w)
    if nbig is not None:
        m.set_nbig(nbig)
    m.set_hill(3.0, mode)
    a, _ = oracle.accel(gm, w.x, w.rcrit, nbig=nbig)
    x, v = w.x, w.v
    for k in range(3):
        st = m.step(w.dt, 1)
        _, rc = oracle.hill(G, w.m_star, w.mass, x, v, n_hill=3.0, mode=mode)
        r = oracle.step(mu, gm, rc, w.dt, x, v, a, nbig=nbig)
        x, v, a = r["x"], r["v"], r["a"]
        ex, ev = _step_err(m, r)
        tol = 1e-13 * (1 + k)
        assert ex <= tol and ev <= tol, (k, ex, ev)
        assert np.max(np.abs(m.get("rcrit") - rc) / rc.clip(1e-300)) <= (2e-15 if mode == 0 else 1e-12)
        got = m.pair_list(st.nce_last)
        # rcrit differs from the oracle's in the last bits: threshold pairs are the oracle's ambiguous ones
        _pairs_ok(got, r)
    # graph replay path gives the same trajectory
    m2 = _mk(M, w)
    if nbig is not None:
        m2.set_nbig(nbig)
    m2.set_hill(3.0, mode)
    m2.step(w.dt, 3)
    assert np.array_equal(m.get("x"), m2.get("x")) and np.array_equal(m.get("v"), m2.get("v"))
    m2.set_hill(0.0, -1)
    m.close(); m2.close()


def test_support_invalid(M):
    w = W.shrink(0, 64)
    m = _mk(M, w)
    L = M.load()
    assert L.mo_hill(m._ctx, 3.0, 2, None) == M.MO_EINVAL
    assert L.mo_hill(m._ctx, float("nan"), 0, None) == M.MO_EINVAL
    assert L.mo_hill(m._ctx, -1.0, 0, None) == M.MO_EINVAL
    assert L.mo_set_hill(m._ctx, 3.0, 5) == M.MO_EINVAL
    assert L.mo_energy(m._ctx, None) == M.MO_EINVAL
    assert L.mo_h2dh(None) == M.MO_EINVAL and L.mo_dh2h(None) == M.MO_EINVAL
    m.close()


# ------------------------------------------------------------------------------ single-CTA step front end (nb <= 1024)
@pytest.mark.parametrize("cfg,N,nbig,hill", [(1, 1025, None, -1), (1, 700, None, 0), (3, 900, None, 1), (1, 800, 2, -1),
                                            (4, 333, 100, 0), (2, 33, None, -1)])
def test_step_small_path_vs_oracle(M, monkeypatch, cfg, N, nbig, hill):
    """nb <= 1024: hill, kick, jump, snapshot, drift, boxes, pair test and second jump run in one kernel."""
    monkeypatch.setenv("MO_SMALL_MAX", "1024")
    w = W.shrink(cfg, N)
    scale = 40.0 if cfg in (2, 4) else 1.0
    rc0 = w.rcrit * scale
    gm, mu = G * w.mass, G * w.m_star
    m = _mk(M, w, rcrit=rc0)
    if nbig is not None:
        m.set_nbig(nbig)
    if hill >= 0:
        m.set_hill(3.0 * scale, hill)
    a, _ = oracle.accel(gm, w.x, rc0, nbig=nbig)
    x, v, rc = w.x, w.v, rc0
    seen = 0
    for k in range(4):
        st = m.step(w.dt, 1)
        if hill >= 0:
            _, rc = oracle.hill(G, w.m_star, w.mass, x, v, n_hill=3.0 * scale, mode=hill)
        r = oracle.step(mu, gm, rc, w.dt, x, v, a, nbig=nbig)
        x, v, a = r["x"], r["v"], r["a"]
        ex, ev = _step_err(m, r)
        tol = 1e-13 * (1 + k)
        assert ex <= tol and ev <= tol, (k, ex, ev)
        assert st.steps_done == k + 1 and st.drift_fail == 0
        got = m.pair_list(st.nce_last)
        _pairs_ok(got, r)
        assert got.tolist() == sorted(got.tolist())
        if r["n_ambig"] == 0:
            assert st.nce_last == r["count"] and np.array_equal(m.get("flag"), r["flag"])
        seen += st.nce_last
        x0, v0 = m.snapshot_tensors()
        assert _rel_vec_err(x0[:, :w.nb].cpu().numpy(), r["x0"]).max() <= tol
        assert _rel_vec_err(v0[:, :w.nb].cpu().numpy(), r["v0"]).max() <= tol
    assert seen > 0 or cfg == 2
    m2 = _mk(M, w, rcrit=rc0)                       # graph replay gives the same trajectory
    if nbig is not None:
        m2.set_nbig(nbig)
    if hill >= 0:
        m2.set_hill(3.0 * scale, hill)
    st2 = m2.step(w.dt, 4)
    assert np.array_equal(m.get("x"), m2.get("x")) and np.array_equal(m.get("v"), m2.get("v"))
    assert st2.nce_last == st.nce_last and st2.nce_total == seen
    m.close(); m2.close()


def test_step_small_path_overflow_and_large_path_agree(M, monkeypatch):
    monkeypatch.setenv("MO_SMALL_MAX", "1024")
    w = W.shrink(4, 500)
    huge = np.full(w.nb, 1e3)
    total = w.nb * (w.nb - 1) // 2
    m = M.Mopal(w.mass, w.x, w.v, huge, cap=777)
    st = m.step(w.dt, 1)
    assert st.status == M.MO_EOVERFLOW
    assert st.nce_last == total and m.get("flag").all()
    got = m.pair_list(st.nce_last)
    ref = [(i, j) for i in range(w.nb) for j in range(i + 1, w.nb)][:777]
    assert got.tolist() == [list(t) for t in ref]
    m.close()
    # the multi-kernel front end (MO_SMALL=0) and the single-CTA one agree to rounding of the two 3-vector sums
    w = W.shrink(1, 900)
    m1 = _mk(M, w); s1 = m1.step(w.dt, 3)
    monkeypatch.setenv("MO_SMALL", "0")
    m2 = _mk(M, w); s2 = m2.step(w.dt, 3)
    monkeypatch.delenv("MO_SMALL")
    assert _rel_vec_err(m1.get("x"), m2.get("x")).max() <= 1e-14 and _rel_vec_err(m1.get("v"), m2.get("v")).max() <= 1e-14
    assert s1.nce_last == s2.nce_last and np.array_equal(m1.pair_list(s1.nce_last), m2.pair_list(s2.nce_last))
    m1.close(); m2.close()


# ------------------------------------------------------------------------------ encounter resolution
# Parity criterion: the kernel has its own step-size / order controller, so
# nothing is compared step for step.  What the paper fixes (PAPER.md:104 fn. 14) is the solution of the encounter
# equations over the step: the kernel's states agree with the oracle's to RES_RTOL(tol) = 20 tol + 5e-14 (each side
# controls its local error to tol relative to |x_i|, |v_i|; a handful of BS steps; FP64 rounding of a few 1e-16 per
# operation on the kernel's side), and with an independent DOP853 integration of the same equations to DOP_RTOL.
def RES_RTOL(tol):
    return 20.0 * tol + 5e-14


DOP_RTOL = 2e-11         # DOP853 at rtol 1e-13 itself (the oracle's own pin uses the same bound)


def _close_pair_system(sep, m=1e-5, extra=600, seed=3):
    """two massive bodies `sep` apart on neighbouring orbits at 1 AU inside a small disk (cfg1 recipe, shrunk)"""
    w = W.shrink(1, extra + 3, seed=seed)
    a = np.array([1.0, 1.0 + 0.6 * sep]); e = np.array([0.01, 0.012]); inc = np.array([0.001, 0.002])
    z = np.zeros(2); Man = np.array([0.3, 0.3 + 0.8 * sep])
    mass = w.mass.copy(); mass[2:4] = m
    x2, vh2 = W.elements_to_state(G * (w.m_star + m), a, e, inc, z, z, Man)
    x = w.x.copy(); x[:, 2:4] = x2
    vh = oracle.dh2h(w.m_star, w.mass, w.v); vh[:, 2:4] = vh2
    v = oracle.h2dh(w.m_star, mass, vh)
    _, rc = oracle.hill(G, w.m_star, mass, x, v, n_hill=3.0)
    return w, mass, x, v, rc


def _dop853_encounter(mu, gm, rc, h, x, v, pairs):
    """the encounter equations (reading X-2) of ALL listed bodies under ALL listed pairs, integrated by scipy's DOP853"""
    from scipy.integrate import solve_ivp
    idx = np.unique(pairs)
    loc = {b: k for k, b in enumerate(idx)}
    n = len(idx)

    def rhs(t, y):
        X = y[:3 * n].reshape(n, 3); V = y[3 * n:].reshape(n, 3)
        A = -mu * X / np.linalg.norm(X, axis=1)[:, None] ** 3
        for i, j in pairs:
            d = X[loc[j]] - X[loc[i]]
            r = np.linalg.norm(d)
            if r > 0:
                u = (1.0 - oracle.changeover(r, max(rc[i], rc[j]))) / r**3
                A[loc[i]] += gm[j] * u * d
                A[loc[j]] -= gm[i] * u * d
        return np.concatenate([V.ravel(), A.ravel()])

    y0 = np.concatenate([x[:, idx].T.ravel(), v[:, idx].T.ravel()])
    sol = solve_ivp(rhs, (0.0, h), y0, method="DOP853", rtol=1e-13, atol=1e-18)
    assert sol.success
    return idx, sol.y[:3 * n, -1].reshape(n, 3).T, sol.y[3 * n:, -1].reshape(n, 3).T


def _gpu_resolve(M, mass, x0, v0, x1, v1, rc, m_star, dt, tol, pairs_ref, nbig=None):
    m = M.Mopal(mass, x0, v0, rc, m_star=m_star, G=G)
    if nbig is not None:
        m.set_nbig(nbig)
    m.snapshot(); m.set("x", x1); m.set("v", v1)
    cnt = m.encounters(dt)
    assert np.array_equal(m.pair_list(cnt), pairs_ref)
    m.resolve(dt, tol)
    st = m.resolve_stats()
    gx, gv = m.get("x"), m.get("v")
    stats = m.stats()
    m.close()
    return gx, gv, st, stats


@pytest.mark.parametrize("sep,dt,tol", [(0.01, 2.0, 1e-12), (0.003, 1.0, 1e-13), (0.02, -3.0, 1e-12), (0.0009, 0.5, 1e-12)])
def test_resolve_vs_oracle_and_dop853(M, sep, dt, tol):
    w, mass, x, v, rc = _close_pair_system(sep)
    mu, gm = G * w.m_star, G * mass
    x1, v1, _ = oracle.drift(mu, dt, x, v)
    enc = oracle.encounters(dt, x, v, x1, v1, rc)
    assert enc["count"] >= 3 and [2, 3] in enc["pairs"].tolist()
    ref = oracle.resolve(mu, gm, rc, dt, x, v, x1, v1, enc["pairs"], tol=tol)
    gx, gv, st, _ = _gpu_resolve(M, mass, x, v, x1, v1, rc, w.m_star, dt, tol, enc["pairs"])
    assert st["fail"] == 0 and st["bodies"] == ref["n"] and st["steps"] >= 1 and st["rhs"] >= 3
    idx = np.unique(enc["pairs"]); rest = np.setdiff1d(np.arange(w.nb), idx)
    assert _rel_vec_err(gx[:, idx], ref["x"][:, idx]).max() <= RES_RTOL(tol) and _rel_vec_err(gv[:, idx], ref["v"][:, idx]).max() <= RES_RTOL(tol)
    assert np.array_equal(gx[:, rest], x1[:, rest]) and np.array_equal(gv[:, rest], v1[:, rest])
    assert _rel_vec_err(gv[:, 2:4], v1[:, 2:4]).max() > 1e-8          # the encounter matters
    # an integrator that shares nothing with either side
    didx, xd, vd = _dop853_encounter(mu, gm, rc, dt, x, v, enc["pairs"])
    assert _rel_vec_err(gx[:, didx], xd).max() <= DOP_RTOL and _rel_vec_err(gv[:, didx], vd).max() <= DOP_RTOL


def test_resolve_several_components_interleaved(M):
    """three interacting components whose members interleave in body order (the oracle's pin X-1 system), in a disk"""
    from tests.test_oracle_resolve import _multi_component_system
    m_star, mass9, x9, v9, rc9, pairs9 = _multi_component_system()
    w = W.shrink(1, 400, seed=11)
    mass = np.concatenate([mass9, w.mass[2:]]); x = np.concatenate([x9, w.x[:, 2:]], axis=1)
    vh = np.concatenate([oracle.dh2h(m_star, mass9, v9), oracle.dh2h(w.m_star, w.mass, w.v)[:, 2:]], axis=1)
    v = oracle.h2dh(m_star, mass, vh)
    _, rc = oracle.hill(G, m_star, mass, x, v, n_hill=3.0)
    mu, gm, dt, tol = G * m_star, G * mass, 2.0, 1e-13
    x1, v1, _ = oracle.drift(mu, dt, x, v)
    enc = oracle.encounters(dt, x, v, x1, v1, rc)
    got = {tuple(p) for p in enc["pairs"].tolist()}
    assert {tuple(p) for p in pairs9.tolist()} <= got
    ref = oracle.resolve(mu, gm, rc, dt, x, v, x1, v1, enc["pairs"], tol=tol)
    gx, gv, st, _ = _gpu_resolve(M, mass, x, v, x1, v1, rc, m_star, dt, tol, enc["pairs"])
    idx = np.unique(enc["pairs"])
    assert st["fail"] == 0 and st["bodies"] == len(idx) == ref["n"]
    assert _rel_vec_err(gx[:, idx], ref["x"][:, idx]).max() <= RES_RTOL(tol) and _rel_vec_err(gv[:, idx], ref["v"][:, idx]).max() <= RES_RTOL(tol)
    didx, xd, vd = _dop853_encounter(mu, gm, rc, dt, x, v, enc["pairs"])       # ONE integration of the union system
    assert _rel_vec_err(gx[:, didx], xd).max() <= DOP_RTOL and _rel_vec_err(gv[:, didx], vd).max() <= DOP_RTOL
    for b in range(7):
        assert np.linalg.norm(gv[:, b] - v1[:, b]) / np.linalg.norm(v1[:, b]) > 1e-8, b


@pytest.mark.parametrize("cfg,N", [(0, 256), (1, 1500), (3, 3000), (3, 9000), (4, 24000)])
def test_resolve_inside_step_vs_oracle(M, cfg, N):
    """mo_set_resolve: kick, jump, snapshot, drift, encounter check, encounter solve, jump, accel, kick.  From 2561 bodies
    on the solve runs BESIDE the pair sum (fixup.cuh: the sum over the drifted positions, then the flagged bodies' terms
    exchanged and their own rows recomputed) - the result is the same step.  (4, 24000): planetesimal pairs only, no long
    chain - after the first step the device flag sends the step the other way (solve, then the pair sum), both in the graph."""
    w = W.make_config(cfg) if N == 256 else W.shrink(cfg, N)
    mu, gm = G * w.m_star, G * w.mass
    m = _mk(M, w)
    m.set_resolve(1e-12)
    a, _ = oracle.accel(gm, w.x, w.rcrit)
    x, v = w.x, w.v
    nres = 0
    for k in range(3):
        st = m.step(w.dt, 1)
        v = oracle.kick(0.5 * w.dt, v, a)
        x, _ = oracle.jump(0.5 * w.dt, mu, gm, x, v)
        x0, v0 = x.copy(), v.copy()
        x, v, _ = oracle.drift(mu, w.dt, x, v)
        enc = oracle.encounters(w.dt, x0, v0, x, v, w.rcrit)
        if enc["count"] > 0:
            r = oracle.resolve(mu, gm, w.rcrit, w.dt, x0, v0, x, v, enc["pairs"])
            assert r["fail"] == 0
            x, v = r["x"], r["v"]
            rs = m.resolve_stats()
            assert rs["fail"] == 0 and rs["bodies"] == r["n"]
            nres += 1
        x, _ = oracle.jump(0.5 * w.dt, mu, gm, x, v)
        a, _ = oracle.accel(gm, x, w.rcrit)
        v = oracle.kick(0.5 * w.dt, v, a)
        tol = (RES_RTOL(1e-12) + 2e-13) * (1 + k)
        assert _rel_vec_err(m.get("x"), x).max() <= tol and _rel_vec_err(m.get("v"), v).max() <= tol, k
        assert st.nce_last == enc["count"] and st.resolve_fail == 0
    assert nres == 3 or cfg == 4
    m2 = _mk(M, w); m2.set_resolve(1e-12); m2.step(w.dt, 3)           # graph replay: bit for bit the same
    assert np.array_equal(m.get("x"), m2.get("x")) and np.array_equal(m.get("v"), m2.get("v"))
    m.close(); m2.close()


def test_resolve_inside_step_headline_size(M):
    """one resolving step at cfg3 (N = 65,536: the giants' stars in clusters of CTAs, the solve beside the pair sum in two
    launches, the flagged bodies' terms exchanged) against the oracle's kick / jump / drift / encounters / resolve / jump /
    accel / kick"""
    w = W.make_config(3)
    mu, gm = G * w.m_star, G * w.mass
    m = _mk(M, w)
    m.set_resolve(1e-12)
    st = m.step(w.dt, 1)
    a, _ = oracle.accel(gm, w.x, w.rcrit)
    v = oracle.kick(0.5 * w.dt, w.v, a)
    x, _ = oracle.jump(0.5 * w.dt, mu, gm, w.x, v)
    x0, v0 = x.copy(), v.copy()
    x, v, _ = oracle.drift(mu, w.dt, x, v)
    enc = oracle.encounters(w.dt, x0, v0, x, v, w.rcrit)
    assert enc["count"] > 500 and st.nce_last == enc["count"] and np.array_equal(m.pair_list(st.nce_last), enc["pairs"])
    r = oracle.resolve(mu, gm, w.rcrit, w.dt, x0, v0, x, v, enc["pairs"])
    assert r["fail"] == 0
    rs = m.resolve_stats()
    assert rs["fail"] == 0 and rs["bodies"] == r["n"] and st.resolve_fail == 0
    x, v = r["x"], r["v"]
    x, _ = oracle.jump(0.5 * w.dt, mu, gm, x, v)
    a, S = oracle.accel(gm, x, w.rcrit)
    v = oracle.kick(0.5 * w.dt, v, a)
    # the flagged bodies that pass a giant closely scatter (see test_resolve_big_star_components): positions to 1e-10 for
    # them - and their accelerations, dominated by the giant 0.02-1 AU away, follow their positions (3 dr / r): 1e-7 S
    idx = np.unique(enc["pairs"]); rest = np.setdiff1d(np.arange(w.nb), idx)
    ag = m.get("a")
    assert np.all(np.abs(ag - a) <= 1e-7 * S) and np.median(np.abs(ag - a) / S) <= 1e-13
    # the strict check of the accelerations (pair sum over the drifted positions + exchanged terms of the flagged bodies +
    # their recomputed rows): against the oracle's sum at the kernel's OWN final positions, every body
    a2, S2 = oracle.accel(gm, m.get("x"), w.rcrit)
    _check_accel(ag, a2, S2, "cfg3 resolving step, accelerations at the step's own positions")
    tol = RES_RTOL(1e-12) + 2e-13
    assert _rel_vec_err(m.get("x")[:, rest], x[:, rest]).max() <= tol and _rel_vec_err(m.get("v")[:, rest], v[:, rest]).max() <= tol
    assert _rel_vec_err(m.get("x")[:, idx], x[:, idx]).max() <= 1e-10 and _rel_vec_err(m.get("v")[:, idx], v[:, idx]).max() <= 1e-10
    ex = _rel_vec_err(m.get("v")[:, idx], v[:, idx])
    assert np.median(ex) <= tol
    m.close()


def test_resolve_energy_and_a_dense_component(M):
    """through a close encounter the resolved step keeps the energy (mo_energy) orders of magnitude better"""
    w, mass, x, v, rc = _close_pair_system(0.004, m=3e-5, extra=300)
    out = []
    for tol in (1e-12, 0.0):
        m = M.Mopal(mass, x, v, rc, m_star=w.m_star, G=w.G)
        m.set_resolve(tol)
        e0 = m.energy()["E"]
        m.step(1.0, 30)
        out.append(abs(m.energy()["E"] - e0) / abs(e0))
        m.close()
    assert out[0] < 1e-7 and out[1] > 50 * out[0], out
    # every body paired with every other (huge radii: K = 0, the solve carries the whole mutual gravity): ONE component of
    # 250 bodies and 31,125 pairs - far beyond the shared-memory kernels, taken by resolve_stream_kernel
    w = W.shrink(4, 251)
    huge = np.full(w.nb, 1e3)
    mu, gm = G * w.m_star, G * w.mass
    x1, v1 = _enc_inputs(w)
    enc = oracle.encounters(w.dt, w.x, w.v, x1, v1, huge, cap=1 << 16)
    assert enc["count"] == w.nb * (w.nb - 1) // 2 > 1023
    ref = oracle.resolve(mu, gm, huge, w.dt, w.x, w.v, x1, v1, enc["pairs"])
    gx, gv, st, stats = _gpu_resolve(M, w.mass, w.x, w.v, x1, v1, huge, w.m_star, w.dt, 1e-12, enc["pairs"])
    assert st["fail"] == 0 and st["bodies"] == w.nb and stats.resolve_fail == 0
    assert _rel_vec_err(gx, ref["x"]).max() <= RES_RTOL(1e-12) and _rel_vec_err(gv, ref["v"]).max() <= RES_RTOL(1e-12)
    m = M.Mopal(w.mass, w.x, w.v, huge, cap=1 << 16)
    L = M.load()
    assert L.mo_resolve(m._ctx, 1.0, 1e-12) == M.MO_EINVAL                  # no snapshot yet
    m.snapshot()
    assert L.mo_resolve(m._ctx, 0.0, 1e-12) == M.MO_EINVAL and L.mo_resolve(m._ctx, 1.0, 0.0) == M.MO_EINVAL
    assert L.mo_resolve_stats(m._ctx, None) == M.MO_EINVAL and L.mo_set_resolve(None, 1.0) == M.MO_EINVAL
    m.close()


def test_resolve_truncated_list_is_reported(M):
    """more pairs than cap: the list is truncated, nothing can be resolved - the bodies keep the drift result, the failure is
    counted (sticky) and the step's status says so"""
    w = W.shrink(1, 1500)
    x1, v1 = _enc_inputs(w)
    m = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G, cap=4)
    m.snapshot(); m.set("x", x1); m.set("v", v1)
    assert m.encounters(w.dt) > 4
    m.resolve(w.dt, 1e-12)
    assert m.resolve_stats()["fail"] >= 1 and np.array_equal(m.get("x"), x1) and np.array_equal(m.get("v"), v1)
    assert m.stats().resolve_fail == 1
    m.close()
    m = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G, cap=4)
    m.set_resolve(1e-12)
    st = m.step(w.dt, 2)
    assert st.status == M.MO_EOVERFLOW and st.resolve_fail == 2          # overflow outranks MO_ERESOLVE; both are sticky
    m.close()


def _giant_star(K, rmin, seed_off=40):
    """a giant with K planetesimals inside its critical radius: one star component of K + 1 bodies"""
    rng = np.random.default_rng(seed_off + K)
    m_star, mg = 1.0, 1e-3
    ang = rng.uniform(0, 2 * np.pi, K); rad = rng.uniform(rmin, 0.85, K); zz = rng.uniform(-0.01, 0.01, K)
    xg = np.array([5.2, 0.0, 0.0])
    X = np.empty((3, K + 1)); X[:, 0] = xg
    X[0, 1:] = xg[0] + rad * np.cos(ang); X[1, 1:] = xg[1] + rad * np.sin(ang); X[2, 1:] = zz
    r = np.linalg.norm(X, axis=0)
    vc = np.sqrt(G * m_star / r)                                   # circular heliocentric speeds
    Vh = np.stack([-vc * X[1] / r, vc * X[0] / r, np.zeros(K + 1)])
    return m_star, mg, X, Vh, rad


@pytest.mark.parametrize("K,rmin", [(5, 0.1), (24, 0.1), (31, 0.1), (32, 0.1), (40, 0.05), (100, 0.02), (300, 0.02), (450, 0.1), (700, 0.15),
                                    (1500, 0.15)])
def test_resolve_big_star_components(M, K, rmin):
    """resolve_small_kernel (at most 31 pairs: a warp per column; K = 31 / 32 sit on either side of its limit), the size
    classes of resolve_solve_kernel (64 / 256 / 512 / 1024 threads), the warp-summed hub with its group sums, and - K = 1500 -
    resolve_stream_kernel, against the oracle.  Planetesimals that pass within a few 0.01 AU of the giant
    amplify the FP64 / long-double rounding difference (the flyby is a scattering): 1e-10 for them, the tolerance-derived
    bound for the bodies that stay farther than 0.3 AU."""
    m_star, mg, X, Vh, rad = _giant_star(K, rmin)
    mass = np.concatenate([[mg], np.full(K, 1e-9)])
    V = oracle.h2dh(m_star, mass, Vh)
    _, rc = oracle.hill(G, m_star, mass, X, V, n_hill=3.0)
    mu, gm, dt = G * m_star, G * mass, 8.0
    x1, v1, _ = oracle.drift(mu, dt, X, V)
    enc = oracle.encounters(dt, X, V, x1, v1, rc)
    assert enc["count"] >= K and (enc["pairs"][:K, 0] == 0).all()
    ref = oracle.resolve(mu, gm, rc, dt, X, V, x1, v1, enc["pairs"])
    assert ref["fail"] == 0 and ref["n"] == K + 1
    gx, gv, st, stats = _gpu_resolve(M, mass, X, V, x1, v1, rc, m_star, dt, 1e-12, enc["pairs"])
    assert st["fail"] == 0 and st["bodies"] == K + 1 and stats.resolve_fail == 0, st
    assert _rel_vec_err(gx, ref["x"]).max() <= 1e-10 and _rel_vec_err(gv, ref["v"]).max() <= 1e-10
    far = np.concatenate([[True], rad > 0.3])
    assert _rel_vec_err(gx[:, far], ref["x"][:, far]).max() <= RES_RTOL(1e-12) and _rel_vec_err(gv[:, far], ref["v"][:, far]).max() <= RES_RTOL(1e-12)
    assert _rel_vec_err(gv[:, :1], v1[:, :1]).max() > 1e-12               # the giant felt its planetesimals


def test_resolve_long_run_keeps_energy_and_angular_momentum(M):
    """300 steps of cfg1 (N = 4096, two giants: ~28,000 encounter pairs in all, a different pair list, component structure
    and launch path - beside or before the pair sum - every step).  No oracle at this length (declared: multi-step
    trajectories beyond ~10 steps are unpinned); what the method fixes instead: the angular momentum to rounding, the
    energy to the symplectic error of the step size, every component resolved - and the same run WITHOUT resolution
    loses energy two orders of magnitude faster (the encounters matter)."""
    w = W.make_config(1)
    out = {}
    for tol in (0.0, 1e-12):
        m = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G, cap=1 << 18)
        if tol > 0:
            m.set_resolve(tol)
        e0 = m.energy()
        st = m.step(w.dt, 300)
        e1 = m.energy()
        assert st.status == 0 and st.resolve_fail == 0 and st.drift_fail == 0 and st.nce_total > 10_000
        L0, L1 = np.array(e0["L"]), np.array(e1["L"])
        assert np.linalg.norm(L1 - L0) <= 1e-13 * np.linalg.norm(L0)
        out[tol] = abs((e1["E"] - e0["E"]) / e0["E"])
        m.close()
    assert out[1e-12] < 1e-8, out
    assert out[0.0] > 30 * out[1e-12], out


def test_resolve_more_star_components_than_clusters(M):
    """twelve giants on different orbits, each with a star of 80-100 planetesimals (64-255 pairs: the 256-thread class on
    clusters of 8 CTAs) and one with 300 (the 512-thread class): more components than the 8 clusters of a class, so a cluster
    takes several components one after the other - its barrier's phases, the warps without a body and the column /
    tableau / error exchange through the CTAs' shared memory carry over from one component to the next."""
    rng = np.random.default_rng(77)
    m_star, mg = 1.0, 1e-3
    Xs, masses, far = [], [], []
    for g in range(12):
        K = 300 if g == 5 else 80 + 2 * g
        a_g, th = 4.0 + 2.2 * g, 0.55 * g
        xg = a_g * np.array([np.cos(th), np.sin(th), 0.0])
        rmax = 0.6 * 3.0 * a_g * (mg / 3.0) ** (1.0 / 3.0)                 # inside 3 Hill radii
        ang = rng.uniform(0, 2 * np.pi, K); rad = rng.uniform(0.12 * rmax, rmax, K); zz = rng.uniform(-0.01, 0.01, K)
        X = np.empty((3, K + 1)); X[:, 0] = xg
        X[0, 1:] = xg[0] + rad * np.cos(ang); X[1, 1:] = xg[1] + rad * np.sin(ang); X[2, 1:] = zz
        Xs.append(X); masses.append(np.concatenate([[mg], np.full(K, 1e-9)])); far.append(np.concatenate([[True], rad > 0.4 * rmax]))
    X = np.concatenate(Xs, axis=1); mass = np.concatenate(masses); far = np.concatenate(far)
    r = np.linalg.norm(X, axis=0); vc = np.sqrt(G * m_star / r)
    Vh = np.stack([-vc * X[1] / r, vc * X[0] / r, np.zeros(X.shape[1])])
    V = oracle.h2dh(m_star, mass, Vh)
    _, rc = oracle.hill(G, m_star, mass, X, V, n_hill=3.0)
    mu, gm, dt, tol = G * m_star, G * mass, 8.0, 1e-12
    x1, v1, _ = oracle.drift(mu, dt, X, V)
    enc = oracle.encounters(dt, X, V, x1, v1, rc)
    ref = oracle.resolve(mu, gm, rc, dt, X, V, x1, v1, enc["pairs"])
    assert ref["fail"] == 0 and ref["n"] == X.shape[1]
    gx, gv, st, stats = _gpu_resolve(M, mass, X, V, x1, v1, rc, m_star, dt, tol, enc["pairs"])
    assert st["fail"] == 0 and stats.resolve_fail == 0 and st["bodies"] == X.shape[1], st
    assert _rel_vec_err(gx, ref["x"]).max() <= 1e-10 and _rel_vec_err(gv, ref["v"]).max() <= 1e-10
    assert _rel_vec_err(gx[:, far], ref["x"][:, far]).max() <= RES_RTOL(tol) and _rel_vec_err(gv[:, far], ref["v"][:, far]).max() <= RES_RTOL(tol)


def test_resolve_big_x_all_thousands_of_detached_systems(M):
    """the production regime at a size the oracle takes a second for (N = 250,000, nbig = 100: ~3,100 listed pairs, ~3,000
    test-particle systems): the label kernel's cluster path (more than 2048 pairs: 8 CTAs, scans and flags exchanged
    through their shared memory), the depth levels of resolve_small_kernel's dispatch, the detached systems' cores."""
    w = W.make_bigsmall(250_000, 100)
    mu, gm, dt, tol = G * w.m_star, G * w.mass, w.dt, 1e-12
    x1, v1, _ = oracle.drift(mu, dt, w.x, w.v)
    enc = oracle.encounters(dt, w.x, w.v, x1, v1, w.rcrit, nbig=100)
    assert enc["count"] > 2048
    ref = oracle.resolve(mu, gm, w.rcrit, dt, w.x, w.v, x1, v1, enc["pairs"])
    assert ref["fail"] == 0
    gx, gv, st, stats = _gpu_resolve(M, w.mass, w.x, w.v, x1, v1, w.rcrit, w.m_star, dt, tol, enc["pairs"], nbig=100)
    idx = np.unique(enc["pairs"]); rest = np.setdiff1d(np.arange(w.nb), idx)
    # counted: the bodies a system wrote back - every listed test particle, and the big bodies that feel another big body (a
    # big body whose partners are all massless feels nothing: it is integrated along in their systems, its drift stands)
    pr = enc["pairs"]; mm = (w.mass[pr[:, 0]] > 0) & (w.mass[pr[:, 1]] > 0)
    n_min = int((w.mass[idx] == 0).sum()) + len(np.unique(pr[mm]))
    assert st["fail"] == 0 and stats.resolve_fail == 0 and n_min <= st["bodies"] <= len(idx), (st, n_min, len(idx))
    ex, ev = _rel_vec_err(gx[:, idx], ref["x"][:, idx]), _rel_vec_err(gv[:, idx], ref["v"][:, idx])
    assert ex.max() <= 1e-10 and ev.max() <= 1e-10                        # (a grazing passage amplifies the FP64 / long-double difference)
    assert np.mean(ex <= RES_RTOL(tol)) > 0.99 and np.mean(ev <= RES_RTOL(tol)) > 0.99
    assert np.array_equal(gx[:, rest], x1[:, rest]) and np.array_equal(gv[:, rest], v1[:, rest])
    assert _rel_vec_err(gv[:, idx], v1[:, idx]).max() > 1e-8               # the encounters matter


@pytest.mark.parametrize("K", [60, 900])
def test_resolve_massless_planetesimals_are_detached(M, K):
    """big x all regime (mo_set_nbig): the K test particles inside a giant's radius are massless, the giant feels nothing.
    The kernel integrates every test particle in a system of its own (giant + particle) instead of one system of K + 1
    bodies; the oracle integrates them together - the same solution.  A second, massive neighbour keeps the bodies in
    its component together."""
    m_star, mg, X, Vh, rad = _giant_star(K, 0.05)
    # body 1: a massive embryo 0.3 AU from the giant; its own test-particle neighbours are NOT detachable
    mass = np.concatenate([[mg, 3e-7], np.zeros(K - 1)])
    V = oracle.h2dh(m_star, mass, Vh)
    _, rc = oracle.hill(G, m_star, mass, X, V, n_hill=3.0)
    rc[2:] = 0.0
    mu, gm, dt, tol = G * m_star, G * mass, 8.0, 1e-12
    x1, v1, _ = oracle.drift(mu, dt, X, V)
    enc = oracle.encounters(dt, X, V, x1, v1, rc, nbig=2)
    assert enc["count"] >= K and [0, 1] in enc["pairs"].tolist()
    ref = oracle.resolve(mu, gm, rc, dt, X, V, x1, v1, enc["pairs"])
    gx, gv, st, stats = _gpu_resolve(M, mass, X, V, x1, v1, rc, m_star, dt, tol, enc["pairs"], nbig=2)
    idx = np.unique(enc["pairs"])
    assert st["fail"] == 0 and stats.resolve_fail == 0 and st["bodies"] == len(idx), (st, len(idx))
    assert _rel_vec_err(gx[:, idx], ref["x"][:, idx]).max() <= 1e-10 and _rel_vec_err(gv[:, idx], ref["v"][:, idx]).max() <= 1e-10
    far = np.concatenate([[True], rad > 0.3])[idx]
    assert _rel_vec_err(gx[:, idx][:, far], ref["x"][:, idx][:, far]).max() <= RES_RTOL(tol)
    assert _rel_vec_err(gv[:, idx][:, far], ref["v"][:, idx][:, far]).max() <= RES_RTOL(tol)
    rest = np.setdiff1d(np.arange(K + 1), idx)
    assert np.array_equal(gx[:, rest], x1[:, rest])
    # without the embryo the giant has no massive partner: it keeps its Kepler drift bit for bit, every particle is detached
    mass2 = mass.copy(); mass2[1] = 0.0
    V2 = oracle.h2dh(m_star, mass2, Vh)
    x1b, v1b, _ = oracle.drift(mu, dt, X, V2)
    enc2 = oracle.encounters(dt, X, V2, x1b, v1b, rc, nbig=1)
    ref2 = oracle.resolve(mu, G * mass2, rc, dt, X, V2, x1b, v1b, enc2["pairs"])
    gx2, gv2, st2, _ = _gpu_resolve(M, mass2, X, V2, x1b, v1b, rc, m_star, dt, tol, enc2["pairs"], nbig=1)
    idx2 = np.unique(enc2["pairs"])
    assert st2["fail"] == 0 and st2["bodies"] == len(idx2) - 1
    assert np.array_equal(gx2[:, 0], x1b[:, 0]) and np.array_equal(gv2[:, 0], v1b[:, 0])
    assert _rel_vec_err(gx2[:, idx2], ref2["x"][:, idx2]).max() <= 1e-10 and _rel_vec_err(gv2[:, idx2], ref2["v"][:, idx2]).max() <= 1e-10


# ------------------------------------------------------------------------------ pair sum sharded over GPUs
class _SeqDist:
    """torch.distributed stand-in for ONE GPU: the 'ranks' are contexts stepped one after the other (nobody waits on
    anybody); all_reduce(SUM) is deferred until every rank has handed in its tensor, then each gets the sum."""
    class ReduceOp:
        SUM = "sum"

    def __init__(self, world):
        self.world, self.pending = world, []

    def all_reduce(self, t, op=None, group=None):
        self.pending.append(t)
        if len(self.pending) == self.world:
            tot = self.pending[0].clone()
            for u in self.pending[1:]:
                tot += u
            for u in self.pending:
                u.copy_(tot)
            self.pending = []


@pytest.mark.parametrize("kind,world", [("sym", 2), ("sym", 3), ("big", 2)])
def test_sharded_pair_sum_and_step_on_one_gpu(M, kind, world):
    """every rank's share of the pair kernel's work units, summed = the unsharded acceleration (oracle tolerance), and
    begin / sum / end = mo_step; the ranks' states stay bit-identical"""
    if kind == "sym":
        w, nbig = W.shrink(3, 9000), None
    else:
        w, nbig = W.make_bigsmall(30000, 40), 40
    gm = G * w.mass

    def mk():
        m = _mk(M, w)
        if nbig is not None:
            m.set_nbig(nbig)
        return m
    ref = mk()
    assert ref.pair_kernel_name() == ("pair_sym_kernel" if kind == "sym" else "pair_big_kernel")
    ranks = [mk() for _ in range(world)]
    for r, m in enumerate(ranks):
        m.set_shard(r, world)
    n, lo0, _ = ranks[0].shard_units()
    assert lo0 == 0 and ranks[-1].shard_units()[2] == n and all(ranks[r].shard_units()[2] == ranks[r + 1].shard_units()[1] for r in range(world - 1))
    # shares of a
    ref.accel()
    tot = None
    for m in ranks:
        m.accel()
        tot = m.a.clone() if tot is None else tot + m.a
    a_ref, S = oracle.accel(gm, w.x, w.rcrit, nbig=nbig)
    _check_accel(tot[:, :w.nb].cpu().numpy(), a_ref, S, "sum of the shares")
    assert np.abs(tot[:, :w.nb].cpu().numpy() - ref.get("a")).max() <= 1e-14 * S.max()
    if kind == "big":                                   # row shares: a rank's rows outside its blocks are exactly 0
        assert float(ranks[0].a[:, w.nb - 100:w.nb].abs().max()) == 0.0
    # steps: the ranks one after the other, the sum when all have handed in their share
    L = M.load()
    assert L.mo_step(ranks[0]._ctx, w.dt, 1, None) == M.MO_EINVAL and L.mo_step_begin(ranks[0]._ctx, w.dt) == M.MO_EINVAL   # a not summed yet
    for m in ranks:
        m.a.copy_(tot); m.accel_summed()
    for _ in range(3):
        for m in ranks:
            m.step_begin(w.dt)
        tot = ranks[0].a.clone()
        for m in ranks[1:]:
            tot += m.a
        for m in ranks:
            m.a.copy_(tot); m.accel_summed()
        sts = [m.step_end(w.dt) for m in ranks]
    s_ref = ref.step(w.dt, 3)
    for m, st in zip(ranks, sts):
        assert np.array_equal(m.get("x"), ranks[0].get("x")) and np.array_equal(m.get("v"), ranks[0].get("v"))
        assert st.nce_last == s_ref.nce_last and st.steps_done == 3
        assert np.array_equal(m.pair_list(st.nce_last), ref.pair_list(s_ref.nce_last))
    assert _rel_vec_err(ranks[0].get("x"), ref.get("x")).max() <= 1e-14 and _rel_vec_err(ranks[0].get("v"), ref.get("v")).max() <= 1e-13
    for m in ranks + [ref]:
        m.close()


def test_sharded_step_with_encounter_resolution(M):
    """the resolving step under sharding: the solve runs replicated on every rank before the rank's share of the pair sum
    (no detour beside the pair sum there) - same step as the unsharded one, which takes the detour"""
    w = W.shrink(3, 6000)
    ref = _mk(M, w); ref.set_resolve(1e-12)
    ranks = [_mk(M, w) for _ in range(2)]
    for r, m in enumerate(ranks):
        m.set_shard(r, 2); m.set_resolve(1e-12)
    tot = None
    for m in ranks:
        m.accel()
        tot = m.a.clone() if tot is None else tot + m.a
    for m in ranks:
        m.a.copy_(tot); m.accel_summed()
    for _ in range(2):
        for m in ranks:
            m.step_begin(w.dt)
        tot = ranks[0].a + ranks[1].a
        for m in ranks:
            m.a.copy_(tot); m.accel_summed()
        sts = [m.step_end(w.dt) for m in ranks]
    s_ref = ref.step(w.dt, 2)
    assert sts[0].nce_last == s_ref.nce_last > 0 and sts[0].resolve_fail == 0 and s_ref.resolve_fail == 0
    assert ranks[0].resolve_stats()["bodies"] == ref.resolve_stats()["bodies"] > 0
    assert np.array_equal(ranks[0].get("x"), ranks[1].get("x")) and np.array_equal(ranks[0].get("v"), ranks[1].get("v"))
    assert _rel_vec_err(ranks[0].get("x"), ref.get("x")).max() <= 1e-13 and _rel_vec_err(ranks[0].get("v"), ref.get("v")).max() <= 1e-12
    for m in ranks + [ref]:
        m.close()


def test_sharded_driver_world1_and_unsupported_sizes(M):
    from paper_2601_19654_b200.sharded import ShardedMopal
    w = W.shrink(3, 9000)
    m1, m2 = _mk(M, w), _mk(M, w)
    sm = ShardedMopal(m1)                              # world 1: plain mo_step
    sm.step(w.dt, 2); m2.step(w.dt, 2)
    assert np.array_equal(m1.get("x"), m2.get("x")) and sm.allreduces == 0
    m1.close(); m2.close()
    # the driver over the sequential stand-in: two ranks, two steps (the deferred sum needs both ranks to have called in,
    # so the ranks' calls are interleaved by hand)
    small = _mk(M, W.shrink(1, 2000))
    L = M.load()
    assert L.mo_set_shard(small._ctx, 0, 2) == M.MO_EINVAL          # below 8192 bodies the pair kernel does not split
    assert L.mo_set_shard(small._ctx, 0, 1) == M.MO_OK
    assert L.mo_set_shard(small._ctx, 2, 2) == M.MO_EINVAL and L.mo_set_shard(None, 0, 1) == M.MO_EINVAL
    assert L.mo_step_begin(small._ctx, 1.0) == M.MO_EINVAL and L.mo_step_end(small._ctx, 1.0, None) == M.MO_EINVAL
    small.close()
