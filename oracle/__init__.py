"""CPU oracle for libmopal - TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes wrapper over ``mopal_oracle.c`` (long double parity build, plus the
plain-double timed build).  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s cpu_baseline / ``--impl reference`` legs may import this package;
nothing under ``paper_2601_19654_b200/`` does, and this package imports nothing
from there.

Arrays are numpy float64, SoA ``[3, ld]`` C-contiguous (component c of body b at
``[c, b]``), bodies 0..nb-1 (the paper's element 1, the star, is not a body:
PAPER.md:134).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mopal_oracle.c")
_LIBS = {"ld": os.path.join(_HERE, "libmopal_oracle.so"),
         "f64": os.path.join(_HERE, "libmopal_oracle_f64.so")}
_loaded = {}


def build(force: bool = False) -> None:
    """Compile both oracle builds with gcc (no CUDA involved)."""
    stale = force or any((not os.path.exists(p)) or os.path.getmtime(p) < os.path.getmtime(_SRC)
                         for p in _LIBS.values())
    if stale:
        subprocess.check_call(["sh", os.path.join(_HERE, "build_oracle.sh")])


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _lib(kind="ld"):
    if kind in _loaded:
        return _loaded[kind]
    build()
    L = C.CDLL(_LIBS[kind])
    D, I, I64 = C.POINTER(C.c_double), C.c_int, C.c_int64
    P32, PU8, PI64 = C.POINTER(C.c_int32), C.POINTER(C.c_uint8), C.POINTER(C.c_int64)
    L.oracle_real_bytes.restype = I
    L.oracle_set_num_threads.restype = I
    L.oracle_set_num_threads.argtypes = [I]
    L.oracle_changeover.restype = C.c_double
    L.oracle_changeover.argtypes = [C.c_double, C.c_double]
    L.oracle_accel_big.restype = I
    L.oracle_accel_big.argtypes = [I, I, I, D, D, D, D, D]
    L.oracle_accel_rows_big.restype = I
    L.oracle_accel_rows_big.argtypes = [I, I, I, D, D, D, P32, I, D, D]
    L.oracle_encounters_big.restype = I64
    L.oracle_encounters_big.argtypes = [I, I, I, C.c_double, D, D, D, D, D, P32, I64, PU8, P32, I64, PI64, I, I]
    L.oracle_boxes_big.restype = I
    L.oracle_boxes_big.argtypes = [I, I, I, C.c_double, D, D, D, D, D, D, D]
    L.oracle_pair_d2min.restype = C.c_double
    L.oracle_pair_d2min.argtypes = [I, C.c_double, D, D, D, D, I, I]
    L.oracle_encounters.restype = I64
    L.oracle_encounters.argtypes = [I, I, C.c_double, D, D, D, D, D, P32, I64, PU8, P32, I64, PI64]
    L.oracle_drift.restype = I
    L.oracle_drift.argtypes = [I, I, C.c_double, C.c_double, D, D, P32]
    L.oracle_kick.restype = I
    L.oracle_kick.argtypes = [I, I, C.c_double, D, D]
    L.oracle_jump.restype = I
    L.oracle_jump.argtypes = [I, I, C.c_double, C.c_double, D, D, D, D]
    L.oracle_step_big.restype = I64
    L.oracle_step_big.argtypes = [I, I, I, C.c_double, D, D, C.c_double, D, D, D, D, D,
                                  P32, I64, PU8, P32, I64, PI64, P32]
    L.oracle_step_noenc.restype = I
    L.oracle_step_noenc.argtypes = [I, I, C.c_double, D, D, C.c_double, D, D, D]
    L.oracle_h2dh.restype = I
    L.oracle_h2dh.argtypes = [I, I, C.c_double, D, D]
    L.oracle_dh2h.restype = I
    L.oracle_dh2h.argtypes = [I, I, C.c_double, D, D]
    L.oracle_hill.restype = I
    L.oracle_hill.argtypes = [I, I, I, C.c_double, C.c_double, C.c_double, D, D, D, D, D]
    L.oracle_energy.restype = I
    L.oracle_energy.argtypes = [I, I, I, C.c_double, C.c_double, D, D, D, D]
    L.oracle_resolve.restype = I
    L.oracle_resolve.argtypes = [I, I, C.c_double, D, D, C.c_double, D, D, D, D, P32, I64, C.c_double, P32]
    _loaded[kind] = L
    return L


def _soa(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    assert a.ndim == 2 and a.shape[0] == 3, a.shape
    return a


def _vec(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def real_bytes(kind="ld") -> int:
    return _lib(kind).oracle_real_bytes()


def set_threads(n: int, kind="ld") -> int:
    """OpenMP threads of the outer body loops of build `kind` (timing only; no result depends on it).
    Returns the thread count in force."""
    os.environ["OMP_NUM_THREADS"] = str(int(n))
    return int(_lib(kind).oracle_set_num_threads(int(n)))


def changeover(r: float, rc: float, kind="ld") -> float:
    """K(r; rc): quintic smoothstep between 0.1 rc and rc (reading A-1)."""
    return float(_lib(kind).oracle_changeover(float(r), float(rc)))


def _nbig(nbig, nb):
    """nbig = number of big bodies = gravity sources / first members of encounter pairs
    (PAPER.md:152-157, 249-260); None = every body (the fully interacting case)."""
    n = nb if nbig is None else int(nbig)
    assert 0 <= n <= nb
    return n


def accel(gm, x, rcrit, kind="ld", nbig=None):
    """O-A.  Returns (a[3,nb], S[3,nb]) with S = sum_j |term| for the tolerance."""
    x = _soa(x); gm = _vec(gm); rcrit = _vec(rcrit)
    nb = x.shape[1]
    a = np.zeros_like(x); S = np.zeros_like(x)
    rc = _lib(kind).oracle_accel_big(nb, _nbig(nbig, nb), nb, _dp(gm), _dp(x), _dp(rcrit), _dp(a), _dp(S))
    assert rc == 0
    return a, S


def accel_rows(gm, x, rcrit, rows, kind="ld", nbig=None):
    """O-A for the chosen bodies only.  Returns (a[3,len(rows)], S[3,len(rows)])."""
    x = _soa(x); gm = _vec(gm); rcrit = _vec(rcrit)
    rows = np.ascontiguousarray(rows, dtype=np.int32)
    nb = x.shape[1]
    a = np.zeros((3, len(rows))); S = np.zeros((3, len(rows)))
    rc = _lib(kind).oracle_accel_rows_big(nb, _nbig(nbig, nb), nb, _dp(gm), _dp(x), _dp(rcrit),
                                      rows.ctypes.data_as(C.POINTER(C.c_int32)), len(rows), _dp(a), _dp(S))
    assert rc == 0
    return a, S


def boxes(h, x0, v0, x1, v1, rcrit, kind="ld", nbig=None):
    """O-B.1.  Returns (lo[2,nb], hi[2,nb]) for x and y."""
    x0, v0, x1, v1 = map(_soa, (x0, v0, x1, v1)); rcrit = _vec(rcrit)
    nb = x0.shape[1]
    lo = np.zeros((2, nb)); hi = np.zeros((2, nb))
    rc = _lib(kind).oracle_boxes_big(nb, _nbig(nbig, nb), nb, float(h), _dp(x0), _dp(v0), _dp(x1), _dp(v1),
                                 _dp(rcrit), _dp(lo), _dp(hi))
    assert rc == 0
    return lo, hi


def pair_d2min(h, x0, v0, x1, v1, i, j, kind="ld") -> float:
    x0, v0, x1, v1 = map(_soa, (x0, v0, x1, v1))
    nb = x0.shape[1]
    return float(_lib(kind).oracle_pair_d2min(nb, float(h), _dp(x0), _dp(v0), _dp(x1), _dp(v1),
                                              int(i), int(j)))


def encounters(h, x0, v0, x1, v1, rcrit, cap=None, kind="ld", row_stride=1, row_phase=0, nbig=None):
    """O-B.  Returns dict(pairs[n,2] sorted, count (true total), flag[nb] uint8,
    ambig[m,2], n_ambig).  row_stride > 1 restricts to rows i % row_stride == row_phase."""
    x0, v0, x1, v1 = map(_soa, (x0, v0, x1, v1)); rcrit = _vec(rcrit)
    nb = x0.shape[1]
    L = _lib(kind)
    if cap is None:
        cap = 1 << 16
    while True:
        pairs = np.zeros((max(cap, 1), 2), dtype=np.int32)
        amb = np.zeros((max(cap, 1), 2), dtype=np.int32)
        flag = np.zeros(max(nb, 1), dtype=np.uint8)
        n_amb = C.c_int64(0)
        cnt = L.oracle_encounters_big(nb, _nbig(nbig, nb), nb, float(h), _dp(x0), _dp(v0), _dp(x1), _dp(v1), _dp(rcrit),
                                       pairs.ctypes.data_as(C.POINTER(C.c_int32)), cap,
                                       flag.ctypes.data_as(C.POINTER(C.c_uint8)),
                                       amb.ctypes.data_as(C.POINTER(C.c_int32)), cap, C.byref(n_amb),
                                       int(row_stride), int(row_phase))
        assert cnt >= 0
        if cnt <= cap and n_amb.value <= cap:
            break
        cap = int(max(cnt, n_amb.value))
    return dict(pairs=pairs[:cnt].copy(), count=int(cnt), flag=flag[:nb].copy(),
                ambig=amb[:n_amb.value].copy(), n_ambig=int(n_amb.value))


def drift(mu, dt, x, v, kind="ld"):
    """O-C.  Returns (x1, v1, iflag[nb])."""
    x = _soa(x).copy(); v = _soa(v).copy()
    nb = x.shape[1]
    iflag = np.zeros(max(nb, 1), dtype=np.int32)
    nf = _lib(kind).oracle_drift(nb, nb, float(mu), float(dt), _dp(x), _dp(v),
                                 iflag.ctypes.data_as(C.POINTER(C.c_int32)))
    assert nf >= 0
    return x, v, iflag[:nb]


def kick(hk, v, a, kind="ld"):
    v = _soa(v).copy(); a = _soa(a)
    _lib(kind).oracle_kick(v.shape[1], v.shape[1], float(hk), _dp(v), _dp(a))
    return v


def jump(hj, mu, gm, x, v, kind="ld"):
    """Returns (x_new, P[3]) with P = sum gm_j v_j."""
    x = _soa(x).copy(); v = _soa(v); gm = _vec(gm)
    P = np.zeros(3)
    _lib(kind).oracle_jump(x.shape[1], x.shape[1], float(hj), float(mu), _dp(gm), _dp(x), _dp(v), _dp(P))
    return x, P


def step(mu, gm, rcrit, h, x, v, a, cap=1 << 16, with_encounters=True, kind="ld", nbig=None):
    """O-D, one hybrid step.  Returns dict(x, v, a, x0, v0, pairs, count, flag, ambig, n_ambig, nfail)."""
    x = _soa(x).copy(); v = _soa(v).copy(); a = _soa(a).copy()
    gm = _vec(gm); rcrit = _vec(rcrit)
    nb = x.shape[1]
    L = _lib(kind)
    if not with_encounters:
        assert nbig is None or int(nbig) == nb
        rc = L.oracle_step_noenc(nb, nb, float(mu), _dp(gm), _dp(rcrit), float(h), _dp(x), _dp(v), _dp(a))
        assert rc == 0
        return dict(x=x, v=v, a=a)
    x0 = np.zeros_like(x); v0 = np.zeros_like(v)
    pairs = np.zeros((cap, 2), dtype=np.int32); amb = np.zeros((cap, 2), dtype=np.int32)
    flag = np.zeros(max(nb, 1), dtype=np.uint8)
    n_amb = C.c_int64(0); nfail = C.c_int32(0)
    P32 = C.POINTER(C.c_int32)
    cnt = L.oracle_step_big(nb, _nbig(nbig, nb), nb, float(mu), _dp(gm), _dp(rcrit), float(h), _dp(x), _dp(v), _dp(a),
                        _dp(x0), _dp(v0), pairs.ctypes.data_as(P32), cap,
                        flag.ctypes.data_as(C.POINTER(C.c_uint8)), amb.ctypes.data_as(P32), cap,
                        C.byref(n_amb), C.byref(nfail))
    assert cnt >= 0
    return dict(x=x, v=v, a=a, x0=x0, v0=v0, pairs=pairs[:min(cnt, cap)].copy(), count=int(cnt),
                flag=flag[:nb].copy(), ambig=amb[:min(n_amb.value, cap)].copy(),
                n_ambig=int(n_amb.value), nfail=int(nfail.value))


# ---- per-step support routines (readings H-1..H-4, E-1..E-3) -------------------
def h2dh(m_star, mass, v, kind="ld"):
    """H-1: heliocentric velocities -> barycentric (democratic heliocentric); positions unchanged."""
    v = _soa(v).copy(); mass = _vec(mass)
    assert _lib(kind).oracle_h2dh(v.shape[1], v.shape[1], float(m_star), _dp(mass), _dp(v)) == 0
    return v


def dh2h(m_star, mass, v, kind="ld"):
    """H-2: barycentric (democratic heliocentric) velocities -> heliocentric."""
    v = _soa(v).copy(); mass = _vec(mass)
    assert _lib(kind).oracle_dh2h(v.shape[1], v.shape[1], float(m_star), _dp(mass), _dp(v)) == 0
    return v


def hill(G, m_star, mass, x, v, n_hill=3.0, mode=0, kind="ld"):
    """H-3/H-4: (r_hill, rcrit = n_hill r_hill); mode 0: from |x| ; mode 1: from the osculating a."""
    x = _soa(x); v = _soa(v); mass = _vec(mass)
    nb = x.shape[1]
    rh = np.zeros(nb); rc = np.zeros(nb)
    assert _lib(kind).oracle_hill(nb, nb, int(mode), float(n_hill), float(G), float(m_star), _dp(mass), _dp(x), _dp(v),
                                  _dp(rh), _dp(rc)) == 0
    return rh, rc


def energy(G, m_star, mass, x, v, nbig=None, kind="ld"):
    """E-1..E-3: dict(T, Us, Up, E, L[3], Eabs, Labs[3]) of star + bodies, barycentric frame."""
    x = _soa(x); v = _soa(v); mass = _vec(mass)
    nb = x.shape[1]
    out = np.zeros(11)
    assert _lib(kind).oracle_energy(nb, _nbig(nbig, nb), nb, float(G), float(m_star), _dp(mass), _dp(x), _dp(v), _dp(out)) == 0
    return dict(T=out[0], Us=out[1], Up=out[2], E=out[3], L=out[4:7].copy(), Eabs=out[7], Labs=out[8:11].copy())


def resolve(mu, gm, rcrit, h, x0, v0, x, v, pairs, tol=1e-12, kind="ld"):
    """X-1..X-5: Bulirsch-Stoer integration of the bodies in ``pairs`` from the snapshot (x0, v0) over h under the
    star's Kepler term and the (1 - K)-weighted listed pair forces; other bodies keep (x, v).
    Returns dict(x, v, n, nsteps, nrhs, fail)."""
    x0 = _soa(x0); v0 = _soa(v0); x = _soa(x).copy(); v = _soa(v).copy()
    gm = _vec(gm); rcrit = _vec(rcrit)
    pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
    nb = x.shape[1]
    st = np.zeros(4, dtype=np.int32)
    rc = _lib(kind).oracle_resolve(nb, nb, float(mu), _dp(gm), _dp(rcrit), float(h), _dp(x0), _dp(v0), _dp(x), _dp(v),
                                   pairs.ctypes.data_as(C.POINTER(C.c_int32)), len(pairs), float(tol),
                                   st.ctypes.data_as(C.POINTER(C.c_int32)))
    assert rc in (0, 1), rc
    return dict(x=x, v=v, n=int(st[0]), nsteps=int(st[1]), nrhs=int(st[2]), fail=int(st[3]))
