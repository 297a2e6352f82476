"""Thin ctypes binding over libmopal.so (include/mopal.h) - argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  torch is used for device
memory and the stream, nothing else.  There is no CPU fallback: if ``libmopal.so`` cannot
be loaded, or there is no CUDA device, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmopal.so")

MO_OK, MO_EINVAL, MO_ENOMEM, MO_ECUDA, MO_EOVERFLOW, MO_ENOCONV, MO_ERESOLVE, MO_ELIMIT = range(8)
_SOFT = (MO_OK, MO_EOVERFLOW, MO_ENOCONV, MO_ERESOLVE)      # statuses reported in Stats.status instead of raised

EXPORTS = ["mo_create", "mo_accel", "mo_drift", "mo_encounters", "mo_step", "mo_destroy",
           "mo_snapshot", "mo_snapshot_ptrs", "mo_snapshot_copy", "mo_invalidate_accel", "mo_get_stats", "mo_launch_count",
           "mo_workspace_bytes", "mo_step_host", "mo_accel_host", "mo_probe_fp64_peak",
           "mo_pair_geometry", "mo_set_kernel_timing", "mo_pair_kernel_ms", "mo_strerror", "mo_version",
           "mo_set_nbig", "mo_pair_kernel_name", "mo_h2dh", "mo_dh2h", "mo_hill", "mo_set_hill", "mo_energy",
           "mo_resolve", "mo_set_resolve", "mo_resolve_stats", "mo_boxes_copy",
           "mo_set_shard", "mo_shard_range", "mo_shard_units", "mo_step_begin", "mo_accel_summed", "mo_step_end",
           "mo_accel_static", "mo_accel_static_max_nb"]


class MoStats(C.Structure):
    _fields_ = [("steps_done", C.c_int64), ("nce_last", C.c_int64), ("nce_total", C.c_int64),
                ("drift_fail", C.c_int32), ("max_newton", C.c_int32), ("resolve_fail", C.c_int32), ("reserved", C.c_int32)]


class MoEnergy(C.Structure):
    _fields_ = [("T", C.c_double), ("Us", C.c_double), ("Up", C.c_double), ("E", C.c_double), ("L", C.c_double * 3)]


class MopalError(RuntimeError):
    def __init__(self, status, what):
        self.status = int(status)
        super().__init__(f"{what}: {strerror(status)} (mo_status {int(status)})")


_lib = None


def load():
    """Load libmopal.so (building it with nvcc first if it is not there).  Raises if it
    cannot be had - there is nothing to fall back to."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        from .build import build_lib
        build_lib()
    L = C.CDLL(LIB_PATH)
    vp, D, I32, I64 = C.c_void_p, C.c_double, C.c_int32, C.c_int64
    L.mo_create.restype = C.c_int
    L.mo_create.argtypes = [C.POINTER(vp), I32, I32, D, D, vp, vp, vp, vp, vp, vp, I64, vp, vp]
    L.mo_accel.restype = C.c_int; L.mo_accel.argtypes = [vp]
    L.mo_drift.restype = C.c_int; L.mo_drift.argtypes = [vp, D]
    L.mo_encounters.restype = C.c_int; L.mo_encounters.argtypes = [vp, D, vp, vp, C.POINTER(I64)]
    L.mo_step.restype = C.c_int; L.mo_step.argtypes = [vp, D, I32, C.POINTER(MoStats)]
    L.mo_destroy.restype = None; L.mo_destroy.argtypes = [vp]
    L.mo_snapshot.restype = C.c_int; L.mo_snapshot.argtypes = [vp]
    L.mo_snapshot_ptrs.restype = C.c_int; L.mo_snapshot_ptrs.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]
    L.mo_snapshot_copy.restype = C.c_int; L.mo_snapshot_copy.argtypes = [vp, vp, vp]
    L.mo_invalidate_accel.restype = C.c_int; L.mo_invalidate_accel.argtypes = [vp]
    L.mo_boxes_copy.restype = C.c_int; L.mo_boxes_copy.argtypes = [vp, vp]
    L.mo_set_nbig.restype = C.c_int; L.mo_set_nbig.argtypes = [vp, I32]
    L.mo_pair_kernel_name.restype = C.c_char_p; L.mo_pair_kernel_name.argtypes = [vp]
    L.mo_h2dh.restype = C.c_int; L.mo_h2dh.argtypes = [vp]
    L.mo_dh2h.restype = C.c_int; L.mo_dh2h.argtypes = [vp]
    L.mo_hill.restype = C.c_int; L.mo_hill.argtypes = [vp, C.c_double, I32, vp]
    L.mo_set_hill.restype = C.c_int; L.mo_set_hill.argtypes = [vp, C.c_double, I32]
    L.mo_energy.restype = C.c_int; L.mo_energy.argtypes = [vp, C.POINTER(MoEnergy)]
    L.mo_resolve.restype = C.c_int; L.mo_resolve.argtypes = [vp, C.c_double, C.c_double]
    L.mo_set_resolve.restype = C.c_int; L.mo_set_resolve.argtypes = [vp, C.c_double]
    L.mo_resolve_stats.restype = C.c_int; L.mo_resolve_stats.argtypes = [vp, C.POINTER(I32)]
    L.mo_set_shard.restype = C.c_int; L.mo_set_shard.argtypes = [vp, I32, I32]
    L.mo_shard_range.restype = C.c_int; L.mo_shard_range.argtypes = [C.c_int64, I32, I32, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.mo_shard_units.restype = C.c_int; L.mo_shard_units.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.mo_step_begin.restype = C.c_int; L.mo_step_begin.argtypes = [vp, C.c_double]
    L.mo_accel_summed.restype = C.c_int; L.mo_accel_summed.argtypes = [vp]
    L.mo_step_end.restype = C.c_int; L.mo_step_end.argtypes = [vp, C.c_double, C.POINTER(MoStats)]
    L.mo_get_stats.restype = C.c_int; L.mo_get_stats.argtypes = [vp, C.POINTER(MoStats)]
    L.mo_launch_count.restype = I64; L.mo_launch_count.argtypes = [vp]
    L.mo_workspace_bytes.restype = I64; L.mo_workspace_bytes.argtypes = [vp]
    L.mo_step_host.restype = C.c_int
    L.mo_step_host.argtypes = [vp, D, I32, vp, vp, vp, I32, vp, I64, C.POINTER(MoStats)]
    L.mo_accel_host.restype = C.c_int; L.mo_accel_host.argtypes = [vp, vp, vp]
    L.mo_accel_static_max_nb.restype = I32; L.mo_accel_static_max_nb.argtypes = []
    L.mo_accel_static.restype = C.c_int
    L.mo_accel_static.argtypes = [I32, I32, vp, vp, vp, vp, vp]
    L.mo_probe_fp64_peak.restype = C.c_int
    L.mo_probe_fp64_peak.argtypes = [vp, I32, C.POINTER(D), C.POINTER(D), C.POINTER(D)]
    L.mo_pair_geometry.restype = C.c_int
    L.mo_pair_geometry.argtypes = [vp, C.POINTER(I32), C.POINTER(I32), C.POINTER(I32), C.POINTER(I32)]
    L.mo_set_kernel_timing.restype = C.c_int; L.mo_set_kernel_timing.argtypes = [vp, I32]
    L.mo_pair_kernel_ms.restype = C.c_int; L.mo_pair_kernel_ms.argtypes = [vp, C.POINTER(D), C.POINTER(I32)]
    L.mo_strerror.restype = C.c_char_p; L.mo_strerror.argtypes = [C.c_int]
    L.mo_version.restype = C.c_char_p; L.mo_version.argtypes = []
    _lib = L
    return L


def strerror(status) -> str:
    return load().mo_strerror(int(status)).decode()


def version() -> str:
    return load().mo_version().decode()


def shard_range(n, rank, world):
    """[lo, hi): rank's contiguous share of n work units (mo_shard_range; host only, no GPU needed)."""
    lo, hi = C.c_int64(0), C.c_int64(0)
    st = load().mo_shard_range(int(n), int(rank), int(world), C.byref(lo), C.byref(hi))
    if st != MO_OK:
        raise MopalError(st, "mo_shard_range")
    return int(lo.value), int(hi.value)


def accel_static_max_nb() -> int:
    return int(load().mo_accel_static_max_nb())


def accel_static(gm, x, rcrit, a=None):
    """a(x) through mo_accel_static - the entry point that allocates nothing (its scratch is a fixed device array inside
    the library; nb <= accel_static_max_nb()).  gm, rcrit: [nb], x: [3, ld] float64 CUDA tensors; returns a [3, ld]
    (the tensor passed as ``a``, else a new one - that allocation is the caller's, not the library's).  Enqueued on
    torch's current stream; calls that overlap on the GPU race on the shared scratch."""
    import torch
    nb, ld = int(gm.numel()), int(x.shape[1])
    for t in (gm, x, rcrit):
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise MopalError(MO_EINVAL, "accel_static: float64 contiguous CUDA tensors")
    if a is None:
        a = torch.zeros_like(x)
    st = load().mo_accel_static(nb, ld, gm.data_ptr(), x.data_ptr(), rcrit.data_ptr(), a.data_ptr(),
                                C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if st == MO_ELIMIT:
        raise MopalError(st, f"mo_accel_static: nb = {nb} > {accel_static_max_nb()}")
    if st != MO_OK:
        raise MopalError(st, "mo_accel_static")
    return a


def probe_fp64_peak(reps: int = 5, with_mean: bool = False):
    """(best TFLOP/s, its ms[, TFLOP/s over the whole train]) of the library's register-resident
    DFMA probe on the current device."""
    import torch
    if not torch.cuda.is_available():
        raise MopalError(MO_ECUDA, "mo_probe_fp64_peak")
    tf, ms, mean = C.c_double(0), C.c_double(0), C.c_double(0)
    st = load().mo_probe_fp64_peak(C.c_void_p(torch.cuda.current_stream().cuda_stream), reps, C.byref(tf), C.byref(ms),
                                   C.byref(mean))
    if st != MO_OK:
        raise MopalError(st, "mo_probe_fp64_peak")
    return (tf.value, ms.value, mean.value) if with_mean else (tf.value, ms.value)


@dataclass
class Stats:
    steps_done: int
    nce_last: int
    nce_total: int
    drift_fail: int
    max_newton: int
    resolve_fail: int = 0
    status: int = MO_OK


def _stats(s: MoStats, status=MO_OK) -> Stats:
    return Stats(int(s.steps_done), int(s.nce_last), int(s.nce_total), int(s.drift_fail), int(s.max_newton),
                 int(s.resolve_fail), int(status))


class Mopal:
    """One libmopal context plus the torch-owned device arrays it borrows.

    mass[nb], x[3,nb], v[3,nb], rcrit[nb]: numpy float64 (host) - copied to the device once.
    State tensors are ``self.x, self.v, self.a`` (``[3, ld]`` float64 cuda), ``self.rcrit``,
    ``self.pairs`` (``[cap, 2]`` int32), ``self.flag`` (``[nb]`` uint8).
    """

    def __init__(self, mass, x, v, rcrit, m_star=1.0, G=2.9591220828559115e-4, cap=1 << 20, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise MopalError(MO_ECUDA, "Mopal(): no CUDA device (libmopal has no CPU path)")
        self._L = load()
        self._torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        nb = int(np.asarray(mass).shape[0])
        self.nb = nb
        self.nbig = nb
        self.ld = (nb + 3) // 4 * 4
        self.cap = int(cap)
        self.m_star, self.G = float(m_star), float(G)
        f64 = torch.float64

        def plane(a):
            t = torch.zeros((3, self.ld), dtype=f64, device=self.device)
            t[:, :nb] = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(self.device)
            return t

        self.x, self.v = plane(x), plane(v)
        self.a = torch.zeros((3, self.ld), dtype=f64, device=self.device)
        self.mass = torch.from_numpy(np.ascontiguousarray(mass, dtype=np.float64)).to(self.device)
        self.rcrit = torch.from_numpy(np.ascontiguousarray(rcrit, dtype=np.float64)).to(self.device)
        self.pairs = torch.zeros((max(self.cap, 1), 2), dtype=torch.int32, device=self.device)
        self.flag = torch.zeros(nb, dtype=torch.uint8, device=self.device)
        self.stream = torch.cuda.current_stream(self.device)
        self._ctx = C.c_void_p(None)
        st = self._L.mo_create(C.byref(self._ctx), nb, self.ld, self.m_star, self.G, self.mass.data_ptr(),
                               self.x.data_ptr(), self.v.data_ptr(), self.a.data_ptr(), self.rcrit.data_ptr(),
                               self.pairs.data_ptr() if self.cap > 0 else None, self.cap, self.flag.data_ptr(),
                               C.c_void_p(self.stream.cuda_stream))
        if st != MO_OK:
            self._ctx = C.c_void_p(None)
            raise MopalError(st, "mo_create")

    # -- the six calls ---------------------------------------------------------------
    def accel(self):
        self._check(self._L.mo_accel(self._ctx), "mo_accel")

    def drift(self, dt):
        self._check(self._L.mo_drift(self._ctx, float(dt)), "mo_drift")

    def encounters(self, dt, x0=None, v0=None, raise_on_overflow=False):
        """Returns the true pair count (synchronises).  x0, v0: cuda [3, ld] tensors or None
        to use the context snapshot."""
        cnt = C.c_int64(0)
        p0 = x0.data_ptr() if x0 is not None else None
        q0 = v0.data_ptr() if v0 is not None else None
        st = self._L.mo_encounters(self._ctx, float(dt), p0, q0, C.byref(cnt))
        if st != MO_OK and not (st == MO_EOVERFLOW and not raise_on_overflow):
            raise MopalError(st, "mo_encounters")
        return int(cnt.value)

    def step(self, dt, nsteps=1, sync=True) -> Stats | None:
        if not sync:
            self._check(self._L.mo_step(self._ctx, float(dt), int(nsteps), None), "mo_step")
            return None
        s = MoStats()
        st = self._L.mo_step(self._ctx, float(dt), int(nsteps), C.byref(s))
        if st not in _SOFT:
            raise MopalError(st, "mo_step")
        return _stats(s, st)

    def close(self):
        ctx = getattr(self, "_ctx", None)
        if ctx is not None and ctx.value:
            self._L.mo_destroy(ctx)
            ctx.value = None          # (no module globals here: close() also runs from __del__ at interpreter exit)

    __del__ = close

    # -- extras ------------------------------------------------------------------------
    def snapshot(self):
        self._check(self._L.mo_snapshot(self._ctx), "mo_snapshot")

    def snapshot_tensors(self):
        """Copies of the context's x0, v0 snapshot as [3, ld] cuda tensors."""
        torch = self._torch
        x0 = torch.empty_like(self.x); v0 = torch.empty_like(self.v)
        self._check(self._L.mo_snapshot_copy(self._ctx, x0.data_ptr(), v0.data_ptr()), "mo_snapshot_copy")
        self.stream.synchronize()
        return x0, v0

    def boxes(self):
        """(lo[2, nb], hi[2, nb]) numpy: the x and y boxes of the last encounter pass (mce_snif LOOP 1-2)."""
        t = self._torch.empty((self.nb, 4), dtype=self._torch.float64, device=self.device)
        self._check(self._L.mo_boxes_copy(self._ctx, t.data_ptr()), "mo_boxes_copy")
        self.stream.synchronize()
        b = t.cpu().numpy()
        return np.stack([b[:, 0], b[:, 2]]), np.stack([b[:, 1], b[:, 3]])

    def set_nbig(self, nbig):
        """Bodies 0..nbig-1 are the big bodies: the only gravity sources and first members of
        encounter pairs; nbig = nb is fully interacting."""
        self._check(self._L.mo_set_nbig(self._ctx, int(nbig)), "mo_set_nbig")
        self.nbig = int(nbig)

    # ---- per-step support routines ----
    def h2dh(self):
        """heliocentric -> barycentric velocities, in place (mco_h2dh)."""
        self._check(self._L.mo_h2dh(self._ctx), "mo_h2dh")

    def dh2h(self):
        """barycentric -> heliocentric velocities, in place (mce_dh2h)."""
        self._check(self._L.mo_dh2h(self._ctx), "mo_dh2h")

    def hill(self, n_hill=3.0, mode=0, rhill=None):
        """rcrit <- n_hill * Hill radius from the current state (mce_hill); ``rhill``: optional
        float64 cuda tensor of nb elements that receives the Hill radii."""
        ptr = None if rhill is None else rhill.data_ptr()
        self._check(self._L.mo_hill(self._ctx, float(n_hill), int(mode), ptr), "mo_hill")

    def set_hill(self, n_hill=3.0, mode=0):
        """mo_step recomputes rcrit at the start of every step (mode -1: off)."""
        self._check(self._L.mo_set_hill(self._ctx, float(n_hill), int(mode)), "mo_set_hill")

    def energy(self):
        """dict(T, Us, Up, E, L[3]) of star + bodies in the barycentric frame (mxx_en)."""
        e = MoEnergy()
        self._check(self._L.mo_energy(self._ctx, C.byref(e)), "mo_energy")
        return dict(T=e.T, Us=e.Us, Up=e.Up, E=e.E, L=np.array(list(e.L)))

    # ---- close-encounter resolution (the paper's mdt_hkce) ----
    def resolve(self, dt, tol=1e-12):
        """Bulirsch-Stoer integration of the bodies of the current pair list from the snapshot over dt."""
        self._check(self._L.mo_resolve(self._ctx, float(dt), float(tol)), "mo_resolve")

    def set_resolve(self, tol=1e-12):
        """mo_step resolves the encounters of every step (tol <= 0: off)."""
        self._check(self._L.mo_set_resolve(self._ctx, float(tol)), "mo_set_resolve")

    def resolve_stats(self):
        out = (C.c_int32 * 4)()
        self._check(self._L.mo_resolve_stats(self._ctx, out), "mo_resolve_stats")
        return dict(bodies=out[0], steps=out[1], rhs=out[2], fail=out[3])

    # ---- pair sum sharded over several GPUs (include/mopal.h: mo_set_shard) ----
    def set_shard(self, rank, world):
        self._check(self._L.mo_set_shard(self._ctx, int(rank), int(world)), "mo_set_shard")

    def shard_units(self):
        """(work units of the pair kernel, lo, hi): this context evaluates the units [lo, hi)."""
        n, lo, hi = C.c_int64(0), C.c_int64(0), C.c_int64(0)
        self._check(self._L.mo_shard_units(self._ctx, C.byref(n), C.byref(lo), C.byref(hi)), "mo_shard_units")
        return int(n.value), int(lo.value), int(hi.value)

    def step_begin(self, dt):
        self._check(self._L.mo_step_begin(self._ctx, float(dt)), "mo_step_begin")

    def accel_summed(self):
        self._check(self._L.mo_accel_summed(self._ctx), "mo_accel_summed")

    def step_end(self, dt, sync=True) -> Stats | None:
        if not sync:
            self._check(self._L.mo_step_end(self._ctx, float(dt), None), "mo_step_end")
            return None
        s = MoStats()
        st = self._L.mo_step_end(self._ctx, float(dt), C.byref(s))
        if st not in _SOFT:
            raise MopalError(st, "mo_step_end")
        return _stats(s, st)

    def invalidate_accel(self):
        self._check(self._L.mo_invalidate_accel(self._ctx), "mo_invalidate_accel")

    def stats(self) -> Stats:
        s = MoStats()
        st = self._L.mo_get_stats(self._ctx, C.byref(s))
        if st not in _SOFT:
            raise MopalError(st, "mo_get_stats")
        return _stats(s, st)

    def launch_count(self) -> int:
        return int(self._L.mo_launch_count(self._ctx))

    def workspace_bytes(self) -> int:
        return int(self._L.mo_workspace_bytes(self._ctx))

    def pair_geometry(self):
        a, b, c, d = C.c_int32(), C.c_int32(), C.c_int32(), C.c_int32()
        self._check(self._L.mo_pair_geometry(self._ctx, C.byref(a), C.byref(b), C.byref(c), C.byref(d)), "mo_pair_geometry")
        return dict(ipt=a.value, jsplit=b.value, ctas=c.value, ctas_per_sm=d.value)

    def pair_kernel_name(self) -> str:
        return self._L.mo_pair_kernel_name(self._ctx).decode()

    def set_kernel_timing(self, on: bool):
        self._check(self._L.mo_set_kernel_timing(self._ctx, 1 if on else 0), "mo_set_kernel_timing")

    def pair_kernel_ms(self):
        ms, n = C.c_double(0), C.c_int32(0)
        self._check(self._L.mo_pair_kernel_ms(self._ctx, C.byref(ms), C.byref(n)), "mo_pair_kernel_ms")
        return ms.value, n.value

    def step_host(self, dt, nsteps, x_host, v_host, rcrit_host=None, a_is_current=False, pairs_host=None) -> Stats:
        """x_host, v_host: pinned (or plain) CPU float64 tensors / arrays of shape [3, ld];
        updated in place.  Host<->device copies happen inside the call."""
        s = MoStats()
        cap_h = 0 if pairs_host is None else int(pairs_host.shape[0])
        st = self._L.mo_step_host(self._ctx, float(dt), int(nsteps), _hptr(x_host), _hptr(v_host),
                                  _hptr(rcrit_host), 1 if a_is_current else 0, _hptr(pairs_host), cap_h, C.byref(s))
        if st not in _SOFT:
            raise MopalError(st, "mo_step_host")
        return _stats(s, st)

    def accel_host(self, x_host, a_host):
        self._check(self._L.mo_accel_host(self._ctx, _hptr(x_host), _hptr(a_host)), "mo_accel_host")

    # -- helpers -----------------------------------------------------------------------
    def _check(self, st, what):
        if st != MO_OK:
            raise MopalError(st, what)

    def get(self, name):
        """numpy copy of a state array restricted to the nb bodies."""
        self.stream.synchronize()
        t = getattr(self, name)
        if t.dim() == 2 and t.shape[1] == self.ld:
            return t[:, :self.nb].cpu().numpy()
        return t.cpu().numpy()

    def set(self, name, arr):
        """Overwrite a state array from numpy; changing x or rcrit invalidates the cached accelerations."""
        if name in ("x", "rcrit"):
            self.invalidate_accel()
        t = getattr(self, name)
        src = self._torch.from_numpy(np.ascontiguousarray(arr)).to(self.device)
        if t.dim() == 2 and t.shape[1] == self.ld:
            t[:, :self.nb] = src
        else:
            t.copy_(src)

    def pair_list(self, count=None):
        if count is None:
            count = self.stats().nce_last
        n = min(int(count), self.cap)
        self.stream.synchronize()
        return self.pairs[:n].cpu().numpy()


def _hptr(a):
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()
