"""mo_accel_static - the entry point that allocates nothing (include/mopal.h, "No-allocation entry point") - against
the existing path (a context's mo_accel) and the oracle, on calls in a row that share its fixed scratch array.
Collected last on purpose (the file name): the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2601_19654_b200 import workloads as W

G = W.G_AU_DAY_MSUN


def _existing_and_static(M, torch, w, a_out=None):
    """(a of the context path, a of mo_accel_static, oracle a, oracle S) for workload w, all [3, nb] numpy."""
    m = M.Mopal(w.mass, w.x, w.v, w.rcrit, m_star=w.m_star, G=w.G, cap=1 << 16)
    m.accel()
    a_ctx = m.get("a")
    nb = a_ctx.shape[1]
    gm = m.mass * w.G
    a_st = M.accel_static(gm, m.x, m.rcrit, a_out)
    torch.cuda.synchronize()
    a_st = a_st[:, :nb].cpu().numpy()
    m.close()
    a_ref, S = oracle.accel(G * w.mass, w.x, w.rcrit)
    return a_ctx, a_st, a_ref, S


def _check(a, b, S, what):
    err = np.abs(a - b)
    assert (err <= 1e-12 * S + 1e-300).all(), f"{what}: worst {np.max(err / (S + 1e-300)):.3e} x S"      # the accel tolerance of test_gpu_parity.py


def test_static_scratch_entry_point_matches_the_context_path_on_calls_in_a_row():
    import torch
    from paper_2601_19654_b200 import mopal as M
    assert M.accel_static_max_nb() == 4096
    big = W.make_config(1)                    # nb = 4095: 32 tiles, 16 row blocks, 272 units - the scratch's full size; two giants
    small = W.make_config(0)                  # nb = 255: two tiles, one row block - leaves most of the last call's contents in place
    mid = W.shrink(1, 1500)                   # a ragged size in between (a partial last tile and a partial last row block)
    first = None
    for k, w in enumerate((big, small, mid, big)):
        a_ctx, a_st, a_ref, S = _existing_and_static(M, torch, w)
        _check(a_st, a_ctx, S, f"call {k} ({w.name}) vs mo_accel")
        _check(a_st, a_ref, S, f"call {k} ({w.name}) vs oracle")
        assert np.isfinite(a_st).all() and np.abs(a_st).max() > 0
        if k == 0:
            first = a_st
    assert np.array_equal(first, a_st)        # the same system again, after two other sizes used the scratch: bit for bit


def test_static_scratch_entry_point_allocates_nothing_and_rejects_sizes_beyond_its_maximum():
    import torch
    from paper_2601_19654_b200 import mopal as M
    w = W.make_config(1)
    nb = len(w.mass)
    ld = (nb + 3) // 4 * 4
    dev = torch.device("cuda:0")
    x = torch.zeros((3, ld), dtype=torch.float64, device=dev)
    x[:, :nb] = torch.from_numpy(np.ascontiguousarray(w.x)).to(dev)
    gm = torch.from_numpy(G * w.mass).to(dev)
    rc = torch.from_numpy(np.ascontiguousarray(w.rcrit)).to(dev)
    a = torch.full((3, ld), 7.0, dtype=torch.float64, device=dev)
    M.accel_static(gm, x, rc, a)              # (the first launch of a kernel may load its module: not counted below)
    torch.cuda.synchronize()
    a1 = a.clone()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(2):
        a.fill_(7.0)
        M.accel_static(gm, x, rc, a)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0          # no device memory was taken or given back
    assert torch.equal(a, a1)
    if ld > nb:
        assert (a[:, nb:] == 7.0).all()                   # nothing outside the rows < nb is written
    # beyond the maximum: a clear error, nothing launched, the output untouched
    L = M.load()
    n2 = M.accel_static_max_nb() + 1
    ld2 = (n2 + 3) // 4 * 4
    big = torch.zeros((3, ld2), dtype=torch.float64, device=dev)
    one = torch.ones(n2, dtype=torch.float64, device=dev)
    out = torch.full((3, ld2), 7.0, dtype=torch.float64, device=dev)
    st = L.mo_accel_static(n2, ld2, one.data_ptr(), big.data_ptr(), one.data_ptr(), out.data_ptr(), None)
    assert st == M.MO_ELIMIT and "maximum" in L.mo_strerror(st).decode()
    with pytest.raises(M.MopalError, match="4097 > 4096"):
        M.accel_static(one, big, one, out)
    torch.cuda.synchronize()
    assert (out == 7.0).all()
    assert L.mo_accel_static(0, 4, one.data_ptr(), big.data_ptr(), one.data_ptr(), out.data_ptr(), None) == M.MO_EINVAL
    assert L.mo_accel_static(8, 6, one.data_ptr(), big.data_ptr(), one.data_ptr(), out.data_ptr(), None) == M.MO_EINVAL
    assert L.mo_accel_static(8, 8, None, big.data_ptr(), one.data_ptr(), out.data_ptr(), None) == M.MO_EINVAL
