"""CPU-side checks of the boundary: libmopal.so loads, exports every
symbol include/mopal.h declares, validates arguments before touching the device, has no CPU
fallback, and the product package never reaches into oracle/.  No compute calls here."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mopal.h")
PKG = os.path.join(ROOT, "paper_2601_19654_b200")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)          # strip comments
    return sorted(set(re.findall(r"\b(mo_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2601_19654_b200 import mopal
    return mopal.load()


def test_header_declares_the_six_north_star_calls():
    names = _declared()
    for n in ("mo_create", "mo_accel", "mo_encounters", "mo_drift", "mo_step", "mo_destroy"):
        assert n in names


def test_library_exports_every_declared_symbol(lib):
    from paper_2601_19654_b200 import mopal
    names = _declared()
    assert len(names) >= 6
    for n in names:
        assert getattr(lib, n) is not None, n
    # the binding marshals exactly the header's functions
    assert sorted(mopal.EXPORTS) == names
    # and the .so exports nothing of ours beyond them (C ABI only: no mangled API)
    out = subprocess.run(["nm", "-D", "--defined-only", mopal.LIB_PATH], capture_output=True, text=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if " T " in ln}
    assert set(names) <= exported
    assert not [s for s in exported if s.startswith("mo_") and s not in names]


def test_strerror_and_version_need_no_device(lib):
    assert lib.mo_version().decode().startswith("libmopal")
    texts = [lib.mo_strerror(k).decode() for k in range(6)]
    assert len(set(texts)) == 6 and texts[0] == "ok"
    assert lib.mo_launch_count(None) == 0 and lib.mo_workspace_bytes(None) == 0
    lib.mo_destroy(None)   # no-op


def test_argument_validation_precedes_any_device_work(lib):
    from paper_2601_19654_b200 import mopal as M
    ctx = C.c_void_p(None)
    fake = 0x10000   # 16-byte aligned, never dereferenced: every case below fails validation first

    def create(nb=4, ld=4, m_star=1.0, G=3e-4, mass=fake, x=fake, v=fake, a=fake, rc=fake, pairs=fake, cap=8, flag=fake):
        return lib.mo_create(C.byref(ctx), nb, ld, m_star, G, mass, x, v, a, rc, pairs, cap, flag, None)

    assert create(nb=0) == M.MO_EINVAL
    assert create(nb=5, ld=4) == M.MO_EINVAL            # ld < nb
    assert create(nb=3, ld=6) == M.MO_EINVAL            # ld % 4
    assert create(m_star=0.0) == M.MO_EINVAL
    assert create(G=float("nan")) == M.MO_EINVAL
    assert create(m_star=float("inf")) == M.MO_EINVAL
    assert create(x=None) == M.MO_EINVAL
    assert create(x=fake + 8) == M.MO_EINVAL            # misaligned
    assert create(cap=-1) == M.MO_EINVAL
    assert create(pairs=None, cap=4) == M.MO_EINVAL
    assert ctx.value is None
    assert lib.mo_create(None, 4, 4, 1.0, 3e-4, fake, fake, fake, fake, fake, fake, 8, fake, None) == M.MO_EINVAL
    for fn in (lib.mo_accel, lib.mo_snapshot, lib.mo_invalidate_accel):
        assert fn(None) == M.MO_EINVAL
    assert lib.mo_drift(None, 1.0) == M.MO_EINVAL
    assert lib.mo_step(None, 1.0, 1, None) == M.MO_EINVAL
    assert lib.mo_encounters(None, 1.0, None, None, None) == M.MO_EINVAL


def test_no_cpu_fallback_without_a_device(lib):
    import numpy as np
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU container")
    from paper_2601_19654_b200 import mopal as M
    # the C ABI refuses (valid arguments, no device) ...
    ctx = C.c_void_p(None)
    fake = 0x10000
    st = lib.mo_create(C.byref(ctx), 4, 4, 1.0, 3e-4, fake, fake, fake, fake, fake, fake, 8, fake, None)
    assert st == M.MO_ECUDA and ctx.value is None
    # ... and so does the binding, loudly
    with pytest.raises(M.MopalError) as ei:
        M.Mopal(np.ones(4), np.zeros((3, 4)), np.zeros((3, 4)), np.zeros(4))
    assert ei.value.status == M.MO_ECUDA
    with pytest.raises(M.MopalError):
        M.probe_fp64_peak()


def test_product_never_touches_the_oracle():
    """Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may use oracle/."""
    bad = []
    for dirpath, _, files in os.walk(PKG):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".c", ".cpp")):
                src = open(os.path.join(dirpath, f), errors="replace").read()
                # imports, attribute use, includes or dlopens of anything under oracle/ (prose is fine)
                if re.search(r"import\s+oracle|from\s+oracle|\boracle\.\w+\(|oracle/|mopal_oracle|liboracle", src):
                    bad.append(os.path.join(dirpath, f))
    assert not bad, bad
    # and the oracle shares nothing with the CUDA path
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".c", ".h", ".py", ".sh")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            # no import / include / dlopen of the product (prose that names it is fine)
            assert not re.search(r"import\s+paper_2601|from\s+paper_2601|#\s*include\s*[\"<].*(mopal\.h|\.cuh)|libmopal\.so",
                                 src), f
