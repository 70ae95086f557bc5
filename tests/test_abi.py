"""The C-ABI library loads and exports every symbol include/fk.h declares; host-only entry
points behave (no compute calls here: these tests run without a GPU)."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2104_14561_b200 import build, binding
    build.build_library()                     # nvcc cross-compiles for sm_100a without a GPU
    binding.lib()
    return binding


def declared_functions():
    text = open(os.path.join(ROOT, "include", "fk.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fk_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_four_north_star_calls():
    names = declared_functions()
    for need in ("fk_create", "fk_set_coeffs", "fk_evolve", "fk_read"):
        assert need in names


def test_library_exports_every_declared_symbol(B):
    L = ctypes.CDLL(B.LIB_PATH)
    names = declared_functions()
    assert len(names) >= 10
    for name in names:
        assert hasattr(L, name), f"{name} declared in include/fk.h but not exported"
    assert sorted(B.EXPORTS) == names, "binding.EXPORTS and include/fk.h disagree"


def test_library_is_built_for_sm_100a_only(B):
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", B.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_gauss_hermite_closed_forms_and_moments(B):
    a, w = B.fk_gauss_hermite(1)
    assert a[0] == 0.0 and abs(w[0] - 1.0) < 1e-15
    a, w = B.fk_gauss_hermite(2)
    np.testing.assert_allclose(a, [-1 / math.sqrt(2), 1 / math.sqrt(2)], atol=1e-15)
    np.testing.assert_allclose(w, [0.5, 0.5], atol=1e-15)
    a, w = B.fk_gauss_hermite(3)
    np.testing.assert_allclose(a, [-math.sqrt(1.5), 0.0, math.sqrt(1.5)], atol=1e-15)
    np.testing.assert_allclose(w, [1 / 6, 2 / 3, 1 / 6], atol=1e-15)
    for Q in (6, 8, 16, 32):
        a, w = B.fk_gauss_hermite(Q)
        assert np.all(np.diff(a) > 0)
        assert abs(w.sum() - 1.0) < 1e-14
        # E[xi^(2m)] = (2m-1)!!/2^m under pi^{-1/2} exp(-xi^2), exact for m < Q
        for m in range(1, min(Q, 8)):
            exact = np.prod(np.arange(2 * m - 1, 0, -2)) / 2.0 ** m
            assert abs((w * a ** (2 * m)).sum() - exact) < 1e-12 * max(1.0, exact)
    with pytest.raises(B.FkError):
        B.fk_gauss_hermite(33)


def test_gauss_hermite_agrees_with_numpy(B):
    for Q in (6, 8, 16):
        a, w = B.fk_gauss_hermite(Q)
        ra, rw = np.polynomial.hermite.hermgauss(Q)
        np.testing.assert_allclose(a, ra, atol=1e-13)
        np.testing.assert_allclose(w, rw / math.sqrt(math.pi), atol=1e-14)


def test_create_validates_and_has_no_cpu_path(B):
    import torch
    x = [np.linspace(-1, 1, 11)]
    kinds, vals = [[0, 0]], [[1.0, 1.0]]
    bad = [dict(dt=-1.0), dict(N=0), dict(Q=[0]), dict(Q=[33]), dict(x=[np.array([0.0, 1.0])]),
           dict(x=[np.array([0.0, 0.5, 0.5, 1.0])]), dict(face_kind=[[0, 7]]), dict(coeff_slots=99)]
    for kw in bad:
        args = dict(x=x, dt=0.01, N=10, Q=[4], face_kind=kinds, face_value=vals)
        args.update(kw)
        with pytest.raises(B.FkError) as e:
            B.fk_create(**args)
        assert e.value.code == B.FK_EINVAL, kw
    if not torch.cuda.is_available():
        with pytest.raises(B.FkError) as e:
            B.fk_create(x, 0.01, 10, [4], kinds, vals)
        assert e.value.code == B.FK_ECUDA
        assert "no CPU path" in str(e.value)


def test_missing_library_fails_loudly(B, monkeypatch):
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", os.path.join(ROOT, "no_such_dir", "libfk_b200.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.lib()
