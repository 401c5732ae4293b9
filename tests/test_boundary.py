"""CPU-side checks of the C-ABI boundary: the library loads without a GPU, exports every symbol that
include/rttda.h declares, the binding lists the same names, host-only helpers work, and compute calls
fail loudly (no CPU fallback)."""
import ctypes as ct
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "rttda.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rttda_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def R():
    import paper_2601_16949_b200 as R
    if not os.path.exists(R.LIB_PATH):
        from paper_2601_16949_b200 import build
        build.build()
    return R


def test_header_symbols_are_exported_and_bound(R):
    names = _declared()
    assert len(names) >= 14
    L = ct.CDLL(R.LIB_PATH)
    for n in names:
        assert hasattr(L, n), "librttda.so does not export %s" % n
    assert sorted(R.EXPORTS) == names


def test_host_helpers_match_definitions_without_gpu(R):
    """rttda_overlap: unit diagonal (R11), symmetric, positive definite; dipole origin-shift rule."""
    from workloads import get_config, make_basis
    basis = make_basis(get_config(1))
    S = R.rttda_overlap(basis)
    assert np.allclose(np.diag(S), 1.0, atol=1e-14) and np.allclose(S, S.T, atol=1e-15)
    assert np.linalg.eigvalsh(S)[0] > 0
    D = R.rttda_dipole_ao(basis)
    shifted = type(basis)(basis.centers + np.array([0.3, -0.2, 0.5]), basis.sh_center, basis.sh_l,
                          basis.sh_nprim, basis.sh_off, basis.exps, basis.coefs)
    D2 = R.rttda_dipole_ao(shifted)
    for k, c in enumerate([0.3, -0.2, 0.5]):
        assert np.allclose(D2[k], D[k] + c * S, atol=1e-13)


def test_no_cpu_fallback(R):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from workloads import get_config, make_basis, make_mos
    cfg = get_config(1)
    basis = make_basis(cfg)
    C_o, C_v, eps, _ = make_mos(cfg, R.rttda_overlap(basis))
    with pytest.raises((R.RttdaError, AssertionError)):
        R.Rttda(basis, torch.from_numpy(C_o), torch.from_numpy(C_v), eps)
    # straight through the C ABI with host pointers: must report "no CUDA device", not compute
    from paper_2601_16949_b200.binding import _BasisHolder
    b = _BasisHolder(basis)
    hnd = ct.c_void_p(0)
    rc = R.lib().rttda_create(ct.byref(hnd), ct.byref(b.c), b.nao, cfg.nocc, cfg.nvirt,
                              ct.c_void_p(C_o.ctypes.data), ct.c_void_p(C_v.ctypes.data),
                              ct.c_void_p(eps.ctypes.data), ct.c_double(1.0), ct.c_double(1e-12), ct.c_void_p(0))
    assert rc == -3 and b"no CUDA device" in R.lib().rttda_last_error()


def test_spectrum_argument_errors_and_no_fallback_without_gpu(R):
    """rttda_spectrum: argument errors are reported before any device work; with valid arguments and no CUDA device
    the call fails (no host DFT behind it)."""
    import torch
    L = R.lib()
    R0 = np.array([[1.0, 0.0]])
    buf = np.zeros((3, 1, 3))
    om, inten = np.zeros(3), np.zeros((2, 3))
    args = lambda n, dt, pad, nout: (1, n, ct.c_void_p(R0.ctypes.data), ct.c_void_p(buf.ctypes.data), ct.c_double(dt),
                                     pad, nout, ct.c_void_p(om.ctypes.data), ct.c_void_p(inten.ctypes.data),
                                     ct.c_void_p(0))
    assert L.rttda_spectrum(*args(3, 0.1, 0, 4)) == -1 and b"nout" in L.rttda_last_error()
    assert L.rttda_spectrum(*args(3, 0.0, 0, 3)) == -1
    assert L.rttda_spectrum(*args(-1, 0.1, 0, 0)) == -1
    assert L.rttda_spectrum(*args(0, 0.1, 0, 0)) == 0            # one sample, no padding: empty frequency grid
    if not torch.cuda.is_available():
        assert L.rttda_spectrum(*args(3, 0.1, 0, 3)) != 0
        assert np.all(om == 0.0) and np.all(inten == 0.0)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2601_16949_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert "oracle" not in open(os.path.join(dp, f)).read().replace("shares nothing with oracle/", "") \
                    .replace("never imports oracle/", ""), f
