"""-m gpu test of rttda_fock_static (include/rttda.h): the Fock build whose every workspace lives in one file-scope
device array of the library, for callers that cannot call cudaMalloc.  Checked against the existing rttda_fock path on
the same inputs, on consecutive calls that share (and must not leak through) the static scratch.

Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test."""
import numpy as np
import pytest

from gpu_common import rel_inf, setup_config

pytestmark = pytest.mark.gpu

FOCK_TOL = 1e-12          # the tolerance of the Fock-matrix parity tests (tests/test_gpu_parity.py, test_gpu_dshells.py)


def _new_handle(ctx, cx=1.0, tau=None):
    import torch
    import paper_2601_16949_b200 as R
    dev = ctx["dev"]
    return R.Rttda(ctx["basis"], torch.from_numpy(ctx["C_o"]).to(dev), torch.from_numpy(ctx["C_v"]).to(dev), ctx["eps"], cx,
                   ctx["tau"] if tau is None else tau)


def _run(fn, T, dev):
    import torch
    Td = torch.from_numpy(np.ascontiguousarray(T)).to(dev)
    F = torch.full_like(Td, float("nan"))                     # every output element must be written
    fn(Td, F)
    torch.cuda.synchronize()
    return F.cpu().numpy()


@pytest.mark.parametrize("k", [1, 6, 2])
def test_fock_static_matches_fock_on_consecutive_calls(k):
    """configs 1 (30 AO, s/p), 6 (60 AO with d shells: general kernel path) and 2 (200 AO): calls in a row with
    different densities and different batch widths (the scratch is laid out per call), each against rttda_fock."""
    import torch
    ctx = setup_config(k)
    N = ctx["basis"].nao
    rng = np.random.default_rng(700 + k)
    h = _new_handle(ctx)
    dev = ctx["dev"]
    free = []
    outs = []
    for nvec in (5, 2, 8, 1):
        T = rng.standard_normal((nvec, N, N))                 # not symmetric
        outs.append((T, _run(h.rttda_fock_static, T, dev)))
        free.append(torch.cuda.mem_get_info()[0])
    # after the first call (lazy kernel loading) the static path leaves the device's free memory untouched
    assert free[1] == free[2] == free[3]
    for T, got in outs:                                        # the existing path, which allocates its workspaces
        ref = _run(h.rttda_fock, T, dev)
        assert np.all(np.isfinite(got))
        assert rel_inf(got, ref) < FOCK_TOL
    # and once more after the allocating path has run: same answer, scratch contents of other calls do not leak
    T, first = outs[0]
    again = _run(h.rttda_fock_static, T, dev)
    assert rel_inf(again, first) < FOCK_TOL
    h.close()


def test_fock_static_exchange_fraction_and_range_separation():
    import paper_2601_16949_b200 as R
    ctx = setup_config(1)
    N = ctx["basis"].nao
    T = np.random.default_rng(77).standard_normal((3, N, N))
    h = _new_handle(ctx, cx=0.19, tau=1e-14)
    h.rttda_set_option(R.OPT_CX_LR, 0.46)
    h.rttda_set_option(R.OPT_RS_OMEGA, 0.33)
    a = _run(h.rttda_fock_static, T, ctx["dev"])
    b = _run(h.rttda_fock, T, ctx["dev"])
    assert rel_inf(a, b) < FOCK_TOL
    h.close()


def test_fock_static_rejects_what_does_not_fit():
    import torch
    import paper_2601_16949_b200 as R
    ctx = setup_config(1)
    N = ctx["basis"].nao
    h = _new_handle(ctx)
    T9 = torch.zeros((9, N, N), dtype=torch.float64, device=ctx["dev"])
    with pytest.raises(R.RttdaError, match="nvec"):
        h.rttda_fock_static(T9, torch.empty_like(T9))
    h.close()
    big = setup_config(7)                                      # 320 basis functions: 140 MB staging buffer alone
    hb = _new_handle(big)
    Tb = torch.zeros((2, 320, 320), dtype=torch.float64, device=big["dev"])
    with pytest.raises(R.RttdaError, match="static array holds"):
        hb.rttda_fock_static(Tb, torch.empty_like(Tb))
    hb.close()
