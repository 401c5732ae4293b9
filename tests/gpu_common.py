"""Shared set-up for the -m gpu parity tests: same seeded inputs to the oracle and to the CUDA library."""
import functools

import numpy as np


@functools.lru_cache(maxsize=None)
def setup_config(k: int, tau=None, dense: bool = False):
    """Inputs of config k with the ORACLE's S used for the MOs; returns a dict incl. an open handle."""
    import torch
    from workloads import get_config, make_basis, make_mos
    from oracle.integrals import OracleBasis
    import paper_2601_16949_b200 as R

    cfg = get_config(k)
    basis = make_basis(cfg)
    ob = OracleBasis(basis)
    S = ob.overlap()
    C_o, C_v, eps, cond = make_mos(cfg, S)
    assert cond < 1e5
    tau = cfg.tau if tau is None else tau
    dev = torch.device("cuda:0")
    h = R.Rttda(basis, torch.from_numpy(C_o).to(dev), torch.from_numpy(C_v).to(dev), eps, 1.0, tau)
    out = dict(cfg=cfg, basis=basis, ob=ob, S=S, C_o=C_o, C_v=C_v, eps=eps, h=h, dev=dev, tau=tau)
    if dense:
        from oracle import tda
        out["A"] = tda.build_A(ob.eri_tensor(), C_o, C_v, eps, 1.0)
    return out


def gpu_sigma(ctx, X):
    import torch
    Xd = torch.from_numpy(np.ascontiguousarray(X)).to(ctx["dev"])
    out = torch.empty_like(Xd)
    ctx["h"].rttda_sigma(Xd, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def gpu_fock(ctx, T):
    import torch
    Td = torch.from_numpy(np.ascontiguousarray(T)).to(ctx["dev"])
    out = torch.empty_like(Td)
    ctx["h"].rttda_fock(Td, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def rel_inf(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))
