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


def read_trajectory_samples(k: int):
    """tests/golden/config{k}_trajectory_samples.txt (oracle-written) -> (meta dict, amp {(traj, step): (idx, values)},
    norm {(traj, step): |y|^2}) or None if the file has not been generated."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config%d_trajectory_samples.txt" % k)
    if not os.path.exists(path):
        return None
    meta, amp, norm = {}, {}, {}
    for line in open(path):
        p = line.split()
        if not p or p[0].startswith("#"):
            continue
        if p[0] == "meta":
            meta[p[1]] = " ".join(p[2:])
        elif p[0] == "norm":
            norm[(int(p[1]), int(p[2]))] = float(p[3])
        elif p[0] == "amp":
            amp.setdefault((int(p[1]), int(p[2])), []).append((int(p[3]), complex(float(p[4]), float(p[5]))))
    if "seconds" not in meta:
        return None                                   # generator still running / interrupted
    out = {}
    for key, lst in amp.items():
        out[key] = (np.array([i for i, _ in lst]), np.array([v for _, v in lst]))
    return meta, out, norm


def max_amp_err(y_traj, samples):
    """y_traj [2][1+ncsf] (q, p planes of one trajectory) against stored (indices, complex values)."""
    idx, val = samples
    return float(np.max(np.abs((y_traj[0, idx] + 1j * y_traj[1, idx]) - val)))
