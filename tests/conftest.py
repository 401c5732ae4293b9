import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running CPU test")


@pytest.fixture(scope="session")
def tiny():
    """Config 1 (30 AOs) with the oracle's own basis, S, MOs and dense A."""
    import numpy as np
    from workloads import get_config, make_basis, make_mos
    from oracle.integrals import OracleBasis
    from oracle import tda
    cfg = get_config(1)
    basis = make_basis(cfg)
    ob = OracleBasis(basis)
    S = ob.overlap()
    C_o, C_v, eps, cond = make_mos(cfg, S)
    eri = ob.eri_tensor()
    A = tda.build_A(eri, C_o, C_v, eps, 1.0)
    D = ob.dipole()
    return dict(cfg=cfg, basis=basis, ob=ob, S=S, C_o=C_o, C_v=C_v, eps=eps, eri=eri, A=A, D=D,
                cond=cond)
