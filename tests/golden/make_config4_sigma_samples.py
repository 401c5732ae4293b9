#!/usr/bin/env python
"""Writes tests/golden/config4_sigma_samples.txt: oracle sigma-vector elements of the 1280-AO molecule.

Calls only oracle/ and workloads/ (never the CUDA path).  sigma = A x (eq. 3 / eq. 11, P:59 / P:97, R1) through the
oracle's matrix-free route with tau_oracle = 1e-15 for the first two seeded trial vectors of config 4; 256 seeded
sample positions per vector plus the position of the largest element.  (tau_oracle = 1e-20, as used for the smaller
configs, keeps ~1.4e12 primitive quartets at 1280 AOs - about a day of CPU time; at 1e-15 the neglected integrals
are 1000 times smaller than those the GPU drops at its tightest tested threshold 1e-14, one pass over ~6e10
primitive quartets: 0.5-1.5 h depending on the core count.)

    python tests/golden/make_config4_sigma_samples.py [output file]
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import tda                      # noqa: E402
from oracle.integrals import OracleBasis, num_threads  # noqa: E402
from workloads import get_config, make_basis, make_mos, make_vectors  # noqa: E402

NVEC, NSAMP, TAU_ORACLE = 2, 256, 1e-15


def main():
    cfg = get_config(4)
    basis = make_basis(cfg)
    ob = OracleBasis(basis)
    S = ob.overlap()
    C_o, C_v, eps, cond = make_mos(cfg, S)
    X = make_vectors(cfg, NVEC)
    t0 = time.time()
    sig, nq, npq = tda.sigma_matrix_free(ob, X, C_o, C_v, eps, 1.0, tau=TAU_ORACLE)
    dt = time.time() - t0
    rng = np.random.default_rng(20260116949)
    out = sys.argv[1] if len(sys.argv) > 1 else os.path.join(os.path.dirname(os.path.abspath(__file__)),
                                                             "config4_sigma_samples.txt")
    with open(out, "w") as f:
        f.write("# oracle sigma samples, config 4 (1280 AO), written by tests/golden/make_config4_sigma_samples.py\n")
        f.write("# definition: sigma = A x, eq. 3 / eq. 11 (P:59, P:97, reading R1), matrix-free oracle route, tau_oracle = %g\n" % TAU_ORACLE)
        f.write("# %d shell quartets, %d primitive quartets, %.0f s on %d threads, cond(S) = %.6g\n" % (nq, npq, dt, num_threads(), cond))
        f.write("# columns: vector index, element index (i*nvirt + a), sigma value; 'norm' lines: vector index, max|sigma|\n")
        for v in range(NVEC):
            f.write("norm %d %.17e\n" % (v, np.max(np.abs(sig[v]))))
            idx = np.unique(np.concatenate([rng.integers(0, sig.shape[1], size=NSAMP), [int(np.argmax(np.abs(sig[v])))]]))
            for i in idx:
                f.write("%d %d %.17e\n" % (v, int(i), sig[v, i]))
    print("wrote", out, "in %.0f s" % dt)


if __name__ == "__main__":
    main()
