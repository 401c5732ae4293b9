#!/usr/bin/env python
"""Writes tests/golden/config4_sigma_samples.txt: oracle sigma-vector elements of the 1280-AO molecule.

Calls only oracle/ and workloads/ (never the CUDA path).  sigma = A x (eq. 3 / eq. 11, P:59 / P:97, R1) through the
oracle's EXTENDED-PRECISION matrix-free route (`tda.sigma_matrix_free_ld`: FP64 integral values, every sum and MO
transform in x87 long double) with tau_oracle = 1e-17, for 8 of the 32 seeded trial vectors of config 5
(`make_vectors(cfg, 32)`; its first 2 / 8 / 16 rows are the vectors of the nvec = 2 / 8 / 16 points): 256 seeded
sample positions per vector plus the position of the largest element.  The neglected integrals are 1e3 (1e5) times
smaller than those the CUDA path drops at tau = 1e-14 (1e-12); the screening error of sigma scales as ~2e3 tau
(DESIGN.md section 11), i.e. ~2e-14 here.  One pass over ~6.7e10 primitive quartets: hours on 8 cores.

The previous file (FP64 accumulation, tau_oracle = 1e-15, vectors 0 and 1, same sample positions) is kept as
config4_sigma_samples_fp64.txt: the difference between the two is the noise floor of the FP64 oracle route at
cond(S) = 4.5e4 (tests/test_oracle_tda.py).

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

NVEC_SET, VECS, NSAMP, TAU_ORACLE = 32, (0, 1, 5, 7, 12, 15, 22, 31), 256, 1e-17


def main():
    cfg = get_config(4)
    basis = make_basis(cfg)
    ob = OracleBasis(basis)
    S = ob.overlap()
    C_o, C_v, eps, cond = make_mos(cfg, S)
    X = make_vectors(cfg, NVEC_SET)[list(VECS)]
    t0 = time.time()
    sig, nq, npq = tda.sigma_matrix_free_ld(ob, X, C_o, C_v, eps, 1.0, tau=TAU_ORACLE)
    sig = sig.astype(np.float64)
    dt = time.time() - t0
    rng = np.random.default_rng(20260116949)
    out = sys.argv[1] if len(sys.argv) > 1 else os.path.join(os.path.dirname(os.path.abspath(__file__)),
                                                             "config4_sigma_samples.txt")
    with open(out, "w") as f:
        f.write("# oracle sigma samples, config 4/5 (1280 AO), written by tests/golden/make_config4_sigma_samples.py\n")
        f.write("# definition: sigma = A x, eq. 3 / eq. 11 (P:59, P:97, reading R1), matrix-free oracle route in long double, tau_oracle = %g\n" % TAU_ORACLE)
        f.write("# %d shell quartets, %d primitive quartets, %.0f s on %d threads, cond(S) = %.6g\n" % (nq, npq, dt, num_threads(), cond))
        f.write("# vectors: rows %s of make_vectors(config 4, %d)\n" % (",".join(map(str, VECS)), NVEC_SET))
        f.write("# columns: vector index, element index (i*nvirt + a), sigma value; 'norm' lines: vector index, max|sigma|\n")
        for k, v in enumerate(VECS):
            f.write("norm %d %.17e\n" % (v, np.max(np.abs(sig[k]))))
            idx = np.unique(np.concatenate([rng.integers(0, sig.shape[1], size=NSAMP), [int(np.argmax(np.abs(sig[k])))]]))
            for i in idx:
                f.write("%d %d %.17e\n" % (v, int(i), sig[k, i]))
    print("wrote", out, "in %.0f s" % dt)


if __name__ == "__main__":
    main()
