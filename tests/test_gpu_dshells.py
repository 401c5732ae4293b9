"""-m gpu parity tests of the Cartesian d shells: the general-angular-momentum path of
csrc/eri_generic.cu against the oracle, on the 60-AO molecule with one d shell per heavy centre (workloads key 6) and on
random molecules with contracted d shells.  Same tolerances as everywhere: sigma 1e-10 relative, amplitudes 1e-8."""
import numpy as np
import pytest

from gpu_common import gpu_fock, gpu_sigma, rel_inf, setup_config

pytestmark = pytest.mark.gpu

SIGMA_TOL = 1e-10
AMP_TOL = 1e-8


def _handle(basis, C_o, C_v, eps, cx, tau):
    import torch
    import paper_2601_16949_b200 as R
    dev = torch.device("cuda:0")
    return R.Rttda(basis, torch.from_numpy(np.ascontiguousarray(C_o)).to(dev),
                   torch.from_numpy(np.ascontiguousarray(C_v)).to(dev), eps, cx, tau)


def _sigma(h, X):
    import torch
    Xd = torch.from_numpy(np.ascontiguousarray(X)).to("cuda:0")
    out = torch.empty_like(Xd)
    h.rttda_sigma(Xd, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def _fock(h, T):
    import torch
    Td = torch.from_numpy(np.ascontiguousarray(T)).to("cuda:0")
    F = torch.empty_like(Td)
    h.rttda_fock(Td, F)
    torch.cuda.synchronize()
    return F.cpu().numpy()


def test_d_molecule_one_electron_and_counts():
    import paper_2601_16949_b200 as R
    ctx = setup_config(6)
    ob, basis = ctx["ob"], ctx["basis"]
    assert basis.nao == 60 and int(np.sum(basis.sh_l == 2)) == 4
    S, D = R.rttda_overlap(basis), R.rttda_dipole_ao(basis)
    assert np.max(np.abs(S - ctx["S"])) < 1e-14
    assert np.max(np.abs(D - ob.dipole())) < 1e-13
    Q = ob.schwarz()
    T = np.random.default_rng(0).standard_normal((1, 60, 60))
    for tau in (1e-12, 1e-6, 1e-3):
        h = _handle(basis, ctx["C_o"], ctx["C_v"], ctx["eps"], 1.0, tau)
        _, _, nq, npq = ob.jk(T, tau=tau, Q=Q)
        assert int(h.rttda_get_info("nquartets")) == nq and int(h.rttda_get_info("nprim_quartets")) == npq
        h.close()


@pytest.mark.parametrize("nvec", [1, 2, 5, 8])
def test_d_molecule_fock_vs_oracle_jk(nvec):
    """F = 2 J[T] - c_x K[T] for non-symmetric densities, every class from (ss|ss) to (dd|dd)."""
    ctx = setup_config(6)
    ob, N = ctx["ob"], ctx["basis"].nao
    T = np.random.default_rng(40 + nvec).standard_normal((nvec, N, N))
    J, K, _, _ = ob.jk(T, tau=0.0)
    for cx in (1.0, 0.3):
        h = _handle(ctx["basis"], ctx["C_o"], ctx["C_v"], ctx["eps"], cx, 0.0)
        assert rel_inf(_fock(h, T), 2 * J - cx * K) < 1e-12
        h.close()


def test_d_molecule_unit_densities_single_integrals():
    """T = e_lam e_sig^T picks single integrals: F_{mu nu} = 2 (mu nu|lam sig) - (mu lam|nu sig); compared element by
    element with the oracle's ERI tensor for AO pairs inside and across the d shells."""
    ctx = setup_config(6)
    ob, basis = ctx["ob"], ctx["basis"]
    N = basis.nao
    eri = ob.eri_tensor()
    off = basis.ao_off
    d_sh = [s for s in range(basis.nshells) if basis.sh_l[s] == 2]
    picks = [(off[d_sh[0]] + 1, off[d_sh[1]] + 4), (off[d_sh[0]], off[d_sh[0]] + 3), (off[d_sh[2]] + 5, 0), (2, off[d_sh[3]] + 2)]
    T = np.zeros((len(picks), N, N))
    for v, (lam, sig) in enumerate(picks):
        T[v, lam, sig] = 1.0
    h = _handle(basis, ctx["C_o"], ctx["C_v"], ctx["eps"], 1.0, 0.0)
    F = _fock(h, T)
    h.close()
    for v, (lam, sig) in enumerate(picks):
        ref = 2 * eri[:, :, lam, sig] - eri[:, lam, :, sig]
        assert np.max(np.abs(F[v] - ref)) < 1e-13 * max(1.0, np.max(np.abs(ref)))


def test_d_molecule_sigma_and_propagation_vs_dense_oracle():
    """sigma = A X against the oracle's dense A (600 x 600 from the N^4 tensor), then 10 RK4 steps under a cw field."""
    import torch
    from workloads import make_vectors
    from oracle import tda
    ctx = setup_config(6, dense=True)
    cfg, A = ctx["cfg"], ctx["A"]
    X = make_vectors(cfg, 6)
    got = gpu_sigma(ctx, X)                                          # the config's tau = 1e-12: screening error included
    assert rel_inf(got, tda.sigma_dense(A, X)) < SIGMA_TOL
    h2 = _handle(ctx["basis"], ctx["C_o"], ctx["C_v"], ctx["eps"], 1.0, 0.0)
    assert rel_inf(_sigma(h2, X), tda.sigma_dense(A, X)) < 1e-12
    h2.close()
    # propagation
    n = A.shape[0]
    D = ctx["ob"].dipole()
    fld = dict(cfg.fields[0])
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(D, ctx["C_o"], ctx["C_v"], fld["dir"])
    y0 = np.zeros(n + 1, dtype=complex); y0[0] = 1.0
    yref, logref = tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, fld, 0.0, cfg.dt, cfg.nsteps)
    y = torch.zeros((1, 2, n + 1), dtype=torch.float64, device=ctx["dev"])
    y[:, 0, 0] = 1.0
    log = torch.zeros((cfg.nsteps, 1, 3), dtype=torch.float64, device=ctx["dev"])
    ctx["h"].rttda_propagate(y, [fld], 0.0, cfg.dt, cfg.nsteps, log)
    torch.cuda.synchronize()
    yy = y.cpu().numpy()
    err = np.max(np.abs((yy[0, 0] + 1j * yy[0, 1]) - yref))
    assert np.max(np.abs(log.cpu().numpy()[:, 0, :] - logref)) < 1e-11
    print("d molecule: amplitude error after %d steps %.2e" % (cfg.nsteps, err))
    assert err < AMP_TOL


@pytest.mark.parametrize("cx,cx_lr,omega", [(0.19, 0.46, 0.33), (0.0, 1.0, 0.8)])
def test_d_molecule_range_separated_exchange(cx, cx_lr, omega):
    """The CAM-type operator on the d-shell molecule: erf-attenuated integrals of the general path."""
    import paper_2601_16949_b200 as R
    from workloads import make_vectors
    from oracle import tda
    ctx = setup_config(6, dense=True)
    ob = ctx["ob"]
    A = tda.build_A_rs(ob.eri_tensor(), ob.eri_tensor_erf(omega), ctx["C_o"], ctx["C_v"], ctx["eps"], cx, cx_lr)
    X = make_vectors(ctx["cfg"], 4)
    h = _handle(ctx["basis"], ctx["C_o"], ctx["C_v"], ctx["eps"], cx, 1e-14)
    h.rttda_set_option(R.OPT_CX_LR, cx_lr)
    h.rttda_set_option(R.OPT_RS_OMEGA, omega)
    assert rel_inf(_sigma(h, X), tda.sigma_dense(A, X)) < 1e-12
    h.close()


@pytest.mark.parametrize("seed", [1, 2, 3, 4, 5, 6, 7, 8])
def test_random_molecules_with_contracted_d_shells(seed):
    """Random centres, s/p/d shells with contraction depths 1..3 on the d shells too, tau in {0, 1e-10}."""
    import paper_2601_16949_b200 as R
    from workloads import Basis
    from workloads.molecules import orthonormalizer
    from oracle.integrals import OracleBasis
    rng = np.random.default_rng(9000 + seed)
    nc = int(rng.integers(2, 5))
    centers = np.zeros((nc, 3))
    for c in range(nc):
        while True:
            x = rng.uniform(0.0, 4.0, size=3)
            if c == 0 or np.min(np.linalg.norm(centers[:c] - x, axis=1)) > 1.6:
                centers[c] = x
                break
    sh_center, sh_l, sh_nprim, exps, coefs = [], [], [], [], []
    for c in range(nc):
        nsh = int(rng.integers(2, 5))
        ls = list(rng.integers(0, 3, size=nsh))
        if c == 0:
            ls[0] = 2
        for l in ls:
            npr = int(rng.integers(1, 4))
            lo, hi = ((0.2, 8.0), (0.3, 2.5), (0.4, 1.8))[l]
            sh_center.append(c); sh_l.append(int(l)); sh_nprim.append(npr)
            exps.extend(np.exp(rng.uniform(np.log(lo), np.log(hi), size=npr)).tolist())
            coefs.extend(rng.uniform(0.2, 1.0, size=npr).tolist())
    sh_nprim = np.asarray(sh_nprim, dtype=np.int32)
    basis = Basis(np.ascontiguousarray(centers), np.asarray(sh_center, dtype=np.int32), np.asarray(sh_l, dtype=np.int32),
                  sh_nprim, np.concatenate([[0], np.cumsum(sh_nprim)[:-1]]).astype(np.int32), np.asarray(exps), np.asarray(coefs))
    ob = OracleBasis(basis)
    N = basis.nao
    S = ob.overlap()
    assert np.max(np.abs(R.rttda_overlap(basis) - S)) < 1e-13
    X12, cond = orthonormalizer(S)
    if cond > 1e6:
        pytest.skip("near-singular overlap (cond %.1e)" % cond)
    Q, _ = np.linalg.qr(rng.standard_normal((N, N)))
    C = X12 @ Q
    nocc = max(1, N // 4)
    eps = np.concatenate([np.sort(rng.uniform(-1.0, -0.3, nocc)), np.sort(rng.uniform(0.05, 2.0, N - nocc))])
    T = rng.standard_normal((3, N, N))
    for tau in (0.0, 1e-10):
        J, K, nq, npq = ob.jk(T, tau=tau)
        h = _handle(basis, C[:, :nocc], C[:, nocc:], eps, 1.0, tau)
        assert rel_inf(_fock(h, T), 2 * J - K) < 1e-12
        assert int(h.rttda_get_info("nquartets")) == nq and int(h.rttda_get_info("nprim_quartets")) == npq
        h.close()


def test_d320_sigma_vs_matrix_free_oracle():
    """320 basis functions with d shells (the size of the paper's smallest Table-3 molecule; workloads key 7):
    sigma for two vectors against the oracle's matrix-free route (screened at 1e-16), 13.9 M unique shell quartets in
    every class from (ss|ss) to (dd|dd), several evaluation blocks and ragged 32-ket batches per class."""
    from workloads import make_vectors
    from oracle import tda
    ctx = setup_config(7, tau=1e-14)
    assert ctx["basis"].nao == 320
    X = make_vectors(ctx["cfg"], 2)
    ref, nq, _ = tda.sigma_matrix_free(ctx["ob"], X, ctx["C_o"], ctx["C_v"], ctx["eps"], 1.0, tau=1e-16)
    got = gpu_sigma(ctx, X)
    err = rel_inf(got, ref)
    print("d-320: sigma rel err %.2e (%d oracle quartets)" % (err, nq))
    assert err < SIGMA_TOL
    assert abs(X[0] @ got[1] - X[1] @ got[0]) < 1e-11                 # A is symmetric


def test_d1884_fock_sampled_elements_and_properties():
    """1884 basis functions in the shape of the paper's largest molecule (Table 3: 120 heavy centres x 15 BF
    with one Cartesian d shell each + 42 H-like x 2 BF; workloads key 8), 1.56e9 unique shell quartets, every kernel of
    the d path at full size (pipeline mode, unrolled evaluation, a-list digestion, (dd|dd) on the general kernels):
    F elements at sampled AO pairs - d, p and s functions - against the oracle's definition-level J and K (no screening,
    no symmetry), plus properties that hold at any size."""
    ctx = setup_config(8)
    ob, basis = ctx["ob"], ctx["basis"]
    N = basis.nao
    assert N == 1884
    rng = np.random.default_rng(8)
    X = rng.standard_normal((2, ctx["cfg"].nocc, ctx["cfg"].nvirt))
    X /= np.linalg.norm(X.reshape(2, -1), axis=1)[:, None, None]
    T = np.stack([ctx["C_o"] @ x @ ctx["C_v"].T for x in X])              # transition densities, non-symmetric
    F = gpu_fock(ctx, T)
    off = basis.ao_off
    d_sh = [s for s in range(basis.nshells) if basis.sh_l[s] == 2]
    p_sh = [s for s in range(basis.nshells) if basis.sh_l[s] == 1]
    mu = np.array([off[d_sh[3]] + 1, off[d_sh[50]] + 3, off[p_sh[7]] + 2, 0, off[d_sh[100]] + 5])
    nu = np.array([off[d_sh[3]] + 4, off[p_sh[90]] + 1, off[d_sh[77]] + 0, N - 1, off[d_sh[100]] + 5])
    J, K = ob.jk_samples(T, mu, nu)
    got = F[:, mu, nu].T
    scale = np.max(np.abs(F))
    err = np.max(np.abs(got - (2 * J - K))) / scale
    print("d-1884: sampled Fock elements, max error / max|F| = %.2e" % err)
    assert err < SIGMA_TOL
    F2 = gpu_fock(ctx, np.stack([T[0] + T[0].T, 2.0 * T[1] - 0.5 * T[0]]))
    assert np.max(np.abs(F2[0] - (F[0] + F[0].T))) / scale < SIGMA_TOL     # F[T^T] = F[T]^T
    assert np.max(np.abs(F2[1] - (2.0 * F[1] - 0.5 * F[0]))) / scale < SIGMA_TOL


def test_d_molecule_eigenpairs_and_sso_step_vs_dense_oracle():
    """The other consumers of the sigma build on a basis with d shells: the lowest TI-TDA eigenpairs (rttda_eigs) against
    eigh of the oracle's dense A, and 10 steps of the paper's split-operator propagator against the oracle's."""
    import torch
    from oracle import tda
    ctx = setup_config(6, dense=True)
    A, h, cfg = ctx["A"], ctx["h"], ctx["cfg"]
    n = A.shape[0]
    w = np.linalg.eigvalsh(A)
    X = torch.zeros((4, n), dtype=torch.float64, device=ctx["dev"])
    om, rs, it, ns = h.rttda_eigs(4, X, 8, tol=1e-9, maxiter=100)
    Xh = X.cpu().numpy()
    assert np.max(np.abs(om - w[:4])) < 1e-8           # tau = 1e-12 in A's integrals: eigenvalues move by ~1e-11
    assert np.max(np.linalg.norm(Xh @ A.T - om[:, None] * Xh, axis=1)) < 5e-8
    fld = dict(cfg.fields[0])
    D = ctx["ob"].dipole()
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(D, ctx["C_o"], ctx["C_v"], fld["dir"])
    y0 = np.zeros(n + 1, dtype=complex); y0[0] = 1.0
    yref, _ = tda.sso_dense(A, Doo, Dvv, Dov, D00, y0, fld, 0.0, cfg.dt, cfg.nsteps)
    y = torch.zeros((1, 2, n + 1), dtype=torch.float64, device=ctx["dev"])
    y[:, 0, 0] = 1.0
    h.rttda_propagate_sso(y, [fld], 0.0, cfg.dt, cfg.nsteps, None)
    torch.cuda.synchronize()
    yy = y.cpu().numpy()
    assert np.max(np.abs((yy[0, 0] + 1j * yy[0, 1]) - yref)) < AMP_TOL
