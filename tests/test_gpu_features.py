"""-m gpu parity tests of the pieces around the sigma build: exchange fraction c_x, pulse shapes on the device path,
host-buffer entry points, wide density batches at a size with several a-list tiles, the DMMA GEMM on its own."""
import numpy as np
import pytest

from gpu_common import gpu_fock, gpu_sigma, rel_inf, setup_config

pytestmark = pytest.mark.gpu

SIGMA_TOL = 1e-10
AMP_TOL = 1e-8


def _handle(ctx, cx, tau):
    import torch
    import paper_2601_16949_b200 as R
    return R.Rttda(ctx["basis"], torch.from_numpy(ctx["C_o"]).to(ctx["dev"]), torch.from_numpy(ctx["C_v"]).to(ctx["dev"]),
                   ctx["eps"], cx, tau)


def _sigma(h, X, dev):
    import torch
    Xd = torch.from_numpy(np.ascontiguousarray(X)).to(dev)
    out = torch.empty_like(Xd)
    h.rttda_sigma(Xd, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("cx", [0.0, 0.5, 1.0])
def test_sigma_exchange_fraction_tiny_dense_and_config2_matrix_free(cx):
    """A = d_eps + 2 (ia|jb) - c_x (ij|ab) (eq. 3 under R1) for c_x != 1: the library's `cx` argument against the
    oracle's dense A(c_x) on config 1 and its matrix-free route on config 2 (nvec 6)."""
    from workloads import make_vectors
    from oracle import tda
    ctx = setup_config(1, dense=True)
    A = tda.build_A(ctx["ob"].eri_tensor(), ctx["C_o"], ctx["C_v"], ctx["eps"], cx)
    X = make_vectors(ctx["cfg"], 5)
    h = _handle(ctx, cx, 1e-12)
    assert rel_inf(_sigma(h, X, ctx["dev"]), tda.sigma_dense(A, X)) < 1e-12
    h.close()
    ctx2 = setup_config(2)
    X = make_vectors(ctx2["cfg"], 6)
    ref, _, _ = tda.sigma_matrix_free(ctx2["ob"], X, ctx2["C_o"], ctx2["C_v"], ctx2["eps"], cx, tau=1e-20)
    h = _handle(ctx2, cx, 1e-12)
    got = _sigma(h, X, ctx2["dev"])
    h.close()
    assert rel_inf(got, ref) < SIGMA_TOL


def test_propagate_chirped_and_tl_pulse_with_exchange_fraction():
    """eq. 18c / 18d on the device path: a chirped and a transform-limited Gaussian pulse as two trajectories of one
    batch, on a handle with c_x = 0.5, against the oracle's dense RK4."""
    import torch
    from oracle import tda
    ctx = setup_config(1, dense=True)
    cx = 0.5
    A = tda.build_A(ctx["ob"].eri_tensor(), ctx["C_o"], ctx["C_v"], ctx["eps"], cx)
    n = A.shape[0]
    D = ctx["ob"].dipole()
    fields = [{"type": "chirp", "E0": 0.05, "omega": 0.45, "beta": 0.6, "t0": 0.9, "sigma": 0.5, "dir": (0.2, -0.5, 0.8)},
              {"type": "tl", "E0": 0.05, "omega": 0.45, "t0": 0.9, "sigma": 0.5, "dir": (0.2, -0.5, 0.8)}]
    dt, nsteps = 0.05, 36
    h = _handle(ctx, cx, 1e-12)
    y = np.zeros((2, 2, n + 1)); y[:, 0, 0] = 1.0
    yd = torch.from_numpy(y).to(ctx["dev"])
    log = torch.zeros((nsteps, 2, 3), dtype=torch.float64, device=ctx["dev"])
    h.rttda_propagate(yd, fields, 0.0, dt, nsteps, log)
    torch.cuda.synchronize()
    yh, lg = yd.cpu().numpy(), log.cpu().numpy()
    h.close()
    finals = []
    for t, f in enumerate(fields):
        Doo, Dvv, Dov, D00 = tda.mo_dipoles(D, ctx["C_o"], ctx["C_v"], f["dir"])
        y0 = np.zeros(n + 1, dtype=complex); y0[0] = 1.0
        yr, lr = tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, f, 0.0, dt, nsteps)
        assert np.max(np.abs(yh[t, 0] - yr.real)) < 1e-12 and np.max(np.abs(yh[t, 1] - yr.imag)) < 1e-12
        assert np.max(np.abs(lg[:, t, :] - lr)) < 1e-12
        finals.append(yr)
    assert np.max(np.abs(finals[0] - finals[1])) > 1e-5            # the chirp does change the trajectory


def test_propagate_host_and_sigma_host_vs_oracle():
    """rttda_propagate_host / rttda_sigma_host (host buffers, copies inside): same numbers as the oracle."""
    from workloads import make_vectors
    from oracle import tda
    ctx = setup_config(1, dense=True)
    A, h = ctx["A"], ctx["h"]
    n = A.shape[0]
    X = make_vectors(ctx["cfg"], 3)
    out = np.zeros_like(X)
    h.rttda_sigma_host(X, out)
    assert rel_inf(out, tda.sigma_dense(A, X)) < 1e-12
    f = {"type": "sin2", "E0": 0.04, "omega": 0.5, "T_env": 1.2, "dir": (0.0, 0.6, 0.8)}
    D = ctx["ob"].dipole()
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(D, ctx["C_o"], ctx["C_v"], f["dir"])
    y0 = np.zeros(n + 1, dtype=complex); y0[0] = 1.0
    yr, lr = tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, f, 0.0, 0.05, 20)
    y = np.zeros((1, 2, n + 1)); y[0, 0, 0] = 1.0
    log = np.zeros((20, 1, 3))
    h.rttda_propagate_host(y, [f], 0.0, 0.05, 20, log)
    assert np.max(np.abs(y[0, 0] - yr.real)) < 1e-12 and np.max(np.abs(y[0, 1] - yr.imag)) < 1e-12
    assert np.max(np.abs(log[:, 0, :] - lr)) < 1e-12


def test_continue_flag_keeps_kick_and_reference():
    """RTTDA_FIELD_CONTINUE: a delta-kick run split into two calls equals the single call (state and R(t) log); without
    the flag the second call kicks again."""
    import torch
    ctx = setup_config(1)
    h = ctx["h"]
    n = h.ncsf
    f = {"type": "delta", "E0": 1e-3, "dir": (0.0, 0.0, 1.0)}
    dev = ctx["dev"]

    def fresh():
        y = np.zeros((1, 2, n + 1)); y[0, 0, 0] = 1.0
        return torch.from_numpy(y).to(dev)
    ya, la = fresh(), torch.zeros((12, 1, 3), dtype=torch.float64, device=dev)
    h.rttda_propagate(ya, [f], 0.0, 0.05, 12, la)
    yb, lb = fresh(), torch.zeros((12, 1, 3), dtype=torch.float64, device=dev)
    h.rttda_propagate(yb, [f], 0.0, 0.05, 5, lb[:5])
    h.rttda_propagate(yb, [dict(f, **{"continue": True})], 0.25, 0.05, 7, lb[5:])
    yc = fresh()
    h.rttda_propagate(yc, [f], 0.0, 0.05, 5, None)
    h.rttda_propagate(yc, [f], 0.25, 0.05, 7, None)                 # kicks a second time
    torch.cuda.synchronize()
    assert np.max(np.abs(ya.cpu().numpy() - yb.cpu().numpy())) < 1e-14
    assert np.max(np.abs(la.cpu().numpy() - lb.cpu().numpy())) < 1e-14
    assert np.max(np.abs(ya.cpu().numpy() - yc.cpu().numpy())) > 1e-5
    import paper_2601_16949_b200 as R
    h2 = _handle(setup_config(1), 1.0, 1e-12)
    with pytest.raises(R.RttdaError):                                # nothing to continue on a fresh handle
        h2.rttda_propagate(fresh(), [dict(f, **{"continue": True})], 0.0, 0.05, 1, None)
    h2.close()


@pytest.mark.parametrize("nvec", [16, 32])
def test_fock_config2_wide_batches_vs_oracle_jk(nvec):
    """Wide density batches (two and four 8-density chunks of the exchange digestion, several Coulomb chunks) on the
    200-AO molecule, where the a-lists are walked over several batches: every Fock element against the oracle's
    matrix-free J and K at tau_oracle = 1e-20."""
    ctx = setup_config(2)
    N = ctx["basis"].nao
    T = np.random.default_rng(160 + nvec).standard_normal((nvec, N, N))
    J, K, _, _ = ctx["ob"].jk(T, tau=1e-20)
    F = gpu_fock(ctx, T)
    assert rel_inf(F, 2.0 * J - K) < SIGMA_TOL


def test_two_primitive_shells_and_counts():
    """2-primitive shells (carried internally as 3 primitives with a zero coefficient): Fock matrix and sigma against
    the oracle, and the R14 counters report the primitive quartets of the basis AS GIVEN."""
    import torch
    import paper_2601_16949_b200 as R
    from workloads import Basis
    from workloads.molecules import orthonormalizer
    from oracle.integrals import OracleBasis
    rng = np.random.default_rng(222)
    centers = rng.uniform(0.0, 5.0, size=(4, 3))
    spec = [(0, 2), (0, 1), (1, 2), (0, 3), (1, 1)]
    sh_center, sh_l, sh_nprim, exps, coefs = [], [], [], [], []
    for c in range(4):
        for l, npr in spec[: 3 + c % 3]:
            sh_center.append(c); sh_l.append(l); sh_nprim.append(npr)
            exps.extend(np.exp(rng.uniform(np.log(0.2), np.log(6.0), size=npr)).tolist())
            coefs.extend(rng.uniform(0.2, 1.0, size=npr).tolist())
    sh_nprim = np.asarray(sh_nprim, dtype=np.int32)
    basis = Basis(np.ascontiguousarray(centers), np.asarray(sh_center, dtype=np.int32), np.asarray(sh_l, dtype=np.int32),
                  sh_nprim, np.concatenate([[0], np.cumsum(sh_nprim)[:-1]]).astype(np.int32), np.asarray(exps), np.asarray(coefs))
    ob = OracleBasis(basis)
    N = basis.nao
    S = ob.overlap()
    assert np.max(np.abs(R.rttda_overlap(basis) - S)) < 1e-13
    X12, _ = orthonormalizer(S)
    Q, _ = np.linalg.qr(rng.standard_normal((N, N)))
    C = X12 @ Q
    nocc = N // 3
    eps = np.concatenate([np.sort(rng.uniform(-1.0, -0.3, nocc)), np.sort(rng.uniform(0.05, 2.0, N - nocc))])
    dev = torch.device("cuda:0")
    tau = 1e-9
    h = R.Rttda(basis, torch.from_numpy(np.ascontiguousarray(C[:, :nocc])).to(dev),
                torch.from_numpy(np.ascontiguousarray(C[:, nocc:])).to(dev), eps, 1.0, tau)
    T = rng.standard_normal((3, N, N))
    J, K, nq, npq = ob.jk(T, tau=tau)
    Td = torch.from_numpy(T).to(dev)
    F = torch.empty_like(Td)
    h.rttda_fock(Td, F)
    torch.cuda.synchronize()
    J0, K0, _, _ = ob.jk(T, tau=0.0)
    assert rel_inf(F.cpu().numpy(), 2 * J - K) < 1e-12
    assert int(h.rttda_get_info("nquartets")) == nq and int(h.rttda_get_info("nprim_quartets")) == npq
    h.close()


@pytest.mark.parametrize("shape", [(1, 1, 1, 1), (7, 5, 3, 2), (64, 64, 16, 1), (65, 63, 17, 3), (130, 200, 77, 2), (400, 880, 1280, 1)])
def test_gemm_f64_vs_numpy_ragged_strided_batched(shape):
    """The DMMA GEMM on its own (steps a1, a5, a6): ragged M, N, K (not multiples of the 64 x 64 x 16 tile), both operand
    orientations (k-fastest and m/n-fastest strides), beta in {0, 1}, alpha != 1, batch > 1, and a strided
    (interleaved) output like the one the MO->AO epilogue writes."""
    import torch
    from paper_2601_16949_b200 import binding
    M, N, K, batch = shape
    rng = np.random.default_rng(M * 1000 + N)
    dev = torch.device("cuda:0")
    for a_kfast in (True, False):
        for b_kfast in (True, False):
            for beta in (0.0, 1.0):
                A = rng.standard_normal((batch, M, K) if a_kfast else (batch, K, M))
                B = rng.standard_normal((batch, N, K) if b_kfast else (batch, K, N))
                C0 = rng.standard_normal((M, N, batch))                       # interleaved: batch index fastest
                Am = A if a_kfast else np.transpose(A, (0, 2, 1))
                Bm = np.transpose(B, (0, 2, 1)) if b_kfast else B
                ref = -1.7 * np.einsum("bmk,bkn->mnb", Am, Bm) + beta * C0
                Ad, Bd, Cd = (torch.from_numpy(np.ascontiguousarray(x)).to(dev) for x in (A, B, C0))
                sa = (K, 1, M * K) if a_kfast else (1, M, M * K)
                sb = (1, K, N * K) if b_kfast else (N, 1, N * K)
                binding.rttda_gemm_f64(M, N, K, batch, -1.7, Ad, sa, Bd, sb, beta, Cd, (N * batch, batch, 1))
                torch.cuda.synchronize()
                scale = max(1.0, float(np.max(np.abs(ref))))
                assert np.max(np.abs(Cd.cpu().numpy() - ref)) / scale < 1e-13 * max(1, K) ** 0.5


@pytest.mark.parametrize("k,nblock", [(1, 1), (4, 4), (5, 8)])
def test_eigs_block_davidson_tiny_vs_eigh(k, nblock):
    """rttda_eigs (NEXT-3, eq. 2): lowest k eigenpairs of A through multi-vector sigma builds against eigh of the
    oracle's dense A: eigenvalues, residual of the returned vectors under the ORACLE's A, orthonormality."""
    import torch
    ctx = setup_config(1, dense=True)
    A, h = ctx["A"], ctx["h"]
    n = A.shape[0]
    w = np.linalg.eigvalsh(A)
    X = torch.zeros((k, n), dtype=torch.float64, device=ctx["dev"])
    om, rs, it, ns = h.rttda_eigs(k, X, nblock, tol=1e-9, maxiter=100)
    Xh = X.cpu().numpy()
    assert np.max(np.abs(om - w[:k])) < 1e-9
    assert np.max(np.linalg.norm(Xh @ A.T - om[:, None] * Xh, axis=1)) < 2e-9 and np.max(rs) <= 1e-9
    assert np.max(np.abs(Xh @ Xh.T - np.eye(k))) < 1e-10
    assert ns <= it * max(nblock, k)


def test_eigs_config2_lowest_states_and_populations():
    """Config 2 (6400 singles): the four lowest TI-TDA states from rttda_eigs (block of 8, one sigma build of up to 8
    vectors per iteration) against the oracle's block Davidson on its dense A; the vectors feed rttda_populations."""
    import torch
    from oracle import tda
    ctx = setup_config(2, dense=True)
    A, h, cfg = ctx["A"], ctx["h"], ctx["cfg"]
    n = A.shape[0]
    diag = (ctx["eps"][cfg.nocc:][None, :] - ctx["eps"][:cfg.nocc][:, None]).reshape(-1)
    om_ref, X_ref, rn_ref, _ = tda.davidson(lambda V: V @ A.T, diag, 4, 8, tol=1e-9)
    X = torch.zeros((4, n), dtype=torch.float64, device=ctx["dev"])
    om, rs, it, ns = h.rttda_eigs(4, X, 8, tol=1e-8, maxiter=100)
    Xh = X.cpu().numpy()
    assert np.max(np.abs(om - om_ref)) < 1e-8
    assert np.max(np.linalg.norm(Xh @ A.T - om[:, None] * Xh, axis=1)) < 5e-8
    Xs = np.zeros((5, n + 1)); Xs[0, 0] = 1.0; Xs[1:, 1:] = Xh
    y = np.zeros((1, 2, n + 1)); y[0, 0, 1:] = Xh[2]                # the third excited state itself
    P = torch.zeros((1, 5), dtype=torch.float64, device=ctx["dev"])
    h.rttda_populations(torch.from_numpy(y).to(ctx["dev"]), torch.from_numpy(Xs).to(ctx["dev"]), P)
    torch.cuda.synchronize()
    assert np.max(np.abs(P.cpu().numpy()[0] - np.array([0.0, 0.0, 0.0, 1.0, 0.0]))) < 1e-9


@pytest.mark.parametrize("cx,cx_lr,omega", [(0.19, 0.46, 0.33), (0.0, 1.0, 0.5), (1.0, 0.3, 2.0)])
def test_range_separated_exchange_tiny_dense_and_config2(cx, cx_lr, omega):
    """NEXT-4: A with the long-range exchange term - c_x^LR (ij|erf(omega r12)/r12|ab) (RTTDA_OPT_CX_LR / _RS_OMEGA: a
    second ERI pass with attenuated integrals) against the oracle's dense A on config 1 and its matrix-free route on
    config 2; switching the option off again restores the plain operator."""
    import paper_2601_16949_b200 as R
    from workloads import make_vectors
    from oracle import tda
    ctx = setup_config(1, dense=True)
    ob = ctx["ob"]
    A = tda.build_A_rs(ob.eri_tensor(), ob.eri_tensor_erf(omega), ctx["C_o"], ctx["C_v"], ctx["eps"], cx, cx_lr)
    X = make_vectors(ctx["cfg"], 5)
    h = _handle(ctx, cx, 1e-12)
    plain = _sigma(h, X, ctx["dev"])
    h.rttda_set_option(R.OPT_CX_LR, cx_lr)
    h.rttda_set_option(R.OPT_RS_OMEGA, omega)
    assert rel_inf(_sigma(h, X, ctx["dev"]), tda.sigma_dense(A, X)) < 1e-12
    h.rttda_set_option(R.OPT_CX_LR, 0.0)
    assert np.array_equal(_sigma(h, X, ctx["dev"]), plain) or rel_inf(_sigma(h, X, ctx["dev"]), plain) < 1e-14
    h.close()
    ctx2 = setup_config(2)
    X = make_vectors(ctx2["cfg"], 6)
    ref, _, _ = tda.sigma_matrix_free_rs(ctx2["ob"], X, ctx2["C_o"], ctx2["C_v"], ctx2["eps"], cx, cx_lr, omega, tau=1e-20)
    h = _handle(ctx2, cx, 1e-12)
    h.rttda_set_option(R.OPT_CX_LR, cx_lr)
    h.rttda_set_option(R.OPT_RS_OMEGA, omega)
    got = _sigma(h, X, ctx2["dev"])
    h.close()
    assert rel_inf(got, ref) < SIGMA_TOL
