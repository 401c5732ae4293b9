"""Pins for oracle/tda.py: A, the CSF dipole matrix, RK4, kick, spectrum, the paper's Rabi value."""
import os

import numpy as np
import pytest

from oracle import tda
from oracle.integrals import OracleBasis, primitive_eri, primitive_norm
from workloads import Basis, make_vectors

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


def paper_values():
    out = {}
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if len(line) >= 2:
            out[line[0]] = float(line[1])
    return out


AU_TIME_FS = 2.4188843265857e-2     # CODATA, 1 au of time in fs
HARTREE_EV = 27.211386245988
H_EV_S = 4.135667696e-15            # Planck constant in eV s
I_AU_WCM2 = 3.50944758e16           # intensity of a 1 au field amplitude, W/cm^2


# ------------------------------------------------------------------------------------ A
def test_A_symmetric_and_psd_blocks(tiny):
    A = tiny["A"]
    assert np.max(np.abs(A - A.T)) < 1e-13
    ovov, oovv = tda.mo_eri_blocks(tiny["eri"], tiny["C_o"], tiny["C_v"])
    n = A.shape[0]
    assert np.linalg.eigvalsh(ovov.reshape(n, n))[0] > -1e-12            # x^T (ia|jb) x = (rho|rho) >= 0
    assert np.linalg.eigvalsh(oovv.transpose(0, 2, 1, 3).reshape(n, n))[0] > -1e-12
    x, y = make_vectors(tiny["cfg"], 2)
    assert abs(x @ A @ y - y @ A @ x) < 1e-14


def test_A_affine_in_cx(tiny):
    args = (tiny["eri"], tiny["C_o"], tiny["C_v"], tiny["eps"])
    A0, A1, A2 = tda.build_A(*args, 0.0), tda.build_A(*args, 1.0), tda.build_A(*args, 2.0)
    assert np.max(np.abs(A2 - 2 * A1 + A0)) < 1e-13


def test_A_1x1_closed_form():
    """2 centres, one s primitive each, nocc = nvirt = 1: A = eps_a - eps_i + 2(ia|ia) - (ii|aa),
    with every AO integral from the independent (ss|ss) closed form."""
    from scipy.special import erf
    R, a, b = 1.4, 0.9, 0.5
    ctr = np.array([[0, 0, 0], [0, 0, R]], dtype=float)
    basis = Basis(ctr, np.array([0, 1], dtype=np.int32), np.zeros(2, dtype=np.int32),
                  np.ones(2, dtype=np.int32), np.array([0, 1], dtype=np.int32),
                  np.array([a, b]), np.ones(2))
    ob = OracleBasis(basis)
    ex, nrm = np.array([a, b]), primitive_norm(np.array([a, b]), 0)

    def F0(T):
        return 1.0 if T < 1e-14 else 0.5 * np.sqrt(np.pi / T) * erf(np.sqrt(T))

    def ssss(i, j, k, l):
        p, q = ex[i] + ex[j], ex[k] + ex[l]
        P = (ex[i] * ctr[i] + ex[j] * ctr[j]) / p
        Qc = (ex[k] * ctr[k] + ex[l] * ctr[l]) / q
        Kab = np.exp(-ex[i] * ex[j] / p * np.sum((ctr[i] - ctr[j]) ** 2))
        Kcd = np.exp(-ex[k] * ex[l] / q * np.sum((ctr[k] - ctr[l]) ** 2))
        return (2 * np.pi ** 2.5 / (p * q * np.sqrt(p + q)) * Kab * Kcd
                * F0(p * q / (p + q) * np.sum((P - Qc) ** 2)) * nrm[i] * nrm[j] * nrm[k] * nrm[l])

    eri = np.array([[[[ssss(i, j, k, l) for l in range(2)] for k in range(2)] for j in range(2)]
                    for i in range(2)])
    s = (np.pi / (a + b)) ** 1.5 * np.exp(-a * b / (a + b) * R * R) * nrm[0] * nrm[1]
    co = np.array([1.0, 1.0]) / np.sqrt(2 + 2 * s)                    # bonding / antibonding MOs
    cv = np.array([1.0, -1.0]) / np.sqrt(2 - 2 * s)
    iaia = np.einsum("mnls,m,n,l,s->", eri, co, cv, co, cv)
    iiaa = np.einsum("mnls,m,n,l,s->", eri, co, co, cv, cv)
    eps = np.array([-0.5, 0.4])
    A = tda.build_A(ob.eri_tensor(), co[:, None], cv[:, None], eps, 1.0)
    assert abs(A[0, 0] - (0.9 + 2 * iaia - iiaa)) < 1e-14


def test_sigma_matrix_free_equals_dense(tiny):
    X = make_vectors(tiny["cfg"], 4)
    s_d = tda.sigma_dense(tiny["A"], X)
    s_m, nq, npq = tda.sigma_matrix_free(tiny["ob"], X, tiny["C_o"], tiny["C_v"], tiny["eps"], 1.0)
    assert np.max(np.abs(s_d - s_m)) / np.max(np.abs(s_d)) < 1e-13
    s_t, nq2, _ = tda.sigma_matrix_free(tiny["ob"], X, tiny["C_o"], tiny["C_v"], tiny["eps"], 1.0, tau=1e-12)
    assert nq2 <= nq and np.max(np.abs(s_t - s_d)) / np.max(np.abs(s_d)) < 1e-10


# ------------------------------------------------------------------------------------ M (eq. 19)
def test_M_explicit_equals_matrix_free(tiny):
    d = np.array([0.3, -0.5, 0.8]); d /= np.linalg.norm(d)
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(tiny["D"], tiny["C_o"], tiny["C_v"], d)
    M = tda.build_M_explicit(Doo, Dvv, Dov, D00)
    assert np.max(np.abs(M - M.T)) < 1e-14
    rng = np.random.default_rng(1)
    y = rng.standard_normal(M.shape[0]) + 1j * rng.standard_normal(M.shape[0])
    assert np.max(np.abs(M @ y - tda.apply_M(y, Doo, Dvv, Dov, D00))) < 1e-13
    # R6: the dipole origin is the electronic centroid of the ground state, so M does not depend on where the AO
    # dipole integrals were taken from (a bare origin shift c would add the multiple -2 nocc (c.d) of the identity),
    # and the ground-state element D_00 vanishes
    c = np.array([1.0, 2.0, -0.5])
    Doo2, Dvv2, Dov2, D002 = tda.mo_dipoles(tiny["ob"].dipole(c), tiny["C_o"], tiny["C_v"], d)
    M2 = tda.build_M_explicit(Doo2, Dvv2, Dov2, D002)
    assert np.max(np.abs(M2 - M)) < 1e-11
    assert abs(D00) < 1e-12 and abs(M[0, 0]) < 1e-12
    # the shifted one-electron matrices are those of the operator (r - centroid).d
    Dd = np.einsum("k,kmn->mn", d, tiny["D"])
    cen = np.trace(tiny["C_o"].T @ Dd @ tiny["C_o"]) / tiny["C_o"].shape[1]
    assert np.max(np.abs(Doo - tiny["C_o"].T @ (Dd - cen * tiny["S"]) @ tiny["C_o"])) < 1e-11
    assert np.max(np.abs(Dvv - tiny["C_v"].T @ (Dd - cen * tiny["S"]) @ tiny["C_v"])) < 1e-11
    assert np.max(np.abs(Dov - tiny["C_o"].T @ (Dd - cen * tiny["S"]) @ tiny["C_v"])) < 1e-11


def test_M_is_slater_condon_of_one_electron_operator():
    """Independent check of the rules incl. the sqrt(2) (19b) and D_00 = 2 tr D_oo (R3): build singlet
    CSFs as explicit spin-orbital determinant combinations for 2 occupied + 2 virtual orbitals and
    evaluate <Phi|sum_i d(i)|Phi'> by brute force over determinants."""
    import itertools
    no, nv = 2, 2
    n = no + nv
    rng = np.random.default_rng(4)
    d = rng.standard_normal((n, n)); d = d + d.T                         # spatial one-electron matrix
    nso = 2 * n                                                           # spin orbital = 2*p + spin

    def det_element(bra, ket):
        """<bra| sum_i h(i) |ket> for ordered occupation tuples of spin orbitals (Slater-Condon
        rules by explicit sign-counting through second quantisation)."""
        tot = 0.0
        for p in range(nso):
            for q in range(nso):
                if p % 2 != q % 2:
                    continue
                h = d[p // 2, q // 2]
                if q not in ket:
                    continue
                lst = list(ket)
                sgn = (-1) ** lst.index(q)
                lst.remove(q)
                if p in lst:
                    continue
                pos = sum(1 for x in lst if x < p)
                sgn *= (-1) ** pos
                lst.insert(pos, p)
                if tuple(lst) == tuple(bra):
                    tot += sgn * h
        return tot

    ground = tuple(range(2 * no))

    def excite(i, a, spin):                                               # a^+_{a s} a_{i s} |0>, sorted
        lst = list(ground)
        k = lst.index(2 * i + spin)
        sgn = (-1) ** k
        lst.remove(2 * i + spin)
        new = 2 * (no + a) + spin
        pos = sum(1 for x in lst if x < new)
        sgn *= (-1) ** pos
        lst.insert(pos, new)
        return sgn, tuple(lst)

    states = [[(1.0, ground)]]
    for i in range(no):
        for a in range(nv):
            sa, da = excite(i, a, 0)
            sb, db = excite(i, a, 1)
            states.append([(sa / np.sqrt(2), da), (sb / np.sqrt(2), db)])
    dim = len(states)
    Mref = np.zeros((dim, dim))
    for I in range(dim):
        for Jx in range(dim):
            Mref[I, Jx] = sum(ci * cj * det_element(bi, bj) for ci, bi in states[I] for cj, bj in states[Jx])
    Doo, Dvv, Dov = d[:no, :no], d[no:, no:], d[:no, no:]
    M = tda.build_M_explicit(Doo, Dvv, Dov, 2 * np.trace(Doo))
    assert np.max(np.abs(M - Mref)) < 1e-13


# ------------------------------------------------------------------------------------ RK4
def _g(z):
    return 1 - 1j * z - z ** 2 / 2 + 1j * z ** 3 / 6 + z ** 4 / 24


def test_rk4_field_free_eigenvector_closed_form(tiny):
    A = tiny["A"]
    w, U = np.linalg.eigh(A)
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(tiny["D"], tiny["C_o"], tiny["C_v"], (0, 0, 1.0))
    dt, n = 0.1, 25
    for I in (0, 7, len(w) - 1):
        y0 = np.zeros(A.shape[0] + 1, dtype=complex); y0[1:] = U[:, I]
        y, log = tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, {"type": "none"}, 0.0, dt, n)
        z = w[I] * dt
        assert np.max(np.abs(y[1:] - _g(z) ** n * U[:, I])) < 1e-13
        # norm drift law |g|^2 - 1 = -z^6/72 + z^8/576
        assert abs(log[0, 0] - (1 - z ** 6 / 72 + z ** 8 / 576)) < 1e-14
        assert abs(log[-1, 1] + 1j * log[-1, 2] - _g(z) ** n) < 1e-13


def test_rk4_ground_state_stationary_and_order(tiny):
    A = tiny["A"]
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(tiny["D"], tiny["C_o"], tiny["C_v"], (0, 0, 1.0))
    y0 = np.zeros(A.shape[0] + 1, dtype=complex); y0[0] = 1.0
    y, _ = tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, {"type": "none"}, 0.0, 0.05, 10)
    assert np.array_equal(y, y0)                                  # zero field: e_0 stays exactly
    # with a cw field: halving dt divides the error against a much finer run by ~16
    f = {"type": "cw", "E0": 0.05, "omega": 0.3}
    ref, _ = tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, f, 0.0, 0.0125, 160)
    e1 = np.max(np.abs(tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, f, 0.0, 0.1, 20)[0] - ref))
    e2 = np.max(np.abs(tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, f, 0.0, 0.05, 40)[0] - ref))
    assert 12 < e1 / e2 < 20


def test_rk4_against_matrix_exponential(tiny):
    from scipy.linalg import expm
    A = tiny["A"]
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(tiny["D"], tiny["C_o"], tiny["C_v"], (0, 0, 1.0))
    rng = np.random.default_rng(9)
    y0 = rng.standard_normal(A.shape[0] + 1) + 1j * rng.standard_normal(A.shape[0] + 1)
    y0 /= np.linalg.norm(y0)
    y, _ = tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, {"type": "none"}, 0.0, 0.01, 100)
    ref = expm(-1j * tda.extend_A(A) * 1.0) @ y0
    assert np.max(np.abs(y - ref)) < 5e-9        # local error (w dt)^5/120 per step, w <= ~3.5


def test_matrix_free_propagation_equals_dense(tiny):
    A, cfg = tiny["A"], tiny["cfg"]
    f = dict(cfg.fields[0])
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(tiny["D"], tiny["C_o"], tiny["C_v"], f["dir"])
    y0 = np.zeros(A.shape[0] + 1, dtype=complex); y0[0] = 1.0
    yd, ld = tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, f, 0.0, cfg.dt, 3)
    ym, lm = tda.rk4_matrix_free(tiny["ob"], tiny["C_o"], tiny["C_v"], tiny["eps"], 1.0, 0.0, None,
                                 Doo, Dvv, Dov, D00, y0, f, 0.0, cfg.dt, 3)
    assert np.max(np.abs(yd - ym)) < 1e-14 and np.max(np.abs(ld - lm)) < 1e-14


# ------------------------------------------------------------------------------------ SSO (NEXT-1, reading R22)
def test_sso_field_free_eigenvector_is_the_leapfrog_map(tiny):
    """For H u = w u one SSO step acts on the (q, p) coefficients of u as the 2x2 leapfrog matrix
    [[1 - z^2/2, z], [-z (1 - z^2/4), 1 - z^2/2]], z = w dt, of determinant 1: n steps = its n-th power."""
    A = tiny["A"]
    w, U = np.linalg.eigh(A)
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(tiny["D"], tiny["C_o"], tiny["C_v"], (0, 0, 1.0))
    dt, n = 0.1, 40
    for I in (0, 5, len(w) - 1):
        y0 = np.zeros(A.shape[0] + 1, dtype=complex); y0[1:] = (0.8 - 0.6j) * U[:, I]
        y, log = tda.sso_dense(A, Doo, Dvv, Dov, D00, y0, {"type": "none"}, 0.0, dt, n)
        z = w[I] * dt
        M = np.array([[1 - z * z / 2, z], [-z * (1 - z * z / 4), 1 - z * z / 2]])
        assert abs(np.linalg.det(M) - 1.0) < 1e-14
        qn, pn = np.linalg.matrix_power(M, n) @ np.array([0.8, -0.6])
        assert np.max(np.abs(y[1:] - (qn + 1j * pn) * U[:, I])) < 1e-12
        assert abs(log[-1, 0] - (qn * qn + pn * pn)) < 1e-12


def test_sso_second_order_stationary_ground_state_and_bounded_norm(tiny):
    from scipy.linalg import expm
    A = tiny["A"]
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(tiny["D"], tiny["C_o"], tiny["C_v"], (0, 0, 1.0))
    y0 = np.zeros(A.shape[0] + 1, dtype=complex); y0[0] = 1.0
    y, _ = tda.sso_dense(A, Doo, Dvv, Dov, D00, y0, {"type": "none"}, 0.0, 0.05, 10)
    assert np.array_equal(y, y0)                                  # zero field: e_0 stays exactly
    rng = np.random.default_rng(11)
    y1 = rng.standard_normal(A.shape[0] + 1) + 1j * rng.standard_normal(A.shape[0] + 1)
    y1 /= np.linalg.norm(y1)
    ref = expm(-1j * tda.extend_A(A) * 1.0) @ y1
    e1 = np.max(np.abs(tda.sso_dense(A, Doo, Dvv, Dov, D00, y1, {"type": "none"}, 0.0, 0.02, 50)[0] - ref))
    e2 = np.max(np.abs(tda.sso_dense(A, Doo, Dvv, Dov, D00, y1, {"type": "none"}, 0.0, 0.01, 100)[0] - ref))
    assert 3.5 < e1 / e2 < 4.5                                    # second order (slope 2)
    _, log = tda.sso_dense(A, Doo, Dvv, Dov, D00, y1, {"type": "none"}, 0.0, 0.05, 400)
    assert np.max(np.abs(log[:, 0] - 1.0)) < 0.02                 # symplectic: the norm error stays bounded
    # driven: converges to the RK4 result of a much finer step, again with ratio 4
    f = {"type": "cw", "E0": 0.05, "omega": 0.3}
    fine, _ = tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, f, 0.0, 0.0125, 160)
    d1 = np.max(np.abs(tda.sso_dense(A, Doo, Dvv, Dov, D00, y0, f, 0.0, 0.05, 40)[0] - fine))
    d2 = np.max(np.abs(tda.sso_dense(A, Doo, Dvv, Dov, D00, y0, f, 0.0, 0.025, 80)[0] - fine))
    assert 3.5 < d1 / d2 < 4.5


# ------------------------------------------------------------------------------------ populations (eq. 22)
def test_populations_completeness_and_stationary_states(tiny):
    A = tiny["A"]
    w, U = np.linalg.eigh(A)
    n = A.shape[0]
    Xs = np.zeros((n + 1, n + 1)); Xs[0, 0] = 1.0; Xs[1:, 1:] = U.T        # ground state + all TI-TDA states
    rng = np.random.default_rng(3)
    y = rng.standard_normal(n + 1) + 1j * rng.standard_normal(n + 1)
    P = tda.populations(Xs, y)
    assert abs(P.sum() - np.vdot(y, y).real) < 1e-12                       # Parseval over a complete basis
    assert abs(P[0] - abs(y[0]) ** 2) < 1e-15
    # a stationary state keeps population 1 (up to the RK4 norm drift) under field-free propagation
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(tiny["D"], tiny["C_o"], tiny["C_v"], (0, 0, 1.0))
    y0 = np.zeros(n + 1, dtype=complex); y0[1:] = U[:, 3]
    yt, _ = tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, {"type": "none"}, 0.0, 0.05, 50)
    Pt = tda.populations(Xs, yt)
    assert abs(Pt[4] - 1.0) < 1e-7 and np.max(np.delete(Pt, 4)) < 1e-20


# ------------------------------------------------------------------------------------ Lanczos (eq. 2)
def test_lanczos_relation_orthogonality_and_ritz_values(tiny):
    A = tiny["A"]
    n = A.shape[0]
    rng = np.random.default_rng(5)
    v0 = rng.standard_normal(n)
    m = 40
    al, be, V = tda.lanczos(lambda x: A @ x, v0, m)
    T = np.diag(al) + np.diag(be[:-1], 1) + np.diag(be[:-1], -1)
    Vm = V[:m].T
    # Lanczos relation A V_m = V_m T_m + beta_m v_{m+1} e_m^T and orthonormal basis: checks of the recurrence itself
    Rm = A @ Vm - Vm @ T
    Rm[:, -1] -= be[-1] * V[m]
    assert np.max(np.abs(Rm)) < 1e-12
    assert np.max(np.abs(V @ V.T - np.eye(m + 1))) < 1e-12
    # extremal Ritz values converge to the extremal eigenvalues of dense A
    w = np.linalg.eigvalsh(A)
    th = np.linalg.eigvalsh(T)
    assert abs(th[0] - w[0]) < 1e-8 and abs(th[-1] - w[-1]) < 1e-8
    # after n steps the Krylov space is the whole space: all eigenvalues
    al, be, V = tda.lanczos(lambda x: A @ x, v0, n - 1)
    T = np.diag(al) + np.diag(be[:-1], 1) + np.diag(be[:-1], -1)
    assert np.max(np.abs(np.linalg.eigvalsh(T)[[0, -1]] - w[[0, -1]])) < 1e-10


# ------------------------------------------------------------------------------------ paper pins
def test_paper_unit_conversions():
    pv = paper_values()
    assert abs(0.1 * AU_TIME_FS * 1e3 - pv["dt_01_au_in_as"]) < 0.005
    assert abs(3000 * AU_TIME_FS - pv["t_3000_au_in_fs"]) < 0.1
    assert abs(2 * np.pi / 3000 * HARTREE_EV - pv["resolution_ev"]) < 5e-4
    assert abs(pv["rabi_freq_hz"] * H_EV_S - pv["rabi_freq_ev"]) < 0.01         # nu, not omega
    assert abs(pv["freq_2p_hz"] * H_EV_S - pv["freq_2p_ev"]) < 0.001
    assert abs(2 * np.sqrt(2 * np.log(2)) - pv["fwhm_factor"]) < 1e-5


def test_rabi_period_matches_paper_table2():
    """Two-level limit of propagator + field coupling (eq. 16, 18b): resonant cw field,
    mu = 1.5624 au, I = 1e12 W/cm^2  =>  T = 2 pi/(mu E0) = 18.22 fs (Table 2)."""
    pv = paper_values()
    mu = pv["rabi_mu_au"]
    E0 = np.sqrt(pv["rabi_intensity_wcm2"] / I_AU_WCM2)
    w0 = pv["rabi_freq_ev"] / HARTREE_EV
    T_exact_fs = 2 * np.pi / (mu * E0) * AU_TIME_FS
    assert abs(T_exact_fs - pv["rabi_period_exact_1"]) < 0.01
    for k in range(1, 6):
        assert abs(k * T_exact_fs - pv["rabi_period_exact_%d" % k]) < 0.03
    # propagate the 2-level model with the oracle's RK4 through its generic interface
    Amat = np.array([[0.0, 0.0], [0.0, w0]])
    Mmat = np.array([[0.0, mu], [mu, 0.0]])
    dt = pv["rabi_dt_au"]
    nsteps = int(1.05 * 2 * np.pi / (mu * E0) / dt)
    f = {"type": "cw", "E0": E0, "omega": w0}
    y = np.array([1.0, 0.0], dtype=complex)
    pops = np.zeros(nsteps)
    # step one at a time through the same routine to record populations (eq. 22)
    yk, t = y, 0.0
    for n in range(nsteps):
        yk, _ = tda.rk4_propagate(lambda z: Amat @ z, lambda z: Mmat @ z, yk, f, t, dt, 1, log=False)
        t = (n + 1) * dt
        pops[n] = abs(yk[0]) ** 2
    # first full return of the ground-state population after the inversion
    half = np.argmin(pops)
    assert pops[half] < 5e-3                                      # complete inversion
    ret = half + np.argmax(pops[half:])
    T_fs = (ret + 1) * dt * AU_TIME_FS
    assert abs(T_fs - pv["rabi_period_exact_1"]) < 0.1            # paper's RT-TDA: 18.26 vs 18.22
    assert abs(T_fs - pv["rabi_period_rttda_1"]) < 0.1


def test_delta_kick_correlation_closed_form_and_spectrum(tiny):
    """Linear kick + field-free RK4 (R8): R(t_n) = 1 + k^2 D00^2 + 2 k^2 sum_I |d_I|^2 g(w_I dt)^n,
    and the spectrum (eq. 21) peaks at eigenvalues of A within 2 pi/T (Table 1)."""
    A = tiny["A"]
    w, U = np.linalg.eigh(A)
    Doo, Dvv, Dov, D00 = tda.mo_dipoles(tiny["D"], tiny["C_o"], tiny["C_v"], (0, 0, 1.0))
    kappa, dt, n = 1e-4, 0.1, 3000
    y0 = np.zeros(A.shape[0] + 1, dtype=complex); y0[0] = 1.0
    f = {"type": "delta", "E0": kappa}
    # propagate in the eigenbasis through the same generic RK4 (dense A would be the same numbers)
    y, log = tda.rk4_dense(A, Doo, Dvv, Dov, D00, y0, f, 0.0, dt, 200)
    dI = U.T @ Dov.reshape(-1)
    ns = np.arange(1, 201)
    Rref = 1 + kappa ** 2 * D00 ** 2 + 2 * kappa ** 2 * np.sum(
        (dI ** 2)[None, :] * _g(w * dt)[None, :] ** ns[:, None], axis=1)
    R = log[:, 1] + 1j * log[:, 2]
    assert np.max(np.abs(R - Rref)) < 1e-15 + 1e-9 * kappa ** 2
    # spectrum of the closed-form series over a long run: strongest peaks sit at eigenvalues
    ns = np.arange(0, n)
    Rlong = 2 * kappa ** 2 * np.sum((dI ** 2)[None, :] * _g(w * dt)[None, :] ** ns[:, None], axis=1)
    om, inten = tda.spectrum(Rlong, dt)
    res = 2 * np.pi / (n * dt)
    strongest = np.argsort(w * dI ** 2)[::-1][:3]
    sel = (om > 0.02) & (om < w.max() + 0.5)
    om, inten = om[sel], inten[sel]
    peaks = [i for i in range(1, len(om) - 1) if inten[i] > inten[i - 1] and inten[i] > inten[i + 1]]
    peaks = sorted(peaks, key=lambda i: -inten[i])[:6]
    for I in strongest[:2]:
        assert min(abs(om[p] - w[I]) for p in peaks) < res


def test_spectrum_pure_tone_closed_form():
    """eq. 21 with the recipe of P:212 on R(t) = exp(-i w t), w on the padded frequency grid: the mirrored series
    (R(-t) = R(t)^*) is the same pure tone on t = -n dt .. n dt, so the transform at w is the plain sum of the Hann
    window, sum_m (1 - cos(2 pi m / (M - 1))) / 2 = (M - 1) / 2 with M = 2n + 1, and the spectrum there is w (M - 1) / 2.
    A mirror without the conjugate, a transform with the opposite sign, a window over the padded length or a
    padding before the window all change this value."""
    n, pad, dt, j = 50, 99, 0.2, 20
    npad = 2 * n + 1 + pad                                       # 200
    w = 2.0 * np.pi * j / (npad * dt)
    R = np.exp(-1j * w * dt * np.arange(n + 1))
    om, inten = tda.spectrum(R, dt, pad=pad)
    assert om.shape[0] == npad // 2
    assert abs(om[j - 1] - w) < 1e-14 * w
    assert int(np.argmax(inten)) == j - 1
    assert abs(inten[j - 1] - w * n) < 1e-12 * w * n
    # two bins away in units of the UNPADDED resolution the Hann transform has its first zero: 2 * npad / (M - 1)
    # is not an integer here, so instead check the mirror symmetry of the line shape about the peak
    assert np.allclose(inten[j - 1 - 5:j - 1] / om[j - 1 - 5:j - 1],
                       (inten[j:j + 5] / om[j:j + 5])[::-1], rtol=1e-9, atol=1e-12)


# ---------------------------------------------------------------- pulses, eq. 18a-d, config-4 envelope (R9)
def _paper(key):
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_values.txt")
    for line in open(path):
        p = line.split()
        if p and p[0] == key:
            return float(p[1])
    raise KeyError(key)


def test_pulse_tl_half_maximum_at_half_fwhm_and_zero_at_centre():
    """eq. 18c with sigma = FWHM / 2.35482: the Gaussian envelope exp(-(t-t0)^2 / 2 sigma^2) is exactly one half
    at t0 +- FWHM/2 (2.35482 = 2 sqrt(2 ln 2)); with omega = pi / FWHM the carrier sin(omega (t - t0)) is +-1 there, so
    E(t0 +- FWHM/2) = +-E0/2.  A sigma^2 in place of 2 sigma^2, or a carrier not referred to t0, fails this."""
    fwhm, E0, t0 = 12.0, 0.04, 31.0
    f = {"type": "tl", "E0": E0, "omega": np.pi / fwhm, "t0": t0, "sigma": fwhm / _paper("fwhm_factor")}
    assert tda.field_value(f, t0) == 0.0
    assert abs(tda.field_value(f, t0 + fwhm / 2) / (0.5 * E0) - 1.0) < 2e-6      # 2.35482 is printed to 6 digits
    assert abs(tda.field_value(f, t0 - fwhm / 2) / (-0.5 * E0) - 1.0) < 2e-6
    s = f["sigma"]
    assert abs(tda.field_value(f, t0 + 2 * s) / (E0 * np.exp(-2.0) * np.sin(f["omega"] * 2 * s)) - 1.0) < 1e-14


def test_pulse_chirp_zero_crossings_follow_the_linear_chirp():
    """eq. 18d: carrier sin((omega + beta (t-t0)/2)(t-t0)), i.e. phase phi(s) = omega s + beta s^2/2 and instantaneous
    frequency omega + beta s.  The zeros of E are where phi = k pi: s_k = (-omega + sqrt(omega^2 + 2 beta k pi)) / beta.
    A missing factor 1/2, a wrong sign of beta or a chirp referred to t = 0 moves them."""
    E0, w, beta, t0, sig = 0.03, 0.4, 0.05, 20.0, 15.0
    f = {"type": "chirp", "E0": E0, "omega": w, "beta": beta, "t0": t0, "sigma": sig}
    for k in range(1, 8):
        sk = (-w + np.sqrt(w * w + 2.0 * beta * k * np.pi)) / beta
        assert abs(tda.field_value(f, t0 + sk)) < 1e-14 * E0 * 50
        # sign pattern of sin just before / after the k-th zero
        assert np.sign(tda.field_value(f, t0 + sk - 1e-3)) == (-1.0) ** (k - 1)
        assert np.sign(tda.field_value(f, t0 + sk + 1e-3)) == (-1.0) ** k
    # finite-difference instantaneous frequency from consecutive zeros: pi / (s_{k+1} - s_k) ~ omega + beta s_mid
    s5, s6 = [(-w + np.sqrt(w * w + 2.0 * beta * k * np.pi)) / beta for k in (5, 6)]
    assert abs(np.pi / (s6 - s5) - (w + beta * 0.5 * (s5 + s6))) < 1e-3
    # beta = 0 is the transform-limited pulse; envelope as in 18c
    g = dict(f, beta=0.0)
    for t in (3.0, 19.0, 26.5):
        assert tda.field_value(g, t) == tda.field_value(dict(g, type="tl"), t)
    assert abs(abs(tda.field_value(f, t0 + 1.0)) - E0 * np.exp(-1.0 / (2 * sig * sig)) * abs(np.sin((w + 0.5 * beta) * 1.0))) < 1e-16


def test_pulse_sin2_envelope_zeros_peak_and_support():
    """R9 (config 4): E0 sin^2(pi t / T_env) sin(omega t) on [0, T_env]: zero at both ends and outside, envelope 1 at
    T_env/2 (with omega T_env / 2 = 5 pi / 2 the carrier is 1 there), envelope symmetric about T_env/2."""
    E0, Te = 0.05, 200.0
    w = 5.0 * np.pi / Te
    f = {"type": "sin2", "E0": E0, "omega": w, "T_env": Te}
    assert tda.field_value(f, 0.0) == 0.0 and abs(tda.field_value(f, Te)) < 1e-17
    assert tda.field_value(f, -1.0) == 0.0 and tda.field_value(f, Te + 1e-9) == 0.0
    assert abs(tda.field_value(f, Te / 2) - E0) < 1e-15
    for t in (10.0, 37.5, 99.0):
        env_a = tda.field_value(f, t) / np.sin(w * t)
        env_b = tda.field_value(f, Te - t) / np.sin(w * (Te - t))
        assert abs(env_a - env_b) < 1e-15 and abs(env_a - E0 * np.sin(np.pi * t / Te) ** 2) < 1e-16
    assert abs(tda.field_value(f, Te / 4) - E0 * 0.5 * np.sin(w * Te / 4)) < 1e-16     # sin^2(pi/4) = 1/2


def test_pulse_cw_and_delta():
    """eq. 18b: E0 sin(omega t) from t = 0; eq. 18a / R8: the delta pulse has no E(t), it is the linearised kick."""
    f = {"type": "cw", "E0": 0.01, "omega": 0.3}
    assert tda.field_value(f, 0.0) == 0.0 and abs(tda.field_value(f, np.pi / 0.6) - 0.01) < 1e-17
    assert tda.field_value({"type": "delta", "E0": 1e-4}, 0.0) == 0.0
    y0 = np.zeros(5, dtype=complex); y0[0] = 1.0
    M = np.arange(25.0).reshape(5, 5); M = M + M.T
    y = tda.kick(y0, {"type": "delta", "E0": 1e-4}, lambda z: M @ z)
    assert np.array_equal(y.real, y0.real) and np.allclose(y.imag, -1e-4 * M[:, 0], rtol=0, atol=1e-20)   # only p(0+) changes


# ---------------------------------------------------------------- noise floor of the FP64 oracle route
def test_fp64_route_noise_floor_against_long_double_route(tiny):
    """sigma through the FP64 J/K route against the extended-precision route (long double densities, sums and MO
    transforms, FP64 integral values): their difference IS the rounding floor of the FP64 oracle.  Config 1 here;
    config 2 (cond(S) = 132): 9e-15, recorded from _work runs; config 4 from the two stored sample files below."""
    X = make_vectors(tiny["cfg"], 3)
    s64, nq, _ = tda.sigma_matrix_free(tiny["ob"], X, tiny["C_o"], tiny["C_v"], tiny["eps"], 1.0, tau=0.0)
    sld, nq2, _ = tda.sigma_matrix_free_ld(tiny["ob"], X, tiny["C_o"], tiny["C_v"], tiny["eps"], 1.0, tau=0.0)
    assert nq == nq2 and sld.dtype == np.longdouble
    floor = np.max(np.abs(s64 - sld.astype(np.float64))) / np.max(np.abs(s64))
    print("FP64 oracle route vs long double route, config 1: %.2e" % floor)
    assert floor < 1e-13
    # and the extended route agrees with the dense-A definition
    assert np.max(np.abs(sld.astype(np.float64) - tda.sigma_dense(tiny["A"], X))) / np.max(np.abs(s64)) < 1e-13
    # cx enters linearly in both routes
    a, _, _ = tda.sigma_matrix_free_ld(tiny["ob"], X, tiny["C_o"], tiny["C_v"], tiny["eps"], 0.25, tau=0.0)
    b, _, _ = tda.sigma_matrix_free(tiny["ob"], X, tiny["C_o"], tiny["C_v"], tiny["eps"], 0.25, tau=0.0)
    assert np.max(np.abs(a.astype(np.float64) - b)) / np.max(np.abs(b)) < 1e-13


def _read_samples(name):
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    if not os.path.exists(path):
        return None, None
    norm, samples = {}, {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        p = line.split()
        if p[0] == "norm":
            norm[int(p[1])] = float(p[2])
        else:
            samples[(int(p[0]), int(p[1]))] = float(p[2])
    return norm, samples


def test_config4_stored_samples_fp64_route_vs_long_double_route():
    """The two stored oracle sample sets of the 1280-AO molecule (cond(S) = 4.5e4): FP64 accumulation with
    tau_oracle = 1e-15 (round 1) against long double with tau_oracle = 1e-17, same vectors 0 and 1, same positions.
    Their difference is the oracle's own FP64 noise floor at the size where the 1e-10 sigma tolerance is tightest."""
    n_ld, s_ld = _read_samples("config4_sigma_samples.txt")
    n_64, s_64 = _read_samples("config4_sigma_samples_fp64.txt")
    if s_ld is None or s_64 is None:
        pytest.skip("stored config-4 samples not generated")
    common = [k for k in s_64 if k in s_ld]
    assert len(common) >= 400
    d = max(abs(s_64[k] - s_ld[k]) / n_ld[k[0]] for k in common)
    print("config-4 oracle samples, FP64/1e-15 vs long double/1e-17: %.2e of max|sigma|" % d)
    # measured 1.28e-10: the FP64 ROUTE of the oracle is itself outside the 1e-10 sigma tolerance at this size, which is
    # why the stored reference of the GPU parity test is the long-double route (the CUDA path differs from it by 2-4e-11
    # on these two vectors); the bound only guards against a gross change of either file
    assert 1e-12 < d < 1e-9


def test_dense_A_by_pair_blocks_equals_tensor_route(tiny):
    """Route (ii) of SURVEY 8(c5) (AO integrals one ket shell pair at a time, half-transformed at once) against the
    plain four-index transform of the full AO tensor, incl. c_x != 1."""
    for cx in (1.0, 0.3):
        A2 = tda.build_A_by_pair_blocks(tiny["ob"], tiny["C_o"], tiny["C_v"], tiny["eps"], cx)
        A1 = tda.build_A(tiny["eri"], tiny["C_o"], tiny["C_v"], tiny["eps"], cx)
        assert np.max(np.abs(A1 - A2)) < 1e-12
    blk = tiny["ob"].eri_pair_block(4, 2)
    o4, o2 = int(tiny["ob"].ao_off[4]), int(tiny["ob"].ao_off[2])
    assert np.max(np.abs(blk - tiny["eri"][:, :, o4:o4 + blk.shape[2], o2:o2 + blk.shape[3]])) < 1e-15


def test_davidson_lowest_eigenpairs_against_eigh(tiny):
    """Block Davidson of the oracle (NEXT-3; eq. 2) against LAPACK's eigh of the dense A: eigenvalues, residuals,
    orthonormality, and the subspace of the lowest roots."""
    A = tiny["A"]
    n = A.shape[0]
    no, nv = tiny["C_o"].shape[1], tiny["C_v"].shape[1]
    eps = tiny["eps"]
    diag = (eps[no:][None, :] - eps[:no][:, None]).reshape(-1)
    w, U = np.linalg.eigh(A)
    for k, nb in ((1, 1), (4, 4), (6, 9)):
        om, X, rn, it = tda.davidson(lambda V: V @ A.T, diag, k, nb, tol=1e-9)
        assert np.max(np.abs(om - w[:k])) < 1e-10
        assert np.max(rn) <= 1e-9 and np.max(np.abs(X @ A.T - om[:, None] * X)) < 1e-8
        assert np.max(np.abs(X @ X.T - np.eye(k))) < 1e-10
        P = U[:, :k] @ U[:, :k].T                                   # projector on the exact lowest-k subspace
        assert np.max(np.abs(X @ P - X)) < 1e-6
        assert it < 60


def test_range_separated_A_limits_and_matrix_free_route(tiny):
    """A with range-separated exchange (NEXT-4): omega -> infinity turns c_x^LR into ordinary exchange
    (A(c_x, c_x^LR, inf) = A(c_x + c_x^LR)), c_x^LR = 0 changes nothing, the long-range block is symmetric PSD, and the
    matrix-free route equals the dense one."""
    ob, C_o, C_v, eps = tiny["ob"], tiny["C_o"], tiny["C_v"], tiny["eps"]
    e_inf = ob.eri_tensor_erf(1e7)
    A = tda.build_A_rs(tiny["eri"], e_inf, C_o, C_v, eps, 0.19, 0.46)
    assert np.max(np.abs(A - tda.build_A(tiny["eri"], C_o, C_v, eps, 0.65))) < 1e-9
    e = ob.eri_tensor_erf(0.33)
    assert np.array_equal(tda.build_A_rs(tiny["eri"], e, C_o, C_v, eps, 0.4, 0.0), tda.build_A(tiny["eri"], C_o, C_v, eps, 0.4))
    A = tda.build_A_rs(tiny["eri"], e, C_o, C_v, eps, 0.19, 0.46)
    assert np.max(np.abs(A - A.T)) < 1e-13
    Klr = (tda.build_A(tiny["eri"], C_o, C_v, eps, 0.19) - A) / 0.46          # (ij|erf|ab) as a matrix in (ia),(jb)
    assert np.linalg.eigvalsh(0.5 * (Klr + Klr.T))[0] > -1e-12
    X = make_vectors(tiny["cfg"], 3)
    for cx in (0.19, 0.0):
        Ad = tda.build_A_rs(tiny["eri"], e, C_o, C_v, eps, cx, 0.46)
        s, _, _ = tda.sigma_matrix_free_rs(ob, X, C_o, C_v, eps, cx, 0.46, 0.33, tau=0.0)
        assert np.max(np.abs(s - tda.sigma_dense(Ad, X))) < 1e-12
