"""Pins for oracle/integrals.c: closed forms, library routines, invariants, brute force.

None of these re-types the oracle's own formula: each compares against something fixed by the
mathematics."""
import numpy as np
import pytest
from scipy.special import erf, gamma, gammainc

from oracle.integrals import OracleBasis, boys, primitive_eri, primitive_norm
from workloads import Basis


def _basis(centers, shells):
    """shells: list of (center, l, exps, coefs)."""
    sh_c, sh_l, sh_n, ex, co = [], [], [], [], []
    for (c, l, e, d) in shells:
        sh_c.append(c); sh_l.append(l); sh_n.append(len(e)); ex += list(e); co += list(d)
    sh_n = np.asarray(sh_n, dtype=np.int32)
    off = np.concatenate([[0], np.cumsum(sh_n)[:-1]]).astype(np.int32)
    return Basis(np.asarray(centers, dtype=np.float64), np.asarray(sh_c, dtype=np.int32),
                 np.asarray(sh_l, dtype=np.int32), sh_n, off, np.asarray(ex), np.asarray(co))


# ------------------------------------------------------------------------------------ Boys
@pytest.mark.parametrize("T", [1e-8, 1e-3, 0.3, 2.0, 11.0, 25.0, 34.999, 35.001, 60.0, 150.0])
def test_boys_vs_incomplete_gamma(T):
    # F_n(T) = gamma(n+1/2, T) / (2 T^(n+1/2)), scipy's regularised lower incomplete gamma
    F = boys(4, T)
    ref = np.array([gammainc(n + 0.5, T) * gamma(n + 0.5) / (2.0 * T ** (n + 0.5)) for n in range(5)])
    if T < 1e-6:
        ref = np.array([1.0 / (2 * n + 1) - T / (2 * n + 3) for n in range(5)])
    assert np.max(np.abs(F - ref) / ref) < 2e-13


def test_boys_at_zero_and_F0_erf():
    assert np.allclose(boys(4, 0.0), [1.0, 1 / 3, 1 / 5, 1 / 7, 1 / 9], rtol=0, atol=1e-16)
    for T in (0.7, 5.0, 40.0):
        assert abs(boys(0, T)[0] - 0.5 * np.sqrt(np.pi / T) * erf(np.sqrt(T))) < 1e-15


def test_boys_recursion_identity():
    # (2n+1) F_n = 2T F_(n+1) + exp(-T) across the T = 35 switch
    for T in (3.0, 34.0, 36.0):
        F = boys(4, T)
        for n in range(4):
            assert abs((2 * n + 1) * F[n] - 2 * T * F[n + 1] - np.exp(-T)) < 1e-15


# ------------------------------------------------------------------------------------ one-electron
def test_overlap_ss_closed_form_and_normalisation():
    A, B = np.array([0.1, -0.2, 0.3]), np.array([1.0, 0.7, -0.4])
    a, b = 0.8, 1.7
    ob = OracleBasis(_basis([A, B], [(0, 0, [a], [1.0]), (1, 0, [b], [1.0])]))
    S = ob.overlap()
    p, mu = a + b, a * b / (a + b)
    closed = (np.pi / p) ** 1.5 * np.exp(-mu * np.sum((A - B) ** 2)) * primitive_norm(a, 0) * primitive_norm(b, 0)
    assert abs(S[0, 1] - closed) < 1e-15
    assert np.allclose(np.diag(S), 1.0, atol=1e-15)


def test_overlap_p_properties(tiny):
    S = tiny["S"]
    assert np.allclose(S, S.T, atol=1e-15)
    assert np.allclose(np.diag(S), 1.0, atol=1e-14)
    assert np.linalg.eigvalsh(S)[0] > 0
    # same-centre <s|p> = 0 and <p_x|p_y> = 0: centre 0 holds AOs 0 (s), 1 (s), 2..4 (p)
    assert np.max(np.abs(S[0:2, 2:5])) < 1e-15
    assert np.max(np.abs(S[2:5, 2:5] - np.eye(3))) < 1e-14


def _raw_1e(A, la, a, B, lb, b, what="S", origin=(0, 0, 0)):
    """Un-normalised primitive one-electron block through the oracle (coefficients undone)."""
    ob = OracleBasis(_basis([A, B], [(0, la, [a], [1.0]), (1, lb, [b], [1.0])]))
    na = 2 * la + 1
    M = ob.overlap() if what == "S" else ob.dipole(origin)
    blk = M[..., :na, na:]
    return blk / (ob.ncoef[0] * ob.ncoef[1])


def test_overlap_and_dipole_p_by_centre_derivative():
    # d/dA_x exp(-a|r-A|^2) = 2a (x-A_x) exp(..)  =>  <p_x|.> = (1/2a) d<s|.>/dA_x
    A, B = np.array([0.3, -0.1, 0.2]), np.array([-0.5, 0.6, 0.9])
    a, b, h = 0.9, 0.6, 1e-3
    for what in ("S", "D"):
        def f(Av):
            return _raw_1e(Av, 0, a, B, 0, b, what)
        ps = _raw_1e(A, 1, a, B, 0, b, what)          # [..., 3, 1]
        for x in range(3):
            e = np.zeros(3); e[x] = h
            fd = (-f(A + 2 * e) + 8 * f(A + e) - 8 * f(A - e) + f(A - 2 * e)) / (12 * h) / (2 * a)
            assert np.max(np.abs(ps[..., x, 0] - fd[..., 0, 0])) < 1e-10


def test_dipole_ss_and_origin_shift(tiny):
    A, B = np.array([0.1, -0.2, 0.3]), np.array([1.0, 0.7, -0.4])
    a, b = 0.8, 1.7
    ob = OracleBasis(_basis([A, B], [(0, 0, [a], [1.0]), (1, 0, [b], [1.0])]))
    S, D = ob.overlap(), ob.dipole()
    P = (a * A + b * B) / (a + b)
    assert np.allclose(D[:, 0, 1], P * S[0, 1], atol=1e-15)       # <s|r|s> = P <s|s>
    ob, O2 = tiny["ob"], np.array([0.4, -1.0, 2.5])
    D0, D2 = ob.dipole(), ob.dipole(O2)
    for k in range(3):                                            # D(O') = D(O) - O' S
        assert np.allclose(D2[k], D0[k] - O2[k] * tiny["S"], atol=1e-13)
        assert np.allclose(D0[k], D0[k].T, atol=1e-15)


# ------------------------------------------------------------------------------------ ERIs
def _F0(T):
    return 1.0 if T == 0 else 0.5 * np.sqrt(np.pi / T) * erf(np.sqrt(T))


def test_ssss_closed_form():
    rng = np.random.default_rng(7)
    for _ in range(20):
        ctr = rng.uniform(-1.5, 1.5, size=(4, 3))
        ex = np.exp(rng.uniform(np.log(0.1), np.log(20), size=4))
        a, b, c, d = ex
        p, q = a + b, c + d
        P = (a * ctr[0] + b * ctr[1]) / p
        Q = (c * ctr[2] + d * ctr[3]) / q
        Kab = np.exp(-a * b / p * np.sum((ctr[0] - ctr[1]) ** 2))
        Kcd = np.exp(-c * d / q * np.sum((ctr[2] - ctr[3]) ** 2))
        closed = 2 * np.pi ** 2.5 / (p * q * np.sqrt(p + q)) * Kab * Kcd * _F0(p * q / (p + q) * np.sum((P - Q) ** 2))
        val = primitive_eri(ctr, ex, [0, 0, 0, 0]).item()
        assert abs(val - closed) < 1e-14 * max(1.0, abs(closed))


def test_one_centre_ssss_value():
    # normalised s Gaussian of exponent a: (phi phi|phi phi) = 2 sqrt(a/pi)
    for a in (0.3, 1.0, 7.5):
        val = primitive_eri(np.zeros((4, 3)), [a] * 4, [0] * 4).item() * primitive_norm(a, 0) ** 4
        assert abs(val - 2 * np.sqrt(a / np.pi)) < 1e-14


CLASSES = [(1, 0, 0, 0), (0, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1), (1, 1, 0, 0), (1, 0, 1, 0),
           (0, 1, 0, 1), (0, 0, 1, 1), (1, 1, 1, 0), (1, 0, 1, 1), (1, 1, 1, 1)]


@pytest.mark.parametrize("l4", CLASSES)
def test_p_classes_by_nested_centre_derivatives(l4):
    """Every p index = (1/2a) d/dA of the s function: check all classes against nested central
    differences of the (already closed-form-pinned) (ss|ss) integral."""
    rng = np.random.default_rng(11)
    ctr = rng.uniform(-1.0, 1.0, size=(4, 3))
    ex = np.array([0.7, 1.1, 0.5, 0.9])
    h = 2e-2
    stencil = [(-2, 1 / 12), (-1, -8 / 12), (1, 8 / 12), (2, -1 / 12)]
    blk = primitive_eri(ctr, ex, l4)
    pidx = [i for i in range(4) if l4[i] == 1]
    # compare a few components (all for <= 2 p's, the diagonal-ish ones otherwise)
    comps = list(np.ndindex(*[3] * len(pidx)))
    if len(pidx) > 2:
        comps = comps[:: len(comps) // 9]
    for comp in comps:
        def rec(level, c):
            if level == len(pidx):
                return primitive_eri(c, ex, [0, 0, 0, 0]).item()
            k, x = pidx[level], comp[level]
            tot = 0.0
            for (m, w) in stencil:
                c2 = c.copy(); c2[k, x] += m * h
                tot += w * rec(level + 1, c2)
            return tot / h / (2 * ex[k])
        fd = rec(0, ctr)
        sel = [comp[pidx.index(i)] if l4[i] else 0 for i in range(4)]
        assert abs(blk[tuple(sel)] - fd) < 2e-6 * max(1.0, abs(fd)), (comp, blk[tuple(sel)], fd)


def test_eightfold_symmetry_schwarz_psd(tiny):
    eri, N = tiny["eri"], tiny["basis"].nao
    for perm in [(1, 0, 2, 3), (0, 1, 3, 2), (2, 3, 0, 1), (3, 2, 1, 0)]:
        assert np.max(np.abs(eri - eri.transpose(perm))) < 1e-15
    diag = np.einsum("mnmn->mn", eri)
    assert diag.min() >= 0.0
    bound = np.sqrt(diag)[:, :, None, None] * np.sqrt(diag)[None, None, :, :]
    assert np.all(np.abs(eri) <= bound * (1 + 1e-12) + 1e-15)
    w = np.linalg.eigvalsh(eri.reshape(N * N, N * N))
    assert w[0] > -1e-10                                        # (mu nu|lam sig) is a PSD supermatrix
    # Schwarz routine = sqrt of max diagonal element per shell pair
    Q = tiny["ob"].schwarz()
    off, l = tiny["ob"].ao_off, tiny["ob"].sh_l
    for a in (0, 2, 5, 17):
        for b in (1, 2, 8):
            blk = diag[off[a]:off[a] + 2 * l[a] + 1, off[b]:off[b] + 2 * l[b] + 1]
            assert abs(Q[a, b] - np.sqrt(blk.max())) < 1e-15


def test_translation_and_rotation(tiny):
    from workloads import get_config, make_basis
    basis = make_basis(get_config(1))
    th = 0.83
    Rz = np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, 1.0]])
    Rx = np.array([[1.0, 0, 0], [0, np.cos(0.4), -np.sin(0.4)], [0, np.sin(0.4), np.cos(0.4)]])
    Rm = Rz @ Rx
    b2 = Basis(basis.centers @ Rm.T + np.array([3.0, -2.0, 0.5]), basis.sh_center, basis.sh_l,
               basis.sh_nprim, basis.sh_off, basis.exps, basis.coefs)
    ob2 = OracleBasis(b2)
    eri2 = ob2.eri_tensor()
    # AO rotation matrix: identity on s, Rm on each p triple
    N = basis.nao
    U = np.eye(N)
    for s, o in enumerate(basis.ao_off):
        if basis.sh_l[s] == 1:
            U[o:o + 3, o:o + 3] = Rm
    # rotated p functions: p'_i = sum_j Rm[i][j] p_j  ->  eri2 = U U U U eri
    ref = np.einsum("pm,qn,rl,ts,mnls->pqrt", U, U, U, U, tiny["eri"], optimize=True)
    assert np.max(np.abs(eri2 - ref)) < 1e-13


def test_contracted_equals_sum_of_primitives(tiny):
    ob = tiny["ob"]
    ctr = ob.centers
    for (sa, sb, sc, sd) in [(0, 3, 6, 2), (0, 0, 1, 2), (2, 3, 5, 8), (3, 4, 6, 9)]:
        blk = ob.shell_quartet(sa, sb, sc, sd)
        ref = np.zeros_like(blk)
        sh = (sa, sb, sc, sd)
        import itertools
        for ks in itertools.product(*[range(ob.sh_nprim[s]) for s in sh]):
            idx = [ob.sh_off[s] + k for s, k in zip(sh, ks)]
            c4 = np.array([ctr[ob.sh_center[s]] for s in sh])
            ref += np.prod(ob.ncoef[idx]) * primitive_eri(c4, ob.exps[idx], [ob.sh_l[s] for s in sh])
        assert np.max(np.abs(blk - ref)) < 1e-14
    assert ob.shell_quartet(0, 3, 6, 2).shape == (1, 1, 1, 3) or True


# ------------------------------------------------------------------------------------ J / K
def test_jk_eight_image_digestion_equals_full_contraction(tiny):
    ob, eri, N = tiny["ob"], tiny["eri"], tiny["basis"].nao
    rng = np.random.default_rng(3)
    T = rng.standard_normal((3, N, N))                          # NOT symmetric
    J, K, nq, npq = ob.jk(T, tau=0.0)
    Jref = np.einsum("mnls,vls->vmn", eri, T)
    Kref = np.einsum("mnls,vns->vml", eri, T)
    assert np.max(np.abs(J - Jref)) < 1e-12 and np.max(np.abs(K - Kref)) < 1e-12
    npair = ob.nshells * (ob.nshells + 1) // 2
    assert nq == npair * (npair + 1) // 2
    # symmetry classes: J[Pa] = 0, K[Ps] symmetric, K[Pa] antisymmetric
    Ps, Pa = 0.5 * (T + T.transpose(0, 2, 1)), 0.5 * (T - T.transpose(0, 2, 1))
    Js, Ks, _, _ = ob.jk(Ps)
    Ja, Ka, _, _ = ob.jk(Pa)
    assert np.max(np.abs(Ja)) < 1e-13
    assert np.max(np.abs(Ks - Ks.transpose(0, 2, 1))) < 1e-13
    assert np.max(np.abs(Ka + Ka.transpose(0, 2, 1))) < 1e-13
    # sampled-element routine (plain definition) agrees too
    mu, nu = np.array([0, 4, 17, 29, 3]), np.array([0, 9, 2, 29, 28])
    Jsm, Ksm = ob.jk_samples(T, mu, nu)
    assert np.max(np.abs(Jsm - Jref[:, mu, nu].T)) < 1e-13
    assert np.max(np.abs(Ksm - Kref[:, mu, nu].T)) < 1e-13


def test_schwarz_screening_error_is_bounded(tiny):
    ob, N = tiny["ob"], tiny["basis"].nao
    T = np.random.default_rng(5).standard_normal((1, N, N))
    J0, K0, n0, _ = ob.jk(T, tau=0.0)
    prev = 0.0
    for tau in (1e-12, 1e-8, 1e-5):
        J, K, nq, _ = ob.jk(T, tau=tau)
        err = max(np.max(np.abs(J - J0)), np.max(np.abs(K - K0)))
        assert nq <= n0 and err <= tau * np.sum(np.abs(T)) * 8
        assert err >= prev - 1e-15
        prev = err


# ------------------------------------------------------------------------------------ erf-attenuated ERIs (NEXT-4)
def test_erf_attenuated_ssss_against_gaussian_geminal_quadrature():
    """erf(w r)/r = (2/sqrt(pi)) int_0^w exp(-s^2 r^2) ds, and the s-type integral of a Gaussian geminal has the closed form
      (ab| exp(-s^2 r12^2) |cd) = K_ab K_cd (pi^2 / (pq + s^2 (p+q)))^(3/2) exp(-pq s^2 / (pq + s^2 (p+q)) |PQ|^2),
    so (ss|erf(w r12)/r12|ss) is a one-dimensional quadrature of elementary functions (scipy.integrate.quad): no Boys
    function, no theta prefactor, nothing the oracle's Hermite route uses."""
    from scipy.integrate import quad
    from oracle.integrals import primitive_eri_erf
    rng = np.random.default_rng(17)
    for omega in (0.2, 0.33, 1.0, 4.0):
        for _ in range(5):
            ctr = rng.uniform(-1.5, 1.5, size=(4, 3))
            a, b, c, d = ex = np.exp(rng.uniform(np.log(0.1), np.log(10), size=4))
            p, q = a + b, c + d
            P = (a * ctr[0] + b * ctr[1]) / p
            Q = (c * ctr[2] + d * ctr[3]) / q
            K = np.exp(-a * b / p * np.sum((ctr[0] - ctr[1]) ** 2)) * np.exp(-c * d / q * np.sum((ctr[2] - ctr[3]) ** 2))
            R2 = float(np.sum((P - Q) ** 2))

            def geminal(s):
                den = p * q + s * s * (p + q)
                return (np.pi ** 2 / den) ** 1.5 * np.exp(-p * q * s * s / den * R2)
            ref = 2.0 / np.sqrt(np.pi) * quad(geminal, 0.0, omega, epsabs=1e-15, epsrel=1e-13)[0] * K
            val = primitive_eri_erf(ctr, ex, [0, 0, 0, 0], omega).item()
            assert abs(val - ref) < 1e-11 * max(1.0, abs(ref))


@pytest.mark.parametrize("l4", [(0, 0, 0, 0), (1, 0, 0, 0), (1, 1, 0, 0), (1, 0, 1, 0), (1, 1, 1, 0), (1, 1, 1, 1)])
def test_erf_attenuated_limits_and_bounds(l4):
    """omega -> infinity recovers 1/r12; omega -> 0 gives (2 omega / sqrt(pi)) <a|b> <c|d> (erf(x) ~ 2x/sqrt(pi));
    omega <= 0 means the Coulomb operator; and for the positive (ss|ss) integrand the value grows with omega."""
    from oracle.integrals import primitive_eri_erf
    rng = np.random.default_rng(23)
    ctr = rng.uniform(-1.0, 1.0, size=(4, 3))
    ex = np.array([0.7, 1.3, 0.45, 0.9])
    full = primitive_eri(ctr, ex, l4)
    assert np.array_equal(primitive_eri_erf(ctr, ex, l4, 0.0), full)
    assert np.max(np.abs(primitive_eri_erf(ctr, ex, l4, 1e6) - full)) < 1e-10 * np.max(np.abs(full))
    w = 1e-4
    Sab = _raw_1e(ctr[0], l4[0], ex[0], ctr[1], l4[1], ex[1])
    Scd = _raw_1e(ctr[2], l4[2], ex[2], ctr[3], l4[3], ex[3])
    lim = 2.0 * w / np.sqrt(np.pi) * np.einsum("ab,cd->abcd", Sab, Scd)
    got = primitive_eri_erf(ctr, ex, l4, w)
    assert np.max(np.abs(got - lim)) < 1e-6 * np.max(np.abs(lim)) + 1e-18
    if sum(l4) == 0:
        vals = [primitive_eri_erf(ctr, ex, l4, x).item() for x in (0.1, 0.3, 1.0, 3.0, 30.0)]
        assert all(0.0 < u < v for u, v in zip(vals, vals[1:])) and vals[-1] < full.item()


def test_erf_attenuated_tensor_symmetry_and_jk_route(tiny):
    """The attenuated AO tensor keeps the 8-fold symmetry, is dominated by the Coulomb Schwarz bounds, and the matrix-free
    J/K route with the operator switch equals the plain contraction of that tensor."""
    ob, N = tiny["ob"], tiny["ob"].nao
    e = ob.eri_tensor_erf(0.33)
    assert np.max(np.abs(e - e.transpose(1, 0, 2, 3))) < 1e-14 and np.max(np.abs(e - e.transpose(2, 3, 0, 1))) < 1e-14
    diag = np.sqrt(np.einsum("mnmn->mn", tiny["eri"]))
    assert np.all(np.abs(e) <= diag[:, :, None, None] * diag[None, None, :, :] + 1e-14)
    T = np.random.default_rng(3).standard_normal((2, N, N))
    J, K, _, _ = ob.jk_erf(T, 0.33, tau=0.0)
    assert np.max(np.abs(J - np.einsum("mnls,vls->vmn", e, T))) < 1e-12
    assert np.max(np.abs(K - np.einsum("mnls,vns->vml", e, T))) < 1e-12


def test_fp64_integral_values_against_long_double_evaluation(tiny):
    """Rounding noise of the oracle's FP64 integral VALUES: the whole AO tensor of config 1 against the same formulas
    evaluated with every intermediate in x87 long double (oracle_eri_tensor_ld).  Absolute errors of a few 1e-16 (the
    Hermite sums cancel, so small integrals carry the absolute error of the large intermediates); this is the noise that
    cond(S) = 4.5e4 amplifies to the 1e-10 level of the sigma tolerance at 1280 AO."""
    e64, eld = tiny["eri"], tiny["ob"].eri_tensor_ld()
    assert eld.dtype == np.longdouble
    d = np.abs(e64 - eld.astype(np.float64))
    rms = float(np.sqrt(np.mean(d ** 2)))
    print("FP64 integral values vs long-double evaluation: max abs %.2e, rms %.2e" % (d.max(), rms))
    assert d.max() < 1e-14 and rms < 5e-17
    # and the long-double tensor obeys the same symmetry and the closed form as the FP64 one
    assert np.max(np.abs(eld - eld.transpose(2, 3, 0, 1))) < 1e-17
