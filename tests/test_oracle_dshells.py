"""Pins for the Cartesian d shells of oracle/integrals.c (the paper's basis is 6-31G*).

As in test_oracle_integrals.py nothing here re-types the oracle's recursions.  The integrals with d functions are pinned
  * against an independent brute-force route: 1/r12 = (2/sqrt(pi)) int_0^inf exp(-u^2 r12^2) du, every u-term a product of
    three 2-D Gaussian moments evaluated by Gauss-Hermite quadrature (exact for these polynomials), the u integral by
    Gauss-Legendre (no Hermite expansion, no Boys function, no recursion);
  * against centre derivatives of the (already pinned) p classes:  (x-A)^2 g = (d/dA_x [(x-A) g] + g) / 2a,
    (x-A)(y-A_y) g = (d/dA_y [(x-A) g]) / 2a;
  * by closed forms of same-centre overlaps, the 8-fold symmetry, rigid-motion covariance of the d components and the
    plain N^4 contraction for J/K.
Reading R11 for d shells (oracle header): every Cartesian component is normalised, so xy, xz, yz carry sqrt(3) relative
to the bare monomial times the xx normalisation.
"""
import itertools

import numpy as np
import pytest

from oracle.integrals import OracleBasis, primitive_eri, primitive_eri_erf, primitive_norm
from workloads import Basis, get_config, make_basis

DPOW = [(2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 2, 0), (0, 1, 1), (0, 0, 2)]
DNORM = np.array([1.0, np.sqrt(3.0), np.sqrt(3.0), 1.0, np.sqrt(3.0), 1.0])


def _powers(l):
    return [(0, 0, 0)] if l == 0 else ([(1, 0, 0), (0, 1, 0), (0, 0, 1)] if l == 1 else DPOW)


def _cnorm(l):
    return DNORM if l == 2 else np.ones(2 * l + 1)


def _basis(centers, shells):
    sh_c, sh_l, sh_n, ex, co = [], [], [], [], []
    for (c, l, e, d) in shells:
        sh_c.append(c); sh_l.append(l); sh_n.append(len(e)); ex += list(e); co += list(d)
    sh_n = np.asarray(sh_n, dtype=np.int32)
    off = np.concatenate([[0], np.cumsum(sh_n)[:-1]]).astype(np.int32)
    return Basis(np.asarray(centers, dtype=np.float64), np.asarray(sh_c, dtype=np.int32),
                 np.asarray(sh_l, dtype=np.int32), sh_n, off, np.asarray(ex), np.asarray(co))


@pytest.fixture(scope="module")
def tinyd():
    basis = make_basis(get_config(6))
    ob = OracleBasis(basis)
    return dict(basis=basis, ob=ob, S=ob.overlap(), eri=ob.eri_tensor())


# ------------------------------------------------------------------------------------ brute force
_GH_X, _GH_W = np.polynomial.hermite.hermgauss(12)          # exact up to degree 23 against exp(-y^2)
_GL_X, _GL_W = np.polynomial.legendre.leggauss(64)


def _moment_2d(u2, a, A, i, b, B, j, c, C, k, d, D, l):
    """int int (x1-A)^i (x1-B)^j (x2-C)^k (x2-D)^l exp(-a(x1-A)^2 - b(x1-B)^2 - c(x2-C)^2 - d(x2-D)^2 - u2 (x1-x2)^2) dx1 dx2
    by a 12 x 12 Gauss-Hermite rule in the principal axes of the quadratic form."""
    p, q = a + b, c + d
    P, Q = (a * A + b * B) / p, (c * C + d * D) / q
    K = np.exp(-a * b / p * (A - B) ** 2 - c * d / q * (C - D) ** 2)
    M = np.array([[p + u2, -u2], [-u2, q + u2]])
    rhs = np.array([p * P, q * Q])
    m = np.linalg.solve(M, rhs)
    # exponent = -(x-m)^T M (x-m) - (p P^2 + q Q^2 - rhs^T m)
    e0 = np.exp(-(p * P * P + q * Q * Q - rhs @ m))
    Lc = np.linalg.cholesky(M)                               # M = Lc Lc^T, y = Lc^T (x - m)
    Y1, Y2 = np.meshgrid(_GH_X, _GH_X, indexing="ij")
    X = np.linalg.solve(Lc.T, np.stack([Y1.ravel(), Y2.ravel()]))
    x1, x2 = X[0] + m[0], X[1] + m[1]
    w = np.outer(_GH_W, _GH_W).ravel()
    poly = (x1 - A) ** i * (x1 - B) ** j * (x2 - C) ** k * (x2 - D) ** l
    return K * e0 * np.sum(w * poly) / np.linalg.det(Lc)


def eri_by_quadrature(ctr, ex, pw, omega=None):
    """(ab|cd) of bare Cartesian primitives (powers pw[4][3]) for 1/r12 (omega None) or erf(omega r12)/r12."""
    a, b, c, d = ex
    p, q = a + b, c + d
    alpha = p * q / (p + q)
    # u^2 = alpha t^2 / (1 - t^2), t in [0, tmax]: the integrand becomes a smooth function of t (for s functions
    # it is exp(-T t^2) up to a constant); tmax = 1 for 1/r12, omega / sqrt(alpha + omega^2) for the attenuated operator
    tmax = 1.0 if omega is None else omega / np.sqrt(alpha + omega * omega)
    tot = 0.0
    for (xg, wg) in zip(_GL_X, _GL_W):
        t = 0.5 * tmax * (xg + 1.0)
        u2 = alpha * t * t / (1.0 - t * t)
        dudt = np.sqrt(alpha) * (1.0 - t * t) ** -1.5
        f = 1.0
        for x in range(3):
            f *= _moment_2d(u2, a, ctr[0][x], pw[0][x], b, ctr[1][x], pw[1][x], c, ctr[2][x], pw[2][x], d, ctr[3][x], pw[3][x])
        tot += 0.5 * tmax * wg * f * dudt
    return 2.0 / np.sqrt(np.pi) * tot


@pytest.mark.parametrize("l4", [(2, 0, 0, 0), (0, 0, 2, 0), (2, 1, 0, 0), (2, 0, 0, 2), (1, 2, 2, 0), (2, 2, 1, 1), (2, 2, 2, 2),
                                (1, 1, 1, 1), (1, 0, 1, 0)])
def test_d_classes_against_gaussian_geminal_quadrature(l4):
    rng = np.random.default_rng(100 + sum(l4) * 7 + l4[0])
    ctr = rng.uniform(-0.9, 0.9, size=(4, 3))
    ex = np.exp(rng.uniform(np.log(0.4), np.log(2.5), size=4))
    blk = primitive_eri(ctr, ex, l4)
    comps = list(np.ndindex(*blk.shape))
    if len(comps) > 24:
        comps = [comps[i] for i in rng.choice(len(comps), size=24, replace=False)]
    scale = np.max(np.abs(blk))
    for comp in comps:
        pw = [_powers(l)[ci] for l, ci in zip(l4, comp)]
        nrm = np.prod([_cnorm(l)[ci] for l, ci in zip(l4, comp)])
        ref = nrm * eri_by_quadrature(ctr, ex, pw)
        assert abs(blk[comp] - ref) < 2e-12 * scale, (comp, blk[comp], ref)


def test_d_classes_erf_attenuated_against_quadrature():
    rng = np.random.default_rng(77)
    ctr = rng.uniform(-0.8, 0.8, size=(4, 3))
    ex = np.array([0.9, 0.6, 1.3, 0.5])
    for l4, omega in (((2, 0, 1, 0), 0.33), ((2, 2, 0, 0), 0.9), ((2, 1, 2, 1), 0.5)):
        blk = primitive_eri_erf(ctr, ex, l4, omega)
        full = primitive_eri(ctr, ex, l4)
        scale = np.max(np.abs(full))
        comps = list(np.ndindex(*blk.shape))
        for comp in [comps[i] for i in rng.choice(len(comps), size=min(12, len(comps)), replace=False)]:
            pw = [_powers(l)[ci] for l, ci in zip(l4, comp)]
            nrm = np.prod([_cnorm(l)[ci] for l, ci in zip(l4, comp)])
            ref = nrm * eri_by_quadrature(ctr, ex, pw, omega)
            assert abs(blk[comp] - ref) < 2e-12 * scale
        assert np.max(np.abs(blk - full)) > 1e-3 * scale        # the attenuation is not a no-op


# ------------------------------------------------------------------------------------ centre derivatives of p
@pytest.mark.parametrize("l4", [(2, 0, 0, 0), (0, 2, 0, 0), (0, 0, 0, 2), (2, 0, 2, 0), (1, 2, 0, 1), (2, 2, 0, 0)])
def test_d_classes_by_centre_derivative_of_p_classes(l4):
    rng = np.random.default_rng(21)
    ctr = rng.uniform(-1.0, 1.0, size=(4, 3))
    ex = np.array([0.7, 1.1, 0.5, 0.9])
    h = 2e-2
    stencil = [(-2, 1 / 12), (-1, -8 / 12), (1, 8 / 12), (2, -1 / 12)]
    blk = primitive_eri(ctr, ex, l4)
    didx = [i for i in range(4) if l4[i] == 2]

    def lower(lcur, sel, c, level):
        """Integral with the d indices didx[level:] still to be reduced; lcur/sel are the current l's / components."""
        if level == len(didx):
            return primitive_eri(c, ex, lcur)[tuple(sel)]
        k = didx[level]
        (i, j, m) = DPOW[sel[k]]
        axes = [0] * i + [1] * j + [2] * m                # the two Cartesian factors of this d component
        x, y = axes
        lp = list(lcur); lp[k] = 1
        sp = list(sel); sp[k] = x                          # p_x about centre k
        tot = 0.0
        for (mm, w) in stencil:                            # d/dA_y of the p_x integral
            c2 = c.copy(); c2[k, y] += mm * h
            tot += w * lower(lp, sp, c2, level + 1)
        val = tot / h
        if x == y:                                         # + the s integral
            ls = list(lcur); ls[k] = 0
            ss = list(sel); ss[k] = 0
            val += lower(ls, ss, c, level + 1)
        return DNORM[sel[k]] * val / (2 * ex[k])

    comps = list(np.ndindex(*blk.shape))
    if len(comps) > 18:
        comps = [comps[i] for i in rng.choice(len(comps), size=18, replace=False)]
    for comp in comps:
        fd = lower(list(l4), list(comp), ctr, 0)
        assert abs(blk[comp] - fd) < 5e-7 * max(1.0, abs(fd)), (comp, blk[comp], fd)


# ------------------------------------------------------------------------------------ one-electron
def test_d_overlap_same_centre_closed_forms():
    a, b = 0.8, 1.9
    ob = OracleBasis(_basis([[0.1, 0.2, -0.3]], [(0, 2, [a, b], [0.6, 0.5]), (0, 0, [a], [1.0]), (0, 1, [b], [1.0])]))
    S = ob.overlap()
    d = S[:6, :6]
    assert np.max(np.abs(np.diag(S) - 1.0)) < 1e-14                    # every component normalised (R11)
    # int x^2 y^2 = (1/3) int x^4 for any radial part: <xx|yy> = 1/3; odd integrands vanish
    expect = np.eye(6)
    for (i, j) in ((0, 3), (0, 5), (3, 5)):
        expect[i, j] = expect[j, i] = 1.0 / 3.0
    assert np.max(np.abs(d - expect)) < 1e-14
    assert np.max(np.abs(S[:6, 7:10])) < 1e-15                         # <d|p> = 0 on one centre
    # <s|xx> for single primitives: N_s N_xx (pi/p)^{3/2} / (2p)
    ob1 = OracleBasis(_basis([[0, 0, 0]], [(0, 2, [a], [1.0]), (0, 0, [b], [1.0])]))
    S1 = ob1.overlap()
    p = a + b
    val = primitive_norm(b, 0) * primitive_norm(a, 2) * (np.pi / p) ** 1.5 / (2 * p)
    assert abs(S1[0, 6] - val) < 1e-15 and abs(S1[3, 6] - val) < 1e-15 and abs(S1[1, 6]) < 1e-16


def _raw_1e(A, la, a, B, lb, b, what, origin=(0.3, -0.2, 0.1)):
    ob = OracleBasis(_basis([A, B], [(0, la, [a], [1.0]), (1, lb, [b], [1.0])]))
    na = (la + 1) * (la + 2) // 2
    M = ob.overlap() if what == "S" else ob.dipole(origin)
    return M[..., :na, na:] / (ob.ncoef[0] * ob.ncoef[1])


@pytest.mark.parametrize("lb", [0, 1, 2])
def test_d_overlap_and_dipole_by_centre_derivative_of_p(lb):
    A, B = np.array([0.3, -0.1, 0.2]), np.array([-0.5, 0.6, 0.9])
    a, b, h = 0.9, 0.6, 1e-3
    for what in ("S", "D"):
        dblk = _raw_1e(A, 2, a, B, lb, b, what)                       # [..., 6, nb]
        s0 = _raw_1e(A, 0, a, B, lb, b, what)
        for ci, (i, j, m) in enumerate(DPOW):
            x, y = ([0] * i + [1] * j + [2] * m)
            e = np.zeros(3); e[y] = h
            f = lambda Av: _raw_1e(Av, 1, a, B, lb, b, what)[..., x, :]
            fd = (-f(A + 2 * e) + 8 * f(A + e) - 8 * f(A - e) + f(A - 2 * e)) / (12 * h)
            ref = DNORM[ci] * (fd + (s0[..., 0, :] if x == y else 0.0)) / (2 * a)
            assert np.max(np.abs(dblk[..., ci, :] - ref)) < 1e-9


# ------------------------------------------------------------------------------------ invariants on the d molecule
def test_d_molecule_symmetry_schwarz_and_jk(tinyd):
    ob, eri, N = tinyd["ob"], tinyd["eri"], tinyd["basis"].nao
    assert N == 60 and np.max(np.abs(np.diag(tinyd["S"]) - 1.0)) < 1e-14
    for perm in [(1, 0, 2, 3), (0, 1, 3, 2), (2, 3, 0, 1), (3, 2, 1, 0)]:
        assert np.max(np.abs(eri - eri.transpose(perm))) < 1e-15
    diag = np.einsum("mnmn->mn", eri)
    assert diag.min() >= 0.0
    bound = np.sqrt(diag)[:, :, None, None] * np.sqrt(diag)[None, None, :, :]
    assert np.all(np.abs(eri) <= bound * (1 + 1e-12) + 1e-15)
    Q = ob.schwarz()
    off, l = ob.ao_off, ob.sh_l
    nc = (l + 1) * (l + 2) // 2
    for a in range(ob.nshells):
        for b in (0, 4, 9):
            blk = diag[off[a]:off[a] + nc[a], off[b]:off[b] + nc[b]]
            assert abs(Q[a, b] - np.sqrt(blk.max())) < 1e-15
    T = np.random.default_rng(3).standard_normal((2, N, N))
    J, K, nq, _ = ob.jk(T, tau=0.0)
    Jref = np.einsum("mnls,vls->vmn", eri, T)
    Kref = np.einsum("mnls,vns->vml", eri, T)
    assert np.max(np.abs(J - Jref)) < 1e-12 and np.max(np.abs(K - Kref)) < 1e-12
    # long-double route of the integrals agrees with the FP64 route to rounding
    eld = ob.eri_tensor_ld()
    dd = np.asarray(eld - eri.astype(np.longdouble), dtype=np.float64)
    assert np.max(np.abs(dd)) < 2e-14


def test_d_molecule_rigid_motion(tinyd):
    basis, eri = tinyd["basis"], tinyd["eri"]
    th = 0.83
    Rz = np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, 1.0]])
    Rx = np.array([[1.0, 0, 0], [0, np.cos(0.4), -np.sin(0.4)], [0, np.sin(0.4), np.cos(0.4)]])
    Rm = Rz @ Rx
    b2 = Basis(basis.centers @ Rm.T + np.array([3.0, -2.0, 0.5]), basis.sh_center, basis.sh_l,
               basis.sh_nprim, basis.sh_off, basis.exps, basis.coefs)
    eri2 = OracleBasis(b2).eri_tensor()
    N = basis.nao
    U = np.eye(N)
    pairs = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]
    Ud = np.zeros((6, 6))
    for c, (i, j) in enumerate(pairs):              # m'_{ij} = sum_{kl} R_ik R_jl m_kl, monomials with k <= l
        for c2, (k, l) in enumerate(pairs):
            v = Rm[i, k] * Rm[j, l] + (Rm[i, l] * Rm[j, k] if k != l else 0.0)
            Ud[c, c2] = DNORM[c] / DNORM[c2] * v
    for s, o in enumerate(basis.ao_off):
        if basis.sh_l[s] == 1:
            U[o:o + 3, o:o + 3] = Rm
        if basis.sh_l[s] == 2:
            U[o:o + 6, o:o + 6] = Ud
    ref = np.einsum("pm,qn,rl,ts,mnls->pqrt", U, U, U, U, eri, optimize=True)
    assert np.max(np.abs(eri2 - ref)) < 1e-13


def test_d_contracted_equals_sum_of_primitives():
    ctrs = [[0, 0, 0], [0.9, 0.3, -0.4], [-0.5, 1.0, 0.6]]
    ob = OracleBasis(_basis(ctrs, [(0, 2, [0.5, 1.4, 0.9], [0.3, 0.8, 0.5]), (1, 2, [0.7, 1.1], [0.6, 0.4]),
                                   (2, 1, [0.8, 0.4], [0.5, 0.5]), (1, 0, [1.2], [1.0])]))
    for sh in [(0, 1, 2, 3), (0, 0, 1, 1), (1, 2, 0, 3)]:
        blk = ob.shell_quartet(*sh)
        ref = np.zeros_like(blk)
        for ks in itertools.product(*[range(ob.sh_nprim[s]) for s in sh]):
            idx = [ob.sh_off[s] + k for s, k in zip(sh, ks)]
            c4 = np.array([ob.centers[ob.sh_center[s]] for s in sh])
            ref += np.prod(ob.ncoef[idx]) * primitive_eri(c4, ob.exps[idx], [ob.sh_l[s] for s in sh])
        assert np.max(np.abs(blk - ref)) < 1e-14
