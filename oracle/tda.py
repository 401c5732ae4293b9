"""ORACLE (test infrastructure, not the product): the RT-TDA definitions in plain numpy, fp64.

Follows PAPER.md section 2 in the paper's order and notation; every reading of an ambiguous passage
is listed in DESIGN.md ("Readings").  Nothing here is blocked, fused or reordered.

  A_{ia,jb} = delta_ij delta_ab (eps_a - eps_i) + 2 (ia|jb) - c_x (ij|ab)        eq. 3, R1
  index ia = i*nvirt + a (virtuals run fastest)
  sigma = A X                                                                      eq. 11
  extended vector: element 0 = KS ground state, A_00 = 0, A_0,ia = 0               P:102, R2
  X = q + i p, (q', p') = (H p, -H q)                                              eq. 12-15
  H(t) = A_ext + E(t) M,  M = CSF matrix of the position operator along d          eq. 16, R5
  M from MO-basis dipoles via the Slater-Condon rules                              eq. 19a-f
  pulses                                                                           eq. 18a-d
  R(t) = X(eps)^dagger X(eps + t)                                                  eq. 20
"""
from __future__ import annotations

import numpy as np

SQRT2 = np.sqrt(2.0)


# ---------------------------------------------------------------- A matrix and sigma (dense route)
def mo_eri_blocks(eri, C_o, C_v):
    """(ia|jb) and (ij|ab) from the AO tensor (mu nu|lam sig) by four quarter transforms (eq. 4)."""
    ovov = np.einsum("mnls,mi,na,lj,sb->iajb", eri, C_o, C_v, C_o, C_v, optimize=True)
    oovv = np.einsum("mnls,mi,nj,la,sb->ijab", eri, C_o, C_o, C_v, C_v, optimize=True)
    return ovov, oovv


def build_A(eri, C_o, C_v, eps, cx=1.0):
    """Dense singles block of A (eq. 3 under R1), shape [nocc*nvirt][nocc*nvirt]."""
    no, nv = C_o.shape[1], C_v.shape[1]
    ovov, oovv = mo_eri_blocks(eri, C_o, C_v)
    A = 2.0 * ovov - cx * np.transpose(oovv, (0, 2, 1, 3))     # (ij|ab) -> [i][a][j][b]
    A = A.reshape(no * nv, no * nv).copy()
    de = (eps[no:][None, :] - eps[:no][:, None]).reshape(-1)    # eps_a - eps_i at ia = i*nv + a
    A[np.diag_indices(no * nv)] += de
    return A


def build_A_rs(eri, eri_lr, C_o, C_v, eps, cx, cx_lr):
    """Range-separated exchange (NEXT-4; CAM-type functionals):
    A_{ia,jb} = delta delta (eps_a - eps_i) + 2 (ia|jb) - c_x (ij|ab) - c_x^LR (ij| erf(omega r12)/r12 |ab),
    `eri_lr` being the AO tensor of the attenuated operator (OracleBasis.eri_tensor_erf)."""
    no, nv = C_o.shape[1], C_v.shape[1]
    A = build_A(eri, C_o, C_v, eps, cx)
    _, oovv_lr = mo_eri_blocks(eri_lr, C_o, C_v)
    return A - cx_lr * np.transpose(oovv_lr, (0, 2, 1, 3)).reshape(no * nv, no * nv)


def sigma_matrix_free_rs(ob, X, C_o, C_v, eps, cx, cx_lr, omega, tau=0.0, Q=None):
    """sigma for the range-separated A through the matrix-free routes: F = 2 J - c_x K - c_x^LR K_erf."""
    T = transition_density(X, C_o, C_v)
    J, K, nq, npq = ob.jk(T, tau=tau, Q=Q)
    _, K_lr, _, _ = ob.jk_erf(T, omega, tau=tau, Q=Q)
    return sigma_from_jk(X, J, K + (cx_lr / cx) * K_lr if cx != 0.0 else K, C_o, C_v, eps, cx) if cx != 0.0 else \
        sigma_from_jk(X, J, K_lr, C_o, C_v, eps, cx_lr), nq, npq


def build_A_by_pair_blocks(ob, C_o, C_v, eps, cx=1.0, tau=0.0, Q=None, progress=None):
    """Dense singles block of A (eq. 3 under R1) for systems whose AO tensor does not fit (SURVEY 8(c5) route ii):
    AO integrals one ket shell pair (lam sig) at a time, half-transformed at once,
        (ia|lam sig) = sum_{mu nu} C_{mu i} C_{nu a} (mu nu|lam sig),   (ij|lam sig) likewise,
    stored for all (lam, sig), then the second half transform over (lam, sig).  Same quarter transforms as
    `mo_eri_blocks`, only ordered so that N^4 doubles never exist at once.  Memory: no*nv*N^2 + no^2*N^2 doubles."""
    no, nv, N = C_o.shape[1], C_v.shape[1], C_o.shape[0]
    if Q is None:
        Q = ob.schwarz()
    ov = np.zeros((no * nv, N, N))
    oo = np.zeros((no * no, N, N))
    for sc in range(ob.nshells):
        for sd in range(sc + 1):
            blk = ob.eri_pair_block(sc, sd, tau, Q)                       # [N][N][nc][nd]
            oc, od = int(ob.ao_off[sc]), int(ob.ao_off[sd])
            for cc in range(blk.shape[2]):
                for cd in range(blk.shape[3]):
                    M = blk[:, :, cc, cd]
                    half = C_o.T @ M                                        # [no][N]
                    via = (half @ C_v).reshape(-1)
                    vij = (half @ C_o).reshape(-1)
                    ov[:, oc + cc, od + cd] = via
                    ov[:, od + cd, oc + cc] = via                           # (mu nu|lam sig) = (mu nu|sig lam)
                    oo[:, oc + cc, od + cd] = vij
                    oo[:, od + cd, oc + cc] = vij
        if progress:
            progress(sc)
    A = np.empty((no * nv, no * nv))
    step = max(1, 2 ** 27 // (N * N))                                      # rows of `ov` per chunk (~1 GB)
    for r0 in range(0, no * nv, step):
        t = ov[r0:r0 + step] @ C_v                                         # [rows][lam][b]
        t = np.einsum("rlb,lj->rjb", t, C_o, optimize=True)                # [rows][j][b]
        A[r0:r0 + step] = 2.0 * t.reshape(t.shape[0], -1)
    del ov
    t = oo @ C_v                                                           # [ij][lam][b]
    oovv = np.einsum("rlb,la->rab", t, C_v, optimize=True).reshape(no, no, nv, nv)   # (ij|ab)
    A -= cx * np.transpose(oovv, (0, 2, 1, 3)).reshape(no * nv, no * nv)
    de = (eps[no:][None, :] - eps[:no][:, None]).reshape(-1)
    A[np.diag_indices(no * nv)] += de
    return A


def extend_A(A):
    """A_ext = diag(A_00 = 0, A), no coupling between element 0 and the singles (R2)."""
    n = A.shape[0]
    Ae = np.zeros((n + 1, n + 1))
    Ae[1:, 1:] = A
    return Ae


def sigma_dense(A, X):
    """sigma_v = A x_v for X [nvec][ncsf] (eq. 11)."""
    return X @ A.T


def transition_density(X, C_o, C_v):
    """T_v = C_o X_v C_v^T  (T_{lam sig} = sum_jb C_{lam j} X_jb C_{sig b}); NOT symmetric."""
    no, nv = C_o.shape[1], C_v.shape[1]
    return np.einsum("lj,vjb,sb->vls", C_o, X.reshape(-1, no, nv), C_v, optimize=True)


def sigma_from_jk(X, J, K, C_o, C_v, eps, cx=1.0):
    """sigma = d_eps o X + C_o^T (2 J - c_x K) C_v  (matrix-free identity of DESIGN.md)."""
    no, nv = C_o.shape[1], C_v.shape[1]
    de = (eps[no:][None, :] - eps[:no][:, None]).reshape(-1)
    F = 2.0 * J - cx * K
    S = np.einsum("mi,vmn,na->via", C_o, F, C_v, optimize=True).reshape(X.shape[0], no * nv)
    return de[None, :] * X + S


def sigma_matrix_free(ob, X, C_o, C_v, eps, cx=1.0, tau=0.0, Q=None):
    """sigma through the oracle's own J/K (ob: oracle.integrals.OracleBasis)."""
    T = transition_density(X, C_o, C_v)
    J, K, nq, npq = ob.jk(T, tau=tau, Q=Q)
    return sigma_from_jk(X, J, K, C_o, C_v, eps, cx), nq, npq


def sigma_matrix_free_ld(ob, X, C_o, C_v, eps, cx=1.0, tau=0.0, Q=None):
    """The same matrix-free identity with every step past the FP64 integral values in x87 long double (SURVEY 8(c):
    long-double J/K sums and MO transforms): T = C_o X C_v^T, J/K by `ob.jk_ld`, sigma = d_eps o X + C_o^T (2J - c_x K) C_v,
    all as np.longdouble matrix products.  Returns (sigma as np.longdouble, n_shell_quartets, n_prim_quartets); the
    difference to `sigma_matrix_free` is the rounding-noise floor of the FP64 route."""
    ld = np.longdouble
    no, nv = C_o.shape[1], C_v.shape[1]
    Co, Cv, Xl = C_o.astype(ld), C_v.astype(ld), np.asarray(X, dtype=ld).reshape(-1, no, nv)
    T = np.stack([Co @ x @ Cv.T for x in Xl])
    J, K, nq, npq = ob.jk_ld(T, tau=tau, Q=Q)
    de = (eps[no:].astype(ld)[None, :] - eps[:no].astype(ld)[:, None]).reshape(-1)
    F = ld(2.0) * J - ld(cx) * K
    S = np.stack([(Co.T @ f @ Cv).reshape(-1) for f in F])
    return de[None, :] * Xl.reshape(-1, no * nv) + S, nq, npq


# ---------------------------------------------------------------- dipole operator in the CSF basis
def mo_dipoles(D_ao, C_o, C_v, d):
    """D_d = sum_k d_k D^k in the MO basis: D_oo, D_vv, D_ov and D_00 = 2 tr D_oo (R3).

    Dipole origin (reading R6): the electronic centroid of the ground state, c = tr(D_oo)/n_occ along d.  The paper's
    dipole operator is the molecular one: for a neutral molecule it does not depend on the origin and its
    ground-state expectation value (eq. 19a) is the permanent dipole moment, O(1) au.  The synthetic centres carry no
    charges (R5), so the bare electronic D_00 = 2 sum_i <i|r|i> would grow with the distance of the molecule from
    the coordinate origin (1e4 au for the 1280-AO molecule: a global phase rotating 500 times faster than any
    excitation, which no fixed-step propagator at the configs' dt can follow).  With orthonormal MOs (C^T S C = 1,
    checked by the tests) the shift r -> r - c acts as D_oo -> D_oo - c 1, D_vv -> D_vv - c 1, D_ov unchanged, and
    D_00 -> 0; eq. 19a-f are applied unchanged to the shifted matrices."""
    Dd = np.einsum("k,kmn->mn", np.asarray(d, dtype=np.float64), D_ao)
    D_oo = C_o.T @ Dd @ C_o
    D_vv = C_v.T @ Dd @ C_v
    D_ov = C_o.T @ Dd @ C_v
    c = np.trace(D_oo) / D_oo.shape[0]
    D_oo = D_oo - c * np.eye(D_oo.shape[0])
    D_vv = D_vv - c * np.eye(D_vv.shape[0])
    return D_oo, D_vv, D_ov, 2.0 * np.trace(D_oo)


def build_M_explicit(D_oo, D_vv, D_ov, D_00):
    """The six Slater-Condon rules of eq. 19, element by element (R3, R4)."""
    no, nv = D_ov.shape
    n = no * nv
    M = np.zeros((n + 1, n + 1))
    M[0, 0] = D_00                                                    # 19a
    for i in range(no):
        for a in range(nv):
            ia = 1 + i * nv + a
            M[0, ia] = M[ia, 0] = SQRT2 * D_ov[i, a]                  # 19b
            for j in range(no):
                for b in range(nv):
                    jb = 1 + j * nv + b
                    if i == j and a == b:
                        M[ia, jb] = D_00 - D_oo[i, i] + D_vv[a, a]    # 19c
                    elif i == j:
                        M[ia, jb] = D_vv[a, b]                        # 19d
                    elif a == b:
                        M[ia, jb] = -D_oo[i, j]                       # 19e
                    # else 0: differ by more than one electron       # 19f
    return M


def apply_M(y, D_oo, D_vv, D_ov, D_00):
    """Matrix-free M y:  (My)_0 = D_00 y_0 + sqrt2 sum D_ov Y;  (My)_ia = [sqrt2 D_ov y_0 + D_00 Y
    + Y D_vv - D_oo Y]_ia.  y may be complex, shape [1+ncsf]."""
    no, nv = D_ov.shape
    Y = y[1:].reshape(no, nv)
    out = np.empty_like(y)
    out[0] = D_00 * y[0] + SQRT2 * np.sum(D_ov * Y)
    out[1:] = (SQRT2 * D_ov * y[0] + D_00 * Y + Y @ D_vv - D_oo @ Y).reshape(-1)
    return out


# ---------------------------------------------------------------- pulses (eq. 18) and propagation
def field_value(f: dict, t: float) -> float:
    """Scalar E(t).  'delta' is applied as a kick by `kick`, its E(t) is 0 (R8)."""
    typ = f.get("type", "none")
    if typ in ("none", "delta"):
        return 0.0
    E0, w = f["E0"], f.get("omega", 0.0)
    if typ == "cw":                                                   # 18b
        return E0 * np.sin(w * t)
    if typ == "tl":                                                   # 18c
        s = t - f["t0"]
        return E0 * np.exp(-s * s / (2.0 * f["sigma"] ** 2)) * np.sin(w * s)
    if typ == "chirp":                                                # 18d
        s = t - f["t0"]
        return E0 * np.exp(-s * s / (2.0 * f["sigma"] ** 2)) * np.sin((w + 0.5 * f["beta"] * s) * s)
    if typ == "sin2":                                                 # R9
        Te = f["T_env"]
        if t < 0.0 or t > Te:
            return 0.0
        return E0 * np.sin(np.pi * t / Te) ** 2 * np.sin(w * t)
    raise ValueError(typ)


def kick(y, f, apply_Md):
    """Linearised delta kick y(0+) = (1 - i kappa M_d) y(0), kappa = E0 (R8)."""
    return y - 1j * f["E0"] * apply_Md(y)


def rk4_propagate(apply_A_ext, apply_Md, y0, f, t_start, dt, nsteps, log=True):
    """Classical RK4 on y' = -i H(t) y, H(t) y = A_ext y + E(t) M_d y (eq. 1, 14-16; R7).

    Stage times t, t+dt/2, t+dt/2, t+dt; weights 1/6, 1/3, 1/3, 1/6.  A 'delta' field is applied
    as the linearised kick at t_start and the run is then field-free.  Returns (y, log) with
    log[n] = (|y|^2, Re R, Im R), R = y(t_start+)^dagger y(t_{n+1}) (eq. 20)."""
    y = np.array(y0, dtype=np.complex128)
    if f.get("type") == "delta":
        y = kick(y, f, apply_Md)
    yref = y.copy()

    def rhs(t, z):
        E = field_value(f, t)
        h = apply_A_ext(z)
        if E != 0.0:
            h = h + E * apply_Md(z)
        return -1j * h

    out = np.zeros((nsteps, 3))
    t = t_start
    for n in range(nsteps):
        k1 = rhs(t, y)
        k2 = rhs(t + 0.5 * dt, y + 0.5 * dt * k1)
        k3 = rhs(t + 0.5 * dt, y + 0.5 * dt * k2)
        k4 = rhs(t + dt, y + dt * k3)
        y = y + (dt / 6.0) * (k1 + 2.0 * k2 + 2.0 * k3 + k4)
        t = t_start + (n + 1) * dt
        if log:
            R = np.vdot(yref, y)
            out[n] = (np.vdot(y, y).real, R.real, R.imag)
    return y, out


def rk4_dense(A, D_oo, D_vv, D_ov, D_00, y0, f, t_start, dt, nsteps):
    """RK4 with the dense singles block A (element 0 decoupled, A_00 = 0)."""
    def apply_A_ext(z):
        o = np.empty_like(z)
        o[0] = 0.0
        o[1:] = A @ z[1:]
        return o
    return rk4_propagate(apply_A_ext, lambda z: apply_M(z, D_oo, D_vv, D_ov, D_00), y0, f,
                         t_start, dt, nsteps)


def rk4_matrix_free(ob, C_o, C_v, eps, cx, tau, Q, D_oo, D_vv, D_ov, D_00, y0, f, t_start, dt,
                    nsteps):
    """RK4 where A_ext z is applied through the oracle's matrix-free sigma (real and imaginary
    parts as two vectors of one J/K pass)."""
    def apply_A_ext(z):
        X = np.stack([z[1:].real, z[1:].imag])
        s, _, _ = sigma_matrix_free(ob, X, C_o, C_v, eps, cx, tau, Q)
        o = np.empty_like(z)
        o[0] = 0.0
        o[1:] = s[0] + 1j * s[1]
        return o
    return rk4_propagate(apply_A_ext, lambda z: apply_M(z, D_oo, D_vv, D_ov, D_00), y0, f,
                         t_start, dt, nsteps)


# ---------------------------------------------------------------- SSO propagator (NEXT-1; reading R22)
def sso_propagate(apply_A_ext, apply_Md, y0, f, t_start, dt, nsteps, log=True):
    """Second-order symplectic split-operator step on (q', p') = (H p, -H q) (eq. 14-15; "SSO").

    The paper names the integrator and its cost (2 sigma builds per step) but prints no update formulas;
    reading R22 takes the Stoermer-Verlet splitting with H evaluated at the time of each sub-step:
        p_half  = p_n    - (dt/2) H(t_n)        q_n
        q_{n+1} = q_n    +  dt    H(t_n + dt/2) p_half
        p_{n+1} = p_half - (dt/2) H(t_{n+1})    q_{n+1}
    H(t_{n+1}) q_{n+1} is reused as the first half-kick of the next step: two applications of H to a REAL vector
    per step.  A 'delta' field is the linearised kick of R8 at t_start.  Returns (y, log) as rk4_propagate."""
    y = np.array(y0, dtype=np.complex128)
    if f.get("type") == "delta":
        y = kick(y, f, apply_Md)
    yref = y.copy()

    def H(t, x):                                    # x real; A_ext and M_d are real operators
        E = field_value(f, t)
        h = apply_A_ext(x.astype(np.complex128)).real
        if E != 0.0:
            h = h + E * apply_Md(x.astype(np.complex128)).real
        return h

    q, p = y.real.copy(), y.imag.copy()
    out = np.zeros((nsteps, 3))
    hq = H(t_start, q)
    for n in range(nsteps):
        t = t_start + n * dt
        p = p - 0.5 * dt * hq
        q = q + dt * H(t + 0.5 * dt, p)
        hq = H(t + dt, q)
        p = p - 0.5 * dt * hq
        if log:
            yy = q + 1j * p
            R = np.vdot(yref, yy)
            out[n] = (np.vdot(yy, yy).real, R.real, R.imag)
    return q + 1j * p, out


def sso_dense(A, D_oo, D_vv, D_ov, D_00, y0, f, t_start, dt, nsteps):
    """SSO with the dense singles block A (element 0 decoupled, A_00 = 0)."""
    def apply_A_ext(z):
        o = np.empty_like(z)
        o[0] = 0.0
        o[1:] = A @ z[1:]
        return o
    return sso_propagate(apply_A_ext, lambda z: apply_M(z, D_oo, D_vv, D_ov, D_00), y0, f,
                         t_start, dt, nsteps)


# ---------------------------------------------------------------- populations (NEXT-2)
def populations(Xs, y):
    """P_i = |X_i^dagger y|^2, eq. 22: projection of the time-dependent vector y (length 1 + N_CSF, complex)
    onto stationary states X_i (rows of Xs, real or complex, same length; the ground state is e_0)."""
    Xs = np.atleast_2d(np.asarray(Xs))
    return np.abs(Xs.conj() @ np.asarray(y)) ** 2


# ---------------------------------------------------------------- Lanczos on A (NEXT-3: TI-TDA eigenvalues, eq. 2)
def lanczos(apply_A, v0, m, reorth=True):
    """m steps of the symmetric Lanczos process on the singles block A (TI-TDA eigenproblem A X = omega X, eq. 2):
        v_1 = v0/|v0|;  w = A v_j - beta_{j-1} v_{j-1};  alpha_j = v_j.w;  w -= alpha_j v_j;
        (reorth: w -= V_j (V_j^T w), applied twice);  beta_j = |w|;  v_{j+1} = w / beta_j.
    Returns alpha [m], beta [m], V [m+1][n]; the Ritz values are the eigenvalues of tridiag(alpha, beta[:-1])."""
    n = v0.shape[0]
    V = np.zeros((m + 1, n))
    alpha, beta = np.zeros(m), np.zeros(m)
    V[0] = v0 / np.linalg.norm(v0)
    for j in range(m):
        w = apply_A(V[j])
        if j > 0:
            w = w - beta[j - 1] * V[j - 1]
        alpha[j] = V[j] @ w
        w = w - alpha[j] * V[j]
        if reorth:
            for _ in range(2):
                w = w - V[: j + 1].T @ (V[: j + 1] @ w)
        beta[j] = np.linalg.norm(w)
        V[j + 1] = w / beta[j]
    return alpha, beta, V


# ---------------------------------------------------------------- block Davidson on A (NEXT-3: TI-TDA eigenpairs, eq. 2)
def davidson(apply_A, diag, k, nblock=None, tol=1e-8, maxiter=200):
    """Lowest k eigenpairs of the singles block A (A X = omega X, eq. 2) by block Davidson:
        V orthonormal search space (rows), W = A V, H = V W^T, Ritz pairs (theta, y) of H;
        x_j = y_j V, r_j = y_j W - theta_j x_j; stop when max_j |r_j| <= tol;
        new directions r_j / (theta_j - diag) for the unconverged roots (|denominator| >= 1e-4), orthonormalised against
        V by two Gram-Schmidt passes; start = unit vectors on the nblock smallest entries of diag = eps_a - eps_i.
    `apply_A` maps rows [m][n] -> [m][n].  Returns (omega [k], X [k][n], residual norms [k], iterations)."""
    n = diag.shape[0]
    nb = min(max(nblock or k, k), n)
    V = np.zeros((nb, n))
    V[np.arange(nb), np.argsort(diag, kind="stable")[:nb]] = 1.0
    W = apply_A(V)
    for it in range(1, maxiter + 1):
        H = V @ W.T
        th, Y = np.linalg.eigh(0.5 * (H + H.T))
        kk = min(nb, V.shape[0])
        X = Y[:, :kk].T @ V
        R = Y[:, :kk].T @ W - th[:kk, None] * X
        rn = np.linalg.norm(R, axis=1)
        if np.max(rn[:k]) <= tol or V.shape[0] >= n:
            return th[:k], X[:k], rn[:k], it
        new = []
        for j in range(kk):
            if j < k and rn[j] <= tol:
                continue
            d = th[j] - diag
            d = np.where(np.abs(d) < 1e-4, np.where(d < 0, -1e-4, 1e-4), d)
            t = R[j] / d
            B = np.vstack([V] + new) if new else V
            for _ in range(2):
                t = t - B.T @ (B @ t)
            nt = np.linalg.norm(t)
            if nt > 1e-12:
                new.append((t / nt)[None, :])
        if not new:
            return th[:k], X[:k], rn[:k], it
        Vn = np.vstack(new)
        V = np.vstack([V, Vn])
        W = np.vstack([W, apply_A(Vn)])
    return th[:k], X[:k], rn[:k], maxiter


# ---------------------------------------------------------------- spectrum (harness for the pins)
def spectrum(R, dt, pad=50000):
    """omega * F[R(t)] with mirroring R(-t) = R(t)^*, Hann window, zero padding (eq. 21).

    R holds R(t_n) for n = 0..n-1 (R[0] = R(0)).  Returns (omega, intensity)."""
    R = np.asarray(R, dtype=np.complex128)
    full = np.concatenate([np.conj(R[:0:-1]), R])                   # t = -(n-1)dt .. (n-1)dt
    full = full * np.hanning(full.shape[0])
    npad = full.shape[0] + pad
    ft = np.fft.fft(full, n=npad)
    om = 2.0 * np.pi * np.fft.fftfreq(npad, d=dt)
    # R(t) = sum |c_I|^2 exp(-i w_I t): peaks sit at om = -w_I in numpy's sign convention
    keep = om < 0
    return -om[keep][::-1], (-om[keep] * np.abs(ft[keep]))[::-1]
