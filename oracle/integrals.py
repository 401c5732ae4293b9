"""ORACLE (test infrastructure, not the product): ctypes front-end of oracle/integrals.c.

Builds liboracle.so with gcc on first use.  Inputs are the plain arrays of `workloads.Basis`
(duck-typed: this package imports neither `workloads` nor the CUDA package).
"""
from __future__ import annotations

import ctypes as ct
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "integrals.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

_dp = ct.POINTER(ct.c_double)
_ip = ct.POINTER(ct.c_int32)


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ct.CDLL(build())
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(_ip)


def boys(nmax: int, T: float) -> np.ndarray:
    F = np.zeros(nmax + 1)
    lib().oracle_boys(ct.c_int(nmax), ct.c_double(T), F.ctypes.data_as(_dp))
    return F


def ncart(l):
    """Cartesian components of a shell: 1 (s), 3 (p), 6 (d: xx, xy, xz, yy, yz, zz)."""
    l = np.asarray(l)
    return (l + 1) * (l + 2) // 2


def primitive_norm(a, l):
    """N(a,0) = (2a/pi)^(3/4); N(a,1) = N(a,0) 2 sqrt(a); N(a,2) = N(a,0) 4a / sqrt(3), the norm of the xx
    component (xy, xz, yz carry sqrt(3) more inside integrals.c)  (definitions)."""
    a = np.asarray(a, dtype=np.float64)
    l = np.asarray(l)
    n = (2.0 * a / np.pi) ** 0.75
    return n * np.where(l == 1, 2.0 * np.sqrt(a), np.where(l == 2, 4.0 * a / np.sqrt(3.0), 1.0))


class OracleBasis:
    """Holds the basis arrays + final coefficients (R11: each contracted AO scaled to <phi|phi>=1,
    the scale taken from this oracle's own overlap routine)."""

    def __init__(self, basis):
        self.centers, self._pc = _d(basis.centers)
        self.sh_center, self._psc = _i(basis.sh_center)
        self.sh_l, self._pl = _i(basis.sh_l)
        self.sh_nprim, self._pn = _i(basis.sh_nprim)
        self.sh_off, self._po = _i(basis.sh_off)
        self.nshells = int(self.sh_l.shape[0])
        n = ncart(self.sh_l.astype(np.int64))
        self.ao_off, self._pa = _i(np.concatenate([[0], np.cumsum(n)[:-1]]))
        self.nao = int(n.sum())
        self.exps, self._pe = _d(basis.exps)
        l_of_prim = np.repeat(self.sh_l, self.sh_nprim)
        raw = np.asarray(basis.coefs, dtype=np.float64) * primitive_norm(self.exps, l_of_prim)
        self.ncoef, self._pk = _d(raw)
        S = self.overlap()
        scale = 1.0 / np.sqrt(np.diag(S))
        sh_scale = scale[self.ao_off]          # first component (x of p, xx of d): the shell's radial part
        self.ncoef, self._pk = _d(raw * np.repeat(sh_scale, self.sh_nprim))

    def _args(self):
        return (ct.c_int(self.nshells), self._pc, self._psc, self._pl, self._pn, self._po,
                self._pa, self._pe, self._pk)

    def overlap(self) -> np.ndarray:
        S = np.zeros((self.nao, self.nao))
        O = np.zeros(3)
        lib().oracle_one_electron(*self._args(), ct.c_int(self.nao), O.ctypes.data_as(_dp),
                                  S.ctypes.data_as(_dp), None)
        return S

    def dipole(self, origin=(0.0, 0.0, 0.0)):
        S = np.zeros((self.nao, self.nao))
        D = np.zeros((3, self.nao, self.nao))
        O = np.asarray(origin, dtype=np.float64)
        lib().oracle_one_electron(*self._args(), ct.c_int(self.nao), O.ctypes.data_as(_dp),
                                  S.ctypes.data_as(_dp), D.ctypes.data_as(_dp))
        return D

    def shell_quartet(self, a, b, c, d) -> np.ndarray:
        n = [int(ncart(int(self.sh_l[s]))) for s in (a, b, c, d)]
        out = np.zeros(n)
        lib().oracle_shell_quartet(*self._args(), ct.c_int(a), ct.c_int(b), ct.c_int(c),
                                   ct.c_int(d), out.ctypes.data_as(_dp))
        return out

    def eri_tensor(self) -> np.ndarray:
        N = self.nao
        if N > 256:                       # memory guard only: 256^4 doubles = 34 GB (config 2 needs 200^4 = 12.8 GB)
            raise ValueError("full N^4 tensor only for small systems (N <= 256)")
        eri = np.zeros((N, N, N, N))
        lib().oracle_eri_tensor(*self._args(), ct.c_int(N), eri.ctypes.data_as(_dp))
        return eri

    def eri_tensor_ld(self) -> np.ndarray:
        """Full AO tensor with every intermediate of the integral evaluation in x87 long double (np.longdouble [N]^4)."""
        N = self.nao
        if N > 128:
            raise ValueError("long-double N^4 tensor only for N <= 128 (16 bytes per element)")
        eri = np.zeros((N, N, N, N), dtype=np.longdouble)
        lib().oracle_eri_tensor_ld(*self._args(), ct.c_int(N), ct.c_void_p(eri.ctypes.data))
        return eri

    def eri_tensor_erf(self, omega: float) -> np.ndarray:
        """Full AO tensor of the attenuated operator erf(omega r12)/r12 (omega <= 0: 1/r12)."""
        N = self.nao
        if N > 256:
            raise ValueError("full N^4 tensor only for small systems (N <= 256)")
        eri = np.zeros((N, N, N, N))
        lib().oracle_eri_tensor_erf(*self._args(), ct.c_int(N), ct.c_double(omega), eri.ctypes.data_as(_dp))
        return eri

    def jk_erf(self, T: np.ndarray, omega: float, tau: float = 0.0, Q: np.ndarray | None = None):
        """J, K of erf(omega r12)/r12 over the quartets with Q_ab Q_cd >= tau (Q: Schwarz bounds of 1/r12)."""
        T = np.ascontiguousarray(T, dtype=np.float64)
        if T.ndim == 2:
            T = T[None]
        if Q is None:
            Q = self.schwarz()
        Q = np.ascontiguousarray(Q)
        J = np.zeros_like(T)
        K = np.zeros_like(T)
        nq = ct.c_int64(0)
        npq = ct.c_int64(0)
        lib().oracle_jk_strided_op(*self._args(), ct.c_int(self.nao), ct.c_int(T.shape[0]), T.ctypes.data_as(_dp),
                                   ct.c_double(tau), Q.ctypes.data_as(_dp), ct.c_int(1), ct.c_int(0), ct.c_double(omega),
                                   J.ctypes.data_as(_dp), K.ctypes.data_as(_dp), ct.byref(nq), ct.byref(npq))
        return J, K, nq.value, npq.value

    def eri_pair_block(self, sc: int, sd: int, tau: float = 0.0, Q: np.ndarray | None = None) -> np.ndarray:
        """(mu nu|lam sig) for all mu, nu and the AOs lam, sig of the shell pair (sc, sd): [N][N][nc][nd]."""
        nc, nd = int(ncart(int(self.sh_l[sc]))), int(ncart(int(self.sh_l[sd])))
        out = np.zeros((self.nao, self.nao, nc, nd))
        if Q is None:
            Q = self.schwarz()
        Q = np.ascontiguousarray(Q)
        lib().oracle_eri_pair_block(*self._args(), ct.c_int(self.nao), ct.c_int(sc), ct.c_int(sd), ct.c_double(tau),
                                    Q.ctypes.data_as(_dp), out.ctypes.data_as(_dp))
        return out

    def schwarz(self) -> np.ndarray:
        Q = np.zeros((self.nshells, self.nshells))
        lib().oracle_schwarz(*self._args(), Q.ctypes.data_as(_dp))
        return Q

    def jk(self, T: np.ndarray, tau: float = 0.0, Q: np.ndarray | None = None):
        """Matrix-free J[T], K[T] for T [nvec][N][N]; returns J, K, n_shell_quartets, n_prim_quartets."""
        T = np.ascontiguousarray(T, dtype=np.float64)
        if T.ndim == 2:
            T = T[None]
        nvec, N = T.shape[0], self.nao
        if Q is None:
            Q = self.schwarz()
        Q = np.ascontiguousarray(Q)
        J = np.zeros_like(T)
        K = np.zeros_like(T)
        nq = ct.c_int64(0)
        npq = ct.c_int64(0)
        lib().oracle_jk(*self._args(), ct.c_int(N), ct.c_int(nvec), T.ctypes.data_as(_dp),
                        ct.c_double(tau), Q.ctypes.data_as(_dp), J.ctypes.data_as(_dp),
                        K.ctypes.data_as(_dp), ct.byref(nq), ct.byref(npq))
        return J, K, nq.value, npq.value

    def jk_ld(self, T: np.ndarray, tau: float = 0.0, Q: np.ndarray | None = None):
        """Extended-precision J[T], K[T] (oracle_jk_ld): T [nvec][N][N] as np.longdouble (x87 80-bit); every product
        and sum past the FP64 integral values is long double.  Returns J, K as np.longdouble [nvec][N][N] + counts."""
        assert np.finfo(np.longdouble).nmant >= 63, "needs x87 80-bit long double"
        T = np.asarray(T, dtype=np.longdouble)
        if T.ndim == 2:
            T = T[None]
        nvec, N = T.shape[0], self.nao
        Tt = np.ascontiguousarray(np.transpose(T, (1, 2, 0)))          # [N][N][nvec]
        if Q is None:
            Q = self.schwarz()
        Q = np.ascontiguousarray(Q)
        J = np.zeros_like(Tt)
        K = np.zeros_like(Tt)
        nq = ct.c_int64(0)
        npq = ct.c_int64(0)
        lib().oracle_jk_ld(*self._args(), ct.c_int(N), ct.c_int(nvec), ct.c_void_p(Tt.ctypes.data),
                           ct.c_double(tau), Q.ctypes.data_as(_dp), ct.c_void_p(J.ctypes.data),
                           ct.c_void_p(K.ctypes.data), ct.byref(nq), ct.byref(npq))
        return (np.ascontiguousarray(np.transpose(J, (2, 0, 1))), np.ascontiguousarray(np.transpose(K, (2, 0, 1))),
                nq.value, npq.value)

    def jk_strided(self, T: np.ndarray, tau: float, Q: np.ndarray, stride: int, phase: int = 0):
        """Bounded SAMPLE of jk(): only bra pairs ab with ab % stride == phase.  Returns the partial
        J, K and the shell / primitive quartet counts of the sample (for timing extrapolation only)."""
        T = np.ascontiguousarray(T, dtype=np.float64)
        if T.ndim == 2:
            T = T[None]
        Q = np.ascontiguousarray(Q)
        J = np.zeros_like(T)
        K = np.zeros_like(T)
        nq = ct.c_int64(0)
        npq = ct.c_int64(0)
        lib().oracle_jk_strided(*self._args(), ct.c_int(self.nao), ct.c_int(T.shape[0]),
                                T.ctypes.data_as(_dp), ct.c_double(tau), Q.ctypes.data_as(_dp),
                                ct.c_int(stride), ct.c_int(phase), J.ctypes.data_as(_dp),
                                K.ctypes.data_as(_dp), ct.byref(nq), ct.byref(npq))
        return J, K, nq.value, npq.value

    def jk_samples(self, T: np.ndarray, mu, nu):
        """J[T]_{mu nu}, K[T]_{mu nu} at sampled AO pairs, from the definitions (no screening)."""
        T = np.ascontiguousarray(T, dtype=np.float64)
        if T.ndim == 2:
            T = T[None]
        nvec = T.shape[0]
        assert nvec <= 64
        mu_a, pm = _i(mu)
        nu_a, pn = _i(nu)
        ns = mu_a.shape[0]
        J = np.zeros((ns, nvec))
        K = np.zeros((ns, nvec))
        lib().oracle_jk_samples(*self._args(), ct.c_int(self.nao), ct.c_int(nvec),
                                T.ctypes.data_as(_dp), ct.c_int(ns), pm, pn,
                                J.ctypes.data_as(_dp), K.ctypes.data_as(_dp))
        return J, K


def primitive_eri(centers4, exps4, l4) -> np.ndarray:
    """Un-normalised primitive ERI block (ab|cd) with unit coefficients, for the pins."""
    c, pc = _d(np.asarray(centers4).reshape(4, 3))
    e, pe = _d(exps4)
    l, pl = _i(l4)
    out = np.zeros([int(ncart(int(x))) for x in l])
    lib().oracle_primitive_eri(pc, pe, pl, out.ctypes.data_as(_dp))
    return out


def primitive_eri_erf(centers4, exps4, l4, omega: float) -> np.ndarray:
    """Primitive block of erf(omega r12)/r12 with unit coefficients (omega <= 0: 1/r12), for the pins."""
    c, pc = _d(np.asarray(centers4).reshape(4, 3))
    e, pe = _d(exps4)
    l, pl = _i(l4)
    out = np.zeros([int(ncart(int(x))) for x in l])
    lib().oracle_primitive_eri_erf(pc, pe, pl, ct.c_double(omega), out.ctypes.data_as(_dp))
    return out


def num_threads() -> int:
    return int(lib().oracle_num_threads())
