"""Thin ctypes binding of librttda.so: argument marshalling only, same names as include/rttda.h.

PyTorch is used by callers for device memory and streams; this module passes raw pointers.  There is
no CPU fallback: if the library cannot be loaded, or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as ct
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librttda.so")
_lib = None

INFO = dict(npairs_total=0, npairs_kept=1, nquartets=2, nprim_quartets=3, nquartets_eval=4,
            nprim_eval=5, flops_eval=6, flops_digest_per_vec=7, jk_launches=8, kernel_launches=9,
            create_ms=10, qmax=11, nvec_chunk=12, eri_buf_bytes=13, eri_all_bytes=14)
OPT_INCORE = 1
OPT_GRAPH = 2
OPT_CX_LR = 3
OPT_RS_OMEGA = 4
FIELD_CONTINUE = 1
PULSE = dict(none=0, delta=1, cw=2, tl=3, chirp=4, sin2=5)
EXPORTS = ["rttda_overlap", "rttda_dipole_ao", "rttda_create", "rttda_destroy", "rttda_sigma",
           "rttda_sigma_host", "rttda_fock", "rttda_fock_static", "rttda_propagate", "rttda_propagate_sso", "rttda_propagate_host",
           "rttda_get_info", "rttda_set_option", "rttda_populations", "rttda_spectrum", "rttda_lanczos", "rttda_eigs", "rttda_last_timings", "rttda_jk_time", "rttda_profile_pass", "rttda_gemm_f64", "rttda_fp64_peak", "rttda_last_error",
           "rttda_version"]


class RttdaError(RuntimeError):
    pass


class ShellT(ct.Structure):
    _fields_ = [("center", ct.c_int32), ("l", ct.c_int32), ("nprim", ct.c_int32), ("prim_off", ct.c_int32)]


class BasisT(ct.Structure):
    _fields_ = [("centers", ct.POINTER(ct.c_double)), ("ncenters", ct.c_int32), ("nshells", ct.c_int32),
                ("shells", ct.POINTER(ShellT)), ("exps", ct.POINTER(ct.c_double)),
                ("coefs", ct.POINTER(ct.c_double))]


class FieldT(ct.Structure):
    _fields_ = [("type", ct.c_int32), ("flags", ct.c_int32), ("E0", ct.c_double), ("omega", ct.c_double),
                ("t0", ct.c_double), ("sigma", ct.c_double), ("beta", ct.c_double), ("T_env", ct.c_double),
                ("dir", ct.c_double * 3)]


def lib():
    """Load librttda.so (fails loudly if it was not built: run paper_2601_16949_b200/build.py)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RttdaError("librttda.so is missing (%s); build it with __graft_entry__.build() -- "
                             "there is no fallback path" % LIB_PATH)
        L = ct.CDLL(LIB_PATH)
        L.rttda_last_error.restype = ct.c_char_p
        L.rttda_version.restype = ct.c_char_p
        for name in EXPORTS:
            getattr(L, name)
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise RttdaError("%s failed (%d): %s" % (what, rc, lib().rttda_last_error().decode()))


def _dptr(x):
    """Device or host pointer from a torch tensor, numpy array or int."""
    if x is None:
        return ct.c_void_p(0)
    if isinstance(x, int):
        return ct.c_void_p(x)
    if isinstance(x, np.ndarray):
        assert x.dtype == np.float64 and x.flags.c_contiguous
        return ct.c_void_p(x.ctypes.data)
    assert x.dtype.is_floating_point and x.element_size() == 8 and x.is_contiguous()
    return ct.c_void_p(x.data_ptr())


def _stream(stream):
    if stream is None:
        return ct.c_void_p(0)
    if isinstance(stream, int):
        return ct.c_void_p(stream)
    return ct.c_void_p(stream.cuda_stream)


class _BasisHolder:
    def __init__(self, basis):
        self.centers = np.ascontiguousarray(basis.centers, dtype=np.float64)
        self.exps = np.ascontiguousarray(basis.exps, dtype=np.float64)
        self.coefs = np.ascontiguousarray(basis.coefs, dtype=np.float64)
        n = int(basis.sh_l.shape[0])
        self.shells = (ShellT * n)()
        for s in range(n):
            self.shells[s] = ShellT(int(basis.sh_center[s]), int(basis.sh_l[s]), int(basis.sh_nprim[s]),
                                    int(basis.sh_off[s]))
        dp = ct.POINTER(ct.c_double)
        self.c = BasisT(self.centers.ctypes.data_as(dp), int(self.centers.shape[0]), n, self.shells,
                        self.exps.ctypes.data_as(dp), self.coefs.ctypes.data_as(dp))
        _l = np.asarray(basis.sh_l, dtype=np.int64)
        self.nao = int(np.sum((_l + 1) * (_l + 2) // 2))


def make_field(f: dict) -> FieldT:
    d = f.get("dir", (0.0, 0.0, 1.0))
    return FieldT(PULSE[f.get("type", "none")], FIELD_CONTINUE if f.get("continue") else 0, float(f.get("E0", 0.0)), float(f.get("omega") or 0.0),
                  float(f.get("t0", 0.0)), float(f.get("sigma", 1.0)), float(f.get("beta", 0.0)),
                  float(f.get("T_env", 0.0)), (ct.c_double * 3)(*[float(x) for x in d]))


def rttda_overlap(basis) -> np.ndarray:
    b = _BasisHolder(basis)
    S = np.zeros((b.nao, b.nao))
    _check(lib().rttda_overlap(ct.byref(b.c), b.nao, _dptr(S)), "rttda_overlap")
    return S


def rttda_dipole_ao(basis) -> np.ndarray:
    b = _BasisHolder(basis)
    D = np.zeros((3, b.nao, b.nao))
    _check(lib().rttda_dipole_ao(ct.byref(b.c), b.nao, _dptr(D)), "rttda_dipole_ao")
    return D


def rttda_fp64_peak(seconds: float = 1.0, stream=None) -> float:
    out = ct.c_double(0.0)
    _check(lib().rttda_fp64_peak(ct.c_double(seconds), ct.byref(out), _stream(stream)), "rttda_fp64_peak")
    return out.value


def rttda_gemm_f64(M, N, K, batch, alpha, A, sa, B, sb, beta, C, sc, stream=None):
    """C = alpha A B + beta C, strided batched (include/rttda.h); sa = (sam, sak, sabatch), sb = (sbk, sbn, sbbatch),
    sc = (scm, scn, scbatch) in doubles; A, B, C CUDA tensors (any shape: only the base pointer is used)."""
    i64 = ct.c_int64
    _check(lib().rttda_gemm_f64(int(M), int(N), int(K), int(batch), ct.c_double(alpha), ct.c_void_p(A.data_ptr()),
                                i64(sa[0]), i64(sa[1]), i64(sa[2]), ct.c_void_p(B.data_ptr()), i64(sb[0]), i64(sb[1]),
                                i64(sb[2]), ct.c_double(beta), ct.c_void_p(C.data_ptr()), i64(sc[0]), i64(sc[1]),
                                i64(sc[2]), _stream(stream)), "rttda_gemm_f64")
    return C


def rttda_spectrum(R0, log, dt: float, pad: int, omega, intensity, stream=None):
    """eq. 21 / 23: log CUDA [n][ntraj][3] (rttda_propagate's log), R0 host [ntraj][2]; omega CUDA [nout],
    intensity CUDA [ntraj + 1][nout], nout = (2n + 1 + pad) // 2."""
    R0 = np.ascontiguousarray(R0, dtype=np.float64)
    ntraj = int(R0.shape[0])
    n = 0 if log is None else int(log.shape[0])
    _check(lib().rttda_spectrum(ntraj, n, _dptr(R0), _dptr(log), ct.c_double(dt), int(pad), int(omega.shape[0]),
                                _dptr(omega), _dptr(intensity), _stream(stream)), "rttda_spectrum")
    return omega, intensity


class Rttda:
    """Handle wrapper.  C_occ / C_virt are CUDA float64 torch tensors [nao][nocc], [nao][nvirt]."""

    def __init__(self, basis, C_occ, C_virt, eps, cx: float = 1.0, tau: float = 1e-12, stream=None):
        self._h = ct.c_void_p(0)
        b = _BasisHolder(basis)
        self.nao, self.nocc, self.nvirt = b.nao, int(C_occ.shape[1]), int(C_virt.shape[1])
        self.ncsf = self.nocc * self.nvirt
        eps = np.ascontiguousarray(eps, dtype=np.float64)
        assert C_occ.is_cuda and C_virt.is_cuda, "C_occ / C_virt must be CUDA tensors (no CPU path)"
        _check(lib().rttda_create(ct.byref(self._h), ct.byref(b.c), self.nao, self.nocc, self.nvirt,
                                  _dptr(C_occ.contiguous()), _dptr(C_virt.contiguous()), _dptr(eps),
                                  ct.c_double(cx), ct.c_double(tau), _stream(stream)), "rttda_create")

    def close(self):
        if self._h:
            lib().rttda_destroy(self._h)
            self._h = ct.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def rttda_sigma(self, X, sigma, stream=None):
        nvec = int(X.shape[0])
        _check(lib().rttda_sigma(self._h, nvec, _dptr(X), _dptr(sigma), _stream(stream)), "rttda_sigma")
        return sigma

    def rttda_sigma_host(self, X: np.ndarray, sigma: np.ndarray, stream=None):
        _check(lib().rttda_sigma_host(self._h, int(X.shape[0]), _dptr(X), _dptr(sigma), _stream(stream)),
               "rttda_sigma_host")
        return sigma

    def rttda_fock(self, T, F, stream=None):
        _check(lib().rttda_fock(self._h, int(T.shape[0]), _dptr(T), _dptr(F), _stream(stream)), "rttda_fock")
        return F

    def rttda_fock_static(self, T, F, stream=None):
        _check(lib().rttda_fock_static(self._h, int(T.shape[0]), _dptr(T), _dptr(F), _stream(stream)), "rttda_fock_static")
        return F

    def _fields(self, fields):
        arr = (FieldT * len(fields))()
        for i, f in enumerate(fields):
            arr[i] = make_field(f)
        return arr

    def rttda_propagate(self, C, fields, t_start, dt, nsteps, log=None, stream=None):
        arr = self._fields(fields)
        _check(lib().rttda_propagate(self._h, len(fields), _dptr(C), arr, ct.c_double(t_start), ct.c_double(dt),
                                     int(nsteps), _dptr(log), _stream(stream)), "rttda_propagate")
        return C

    def rttda_propagate_sso(self, C, fields, t_start, dt, nsteps, log=None, stream=None):
        arr = self._fields(fields)
        _check(lib().rttda_propagate_sso(self._h, len(fields), _dptr(C), arr, ct.c_double(t_start), ct.c_double(dt),
                                         int(nsteps), _dptr(log), _stream(stream)), "rttda_propagate_sso")
        return C

    def rttda_propagate_host(self, C: np.ndarray, fields, t_start, dt, nsteps, log=None, stream=None):
        arr = self._fields(fields)
        _check(lib().rttda_propagate_host(self._h, len(fields), _dptr(C), arr, ct.c_double(t_start),
                                          ct.c_double(dt), int(nsteps), _dptr(log), _stream(stream)),
               "rttda_propagate_host")
        return C

    def rttda_lanczos(self, m: int, v0, V, stream=None):
        """Returns (alpha, beta) as numpy arrays; V (CUDA tensor [m+1][ncsf]) receives the Lanczos vectors."""
        alpha, beta = np.zeros(m), np.zeros(m)
        _check(lib().rttda_lanczos(self._h, int(m), _dptr(v0), _dptr(alpha), _dptr(beta), _dptr(V), _stream(stream)),
               "rttda_lanczos")
        return alpha, beta

    def rttda_eigs(self, k: int, X, nblock: int = 0, tol: float = 1e-8, maxiter: int = 100, stream=None,
                   allow_nonconverged: bool = False):
        """Lowest k eigenpairs of A by block Davidson; X CUDA tensor [k][ncsf] receives the vectors.
        Returns (omega [k], residual norms [k], iterations, sigma vectors built).  RTTDA_ENOCONV raises unless
        allow_nonconverged (the outputs then hold the current Ritz pairs and their residuals)."""
        om, rs = np.zeros(k), np.zeros(k)
        it, ns = ct.c_int32(0), ct.c_int32(0)
        rc = lib().rttda_eigs(self._h, int(k), int(nblock or k), ct.c_double(tol), int(maxiter), _dptr(om), _dptr(X),
                              _dptr(rs), ct.byref(it), ct.byref(ns), _stream(stream))
        if not (allow_nonconverged and rc == -4):
            _check(rc, "rttda_eigs")
        return om, rs, it.value, ns.value

    def rttda_populations(self, C, Xs, P, stream=None):
        _check(lib().rttda_populations(self._h, int(C.shape[0]), _dptr(C), int(Xs.shape[0]), _dptr(Xs), _dptr(P),
                                       _stream(stream)), "rttda_populations")
        return P

    def rttda_set_option(self, option: int, value: float):
        _check(lib().rttda_set_option(self._h, int(option), ct.c_double(value)), "rttda_set_option")

    def rttda_get_info(self, key) -> float:
        out = ct.c_double(0.0)
        k = INFO[key] if isinstance(key, str) else int(key)
        _check(lib().rttda_get_info(self._h, k, ct.byref(out)), "rttda_get_info")
        return out.value

    def rttda_last_timings(self):
        ms = (ct.c_double * 3)()
        _check(lib().rttda_last_timings(self._h, ms), "rttda_last_timings")
        return dict(jk_ms=ms[0], mo2ao_ms=ms[1], ao2mo_ms=ms[2])

    def rttda_jk_time(self):
        s, c = ct.c_double(0.0), ct.c_double(0.0)
        _check(lib().rttda_jk_time(self._h, ct.byref(s), ct.byref(c)), "rttda_jk_time")
        return s.value, int(c.value)

    def rttda_profile_pass(self, nvec: int, stream=None) -> np.ndarray:
        """One extra ERI pass with per-segment CUDA-event timings; rows as documented in include/rttda.h."""
        rows = np.zeros((512, 16))                    # at most 24 x 25 / 2 = 300 segments (6 pair types x 4 contraction sub-classes)
        n = ct.c_int32(0)
        _check(lib().rttda_profile_pass(self._h, int(nvec), _dptr(rows), 512, ct.byref(n), _stream(stream)),
               "rttda_profile_pass")
        return rows[: n.value]

    def info(self) -> dict:
        return {k: self.rttda_get_info(k) for k in INFO}
