"""Seed-generated synthetic molecules, MOs, energies and trial vectors (no method arithmetic).

Recipe = BASELINE.json `configs` (BJ:configs[0..4]) under DESIGN.md readings:
  R11 contraction coefficients d_k ~ U[0.2, 1.0] on normalised primitives (each side renormalises
      the contracted function itself);
  R12 config-4 heavy centre = s(3), s(3), s(1), p(3), p(1) (9 AOs), H-like = s(3), s(1) (2 AOs);
      the d-shell test molecule ("tiny-d", key 6): heavy = s(3), s(1), p(3), p(1), d(1) (14 AOs, Cartesian d);
  R13 box edge L = 8 (n_centres/6)^(1/3) bohr, rejection sampling for the 1.8 bohr minimum;
  R17 trial vectors iid N(0,1), scaled to unit 2-norm;
  R18 C = S^-1/2 Q, Q = sign-fixed QR of an N x N N(0,1) matrix; eps_occ ~ U[-1,-0.3],
      eps_virt ~ U[0.05, 2], each sorted ascending.
Draw order is fixed: centres -> per centre, per shell: exponents then coefficients -> Q -> eps.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

SEED = 260116949


@dataclass
class Basis:
    centers: np.ndarray      # [ncenters][3] float64, bohr
    sh_center: np.ndarray    # [nshells] int32
    sh_l: np.ndarray         # [nshells] int32, 0 = s, 1 = p (x, y, z), 2 = d (xx, xy, xz, yy, yz, zz)
    sh_nprim: np.ndarray     # [nshells] int32
    sh_off: np.ndarray       # [nshells] int32, offset into exps / coefs
    exps: np.ndarray         # [sum nprim] float64
    coefs: np.ndarray        # [sum nprim] float64, multiply NORMALISED primitives (R11)

    @property
    def nshells(self) -> int:
        return int(self.sh_l.shape[0])

    @property
    def ncenters(self) -> int:
        return int(self.centers.shape[0])

    @property
    def nao(self) -> int:
        l = self.sh_l.astype(np.int64)
        return int(np.sum((l + 1) * (l + 2) // 2))

    @property
    def ao_off(self) -> np.ndarray:
        l = self.sh_l.astype(np.int64)
        n = (l + 1) * (l + 2) // 2
        return np.concatenate([[0], np.cumsum(n)[:-1]]).astype(np.int32)


@dataclass
class Config:
    name: str
    n_heavy: int             # centres with the "heavy" shell recipe
    n_h: int                 # H-like centres (config 4/5 only)
    heavy_shells: tuple      # tuple of (l, nprim)
    h_shells: tuple
    nocc: int
    nvirt: int
    tau: float               # Schwarz threshold (R15)
    dt: float
    nsteps: int
    fields: tuple = field(default_factory=tuple)   # tuple of dicts, one per trajectory
    k: int = 0               # 1-based config number (seed offset)
    bump: int = 0            # default re-draw index of make_basis / make_mos (R18: a draw with a too ill-conditioned S is re-drawn)

    @property
    def ncenters(self) -> int:
        return self.n_heavy + self.n_h

    @property
    def box(self) -> float:
        return 8.0 * (self.ncenters / 6.0) ** (1.0 / 3.0)


_SP5 = ((0, 3), (0, 1), (1, 1))                      # BJ:configs[0]: 2 s shells (3, 1 prims) + p(1)
_HEAVY9 = ((0, 3), (0, 3), (0, 1), (1, 3), (1, 1))   # R12
_H2 = ((0, 3), (0, 1))
_SPD15 = ((0, 3), (0, 3), (0, 1), (1, 3), (1, 1), (2, 1))   # 6-31G*-like heavy centre: 3 s + 2 p + 1 Cartesian d shell = 15 BF
_SPD14 = ((0, 3), (0, 1), (1, 3), (1, 1), (2, 1))    # 6-31G*-like heavy centre with one Cartesian d shell (NEXT-4)

CONFIGS = {
    1: Config("tiny", 6, 0, _SP5, (), 5, 25, 1e-12, 0.05, 10,
              ({"type": "cw", "E0": 0.01, "omega": 0.3, "dir": (0.0, 0.0, 1.0)},), 1),
    2: Config("delta-kick", 40, 0, _SP5, (), 40, 160, 1e-12, 0.1, 2000,
              tuple({"type": "delta", "E0": 1e-4, "dir": d} for d in
                    ((1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0))), 2),
    3: Config("rabi", 80, 0, _SP5, (), 80, 320, 1e-12, 0.05, 4000,
              tuple({"type": "cw", "E0": e, "omega": None, "dir": (0.0, 0.0, 1.0)}
                    for e in (0.005, 0.02)), 3),
    4: Config("two-photon", 120, 100, _HEAVY9, _H2, 400, 880, 1e-12, 0.1, 2000,
              tuple({"type": "sin2", "E0": e, "omega": None, "T_env": 200.0,
                     "dir": (0.0, 0.0, 1.0)} for e in (0.01, 0.03, 0.05)), 4),
    5: Config("sigma-microbench", 120, 100, _HEAVY9, _H2, 400, 880, 1e-12, 0.0, 0, (), 4),
    # not a BASELINE.json config: the small d-shell molecule of the NEXT-4 tests (4 heavy centres + 2 H-like, 60 AOs)
    6: Config("tiny-d", 4, 2, _SPD14, _H2, 10, 50, 1e-12, 0.05, 10,
              ({"type": "cw", "E0": 0.01, "omega": 0.3, "dir": (0.0, 0.0, 1.0)},), 6, 2),   # draw 2: cond(S) = 144
    # 320 basis functions with d shells: the size of the paper's smallest Table-3 molecule (320 BF, 6-31G*),
    # 20 heavy centres (14 AOs) + 20 H-like (2 AOs); measurement and parity case of the d-shell path
    7: Config("d-320", 20, 20, _SPD14, _H2, 60, 260, 1e-12, 0.05, 100,
              ({"type": "cw", "E0": 0.01, "omega": 0.3, "dir": (0.0, 0.0, 1.0)},), 7, 1),       # draw 1: cond(S) = 1.9e3
    # the SHAPE of the paper's largest molecule (Table 3: F-Coronene C108 H42 N12, 120 heavy atoms x 15 BF +
    # 42 H x 2 BF = 1884 BF, 387 occupied orbitals); synthetic centres and exponents as everywhere
    8: Config("d-1884", 120, 42, _SPD15, _H2, 387, 1497, 1e-12, 0.1, 0,
              ({"type": "cw", "E0": 0.01, "omega": 0.3, "dir": (0.0, 0.0, 1.0)},), 8, 2),   # draw 2: cond(S) = 5.5e4
}


def get_config(k: int) -> Config:
    return CONFIGS[k]


def _rng(k: int, stream: int, bump: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED + 10 * k + stream + 1000 * bump))


def _place_centers(rng: np.random.Generator, n: int, L: float, dmin: float = 1.8) -> np.ndarray:
    pts = np.zeros((n, 3))
    m = 0
    while m < n:
        c = rng.uniform(0.0, L, size=3)
        if m == 0 or np.min(np.linalg.norm(pts[:m] - c, axis=1)) >= dmin:
            pts[m] = c
            m += 1
    return pts


def make_basis(cfg: Config, bump: int | None = None) -> Basis:
    """Centres, shell table, exponents and coefficients of config `cfg` (seed stream 0)."""
    bump = cfg.bump if bump is None else bump
    rng = _rng(cfg.k, 0, bump)
    n = cfg.ncenters
    centers = _place_centers(rng, n, cfg.box)
    # heavy and H-like centres mixed uniformly (R13): a seeded permutation decides which is which
    kinds = np.zeros(n, dtype=np.int32)
    if cfg.n_h:
        kinds[rng.permutation(n)[: cfg.n_h]] = 1
    sh_center, sh_l, sh_nprim, exps, coefs = [], [], [], [], []
    for c in range(n):
        for (l, nprim) in (cfg.h_shells if kinds[c] else cfg.heavy_shells):
            lo, hi = (0.1, 20.0) if l == 0 else ((0.2, 2.0) if l == 1 else (0.3, 1.5))
            e = np.exp(rng.uniform(np.log(lo), np.log(hi), size=nprim))
            d = rng.uniform(0.2, 1.0, size=nprim)
            sh_center.append(c)
            sh_l.append(l)
            sh_nprim.append(nprim)
            exps.extend(e.tolist())
            coefs.extend(d.tolist())
    sh_nprim = np.asarray(sh_nprim, dtype=np.int32)
    sh_off = np.concatenate([[0], np.cumsum(sh_nprim)[:-1]]).astype(np.int32)
    return Basis(np.ascontiguousarray(centers), np.asarray(sh_center, dtype=np.int32),
                 np.asarray(sh_l, dtype=np.int32), sh_nprim, sh_off,
                 np.asarray(exps, dtype=np.float64), np.asarray(coefs, dtype=np.float64))


def orthonormalizer(S: np.ndarray):
    """S^-1/2 by symmetric eigendecomposition, plus cond(S) (R18). S is an input."""
    w, U = np.linalg.eigh(S)
    if w[0] <= 0:
        raise ValueError("overlap matrix not positive definite")
    return (U / np.sqrt(w)) @ U.T, float(w[-1] / w[0])


def make_mos(cfg: Config, S: np.ndarray, bump: int | None = None):
    """Synthetic MOs C = S^-1/2 Q (seed stream 1) and orbital energies (seed stream 2).

    Returns (C_occ [N][nocc], C_virt [N][nvirt], eps [nocc+nvirt], cond(S)).  The caller rejects
    cond(S) > 1e5 by re-drawing the basis with bump+1 (recorded in its output).
    """
    N = S.shape[0]
    assert N == cfg.nocc + cfg.nvirt
    bump = cfg.bump if bump is None else bump
    X, cond = orthonormalizer(S)
    g = _rng(cfg.k, 1, bump).standard_normal((N, N))
    Q, R = np.linalg.qr(g)
    Q = Q * np.sign(np.diag(R))
    C = X @ Q
    r2 = _rng(cfg.k, 2, bump)
    eo = np.sort(r2.uniform(-1.0, -0.3, size=cfg.nocc))
    ev = np.sort(r2.uniform(0.05, 2.0, size=cfg.nvirt))
    return (np.ascontiguousarray(C[:, : cfg.nocc]), np.ascontiguousarray(C[:, cfg.nocc:]),
            np.concatenate([eo, ev]), cond)


def make_vectors(cfg: Config, nvec: int, stream: int = 3) -> np.ndarray:
    """nvec iid-Gaussian unit-norm real trial vectors [nvec][nocc*nvirt] (R17)."""
    x = _rng(cfg.k, stream).standard_normal((nvec, cfg.nocc * cfg.nvirt))
    return x / np.linalg.norm(x, axis=1, keepdims=True)
