"""Seeded synthetic workloads (the five BASELINE.json configs and shrunk variants).

This module is the ONLY code shared by the CUDA path and the oracle.  It holds no step of
the method (no FFT, no H apply, no eigensolver): it only evaluates the input recipe of
BASELINE.json `configs` / SURVEY.md §8(d) -- cell, atoms, k, the plane-wave list in the
canonical order (reading C3), V_loc(G) on the FFT grid (C6, C7), the Kleinman-Bylander
projectors beta and D (Eq. 3-4; readings C8, C9) and the start vectors
psi0 (C17) -- and hands them to both sides as plain numpy arrays.

numpy only.  Draw order of the generator is part of the recipe:
positions, then per k-point `re` and `im` of psi0.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Sequence

import numpy as np

A_LOC = 4.0      # Ry, depth parameter of the Gaussian wells (BASELINE.json configs[0])
SIGMA_LOC = 0.8  # bohr
A0_DIAMOND = 10.26

_BASIS8 = np.array(
    [(0, 0, 0), (0, .5, .5), (.5, 0, .5), (.5, .5, 0),
     (.25, .25, .25), (.25, .75, .75), (.75, .25, .75), (.75, .75, .25)], dtype=np.float64)

# (l, r_c, D) channels per atom, reading C9.
_CH4 = ((0, 1.0, 2.0), (1, 1.0, -1.0))
_CH8 = ((0, 1.0, 2.0), (0, 1.4, 0.5), (1, 1.0, -1.0), (1, 1.4, -0.3))

_MP4 = (-0.375, -0.125, 0.125, 0.375)


@dataclasses.dataclass(frozen=True)
class Config:
    index: int
    name: str
    cell: np.ndarray          # [3][3], rows a1 a2 a3 (bohr)
    ecutwfc: float            # Ry
    grid: tuple               # (n1, n2, n3)
    nbands: int
    kpts: tuple               # tuple of fractional k (units of b1 b2 b3)
    channels: tuple
    natom: int
    seed: int


def _diamond_sites(rep: int) -> np.ndarray:
    out = []
    for ix in range(rep):
        for iy in range(rep):
            for iz in range(rep):
                for s in range(8):
                    out.append((np.array([ix, iy, iz], dtype=np.float64) + _BASIS8[s]) * A0_DIAMOND)
    return np.array(out)


def config(c: int) -> Config:
    """The five BASELINE.json configs."""
    g = (0.0, 0.0, 0.0)
    if c == 0:
        return Config(0, "tiny-cubic", np.eye(3) * 10.0, 10.0, (24, 24, 24), 8, (g,), _CH4, 2, 1000)
    if c == 1:
        return Config(1, "Si64-like", np.eye(3) * 20.52, 40.0, (96, 96, 96), 160, (g,), _CH8, 64, 1001)
    if c == 2:
        ks = tuple((a, b, d) for a in _MP4 for b in _MP4 for d in _MP4)  # kx slowest, kz fastest (C15)
        return Config(2, "diamond8-4x4x4", np.eye(3) * 10.26, 60.0, (54, 54, 54), 32, ks, _CH8, 8, 1002)
    if c == 3:
        return Config(3, "Si216-like", np.eye(3) * 30.78, 40.0, (128, 128, 128), 520, (g,), _CH8, 216, 1003)
    if c == 4:
        return Config(4, "slab64", np.diag([20.52, 20.52, 61.56]), 40.0, (96, 96, 288), 160, (g,), _CH8, 64, 1004)
    raise ValueError("config index must be 0..4")


def reciprocal(cell: np.ndarray) -> np.ndarray:
    """rows b1 b2 b3 with a_i . b_j = 2 pi delta_ij."""
    return 2.0 * math.pi * np.linalg.inv(cell).T


def pw_list(cell: np.ndarray, k_frac: Sequence[float], ecutwfc: float):
    """Plane waves with |k+G|^2 <= ecutwfc in the canonical order of reading C3
    (m1 slowest, m3 fastest, each ascending).  Returns (miller[npw][3] int32, g2[npw], q[npw][3])."""
    cell = np.asarray(cell, dtype=np.float64)
    b = reciprocal(cell)
    k = np.asarray(k_frac, dtype=np.float64)
    kc = k @ b
    rmax = math.sqrt(ecutwfc) + float(np.linalg.norm(kc))
    M = [int(math.floor(rmax * np.linalg.norm(cell[i]) / (2 * math.pi))) + 1 for i in range(3)]
    m1, m2, m3 = np.meshgrid(*[np.arange(-Mi, Mi + 1) for Mi in M], indexing="ij")
    m = np.stack([m1.ravel(), m2.ravel(), m3.ravel()], axis=1)
    q = (m + k) @ b
    g2 = np.einsum("ij,ij->i", q, q)
    keep = g2 <= ecutwfc
    return m[keep].astype(np.int32), g2[keep].copy(), q[keep].copy()


def _signed(n: int) -> np.ndarray:
    i = np.arange(n)
    return np.where(i > n // 2, i - n, i)  # index n/2 (even n) -> +n/2; V is zero there anyway


def vloc_g(cell, tau, grid, gcut2: float) -> np.ndarray:
    """V_loc(G) = -(A/Omega)(2 pi sigma^2)^{3/2} exp(-sigma^2 G^2/2) sum_a exp(-i G.tau_a) on the FFT
    grid in FFT index order [n1][n2][n3], zero for |G|^2 > gcut2 (readings C6, C7)."""
    cell = np.asarray(cell, dtype=np.float64)
    b = reciprocal(cell)
    omega = abs(np.linalg.det(cell))
    frac = np.asarray(tau) @ np.linalg.inv(cell)           # tau = frac @ cell
    ms = [_signed(n) for n in grid]
    ph = [np.exp(-2j * math.pi * np.outer(frac[:, i], ms[i])) for i in range(3)]  # [natom][n_i]
    sfac = np.einsum("ax,ay,az->xyz", ph[0], ph[1], ph[2], optimize=True)
    G = (ms[0][:, None, None, None] * b[0] + ms[1][None, :, None, None] * b[1]
         + ms[2][None, None, :, None] * b[2])
    G2 = np.einsum("xyzc,xyzc->xyz", G, G)
    pref = -(A_LOC / omega) * (2 * math.pi * SIGMA_LOC ** 2) ** 1.5
    v = pref * np.exp(-0.5 * SIGMA_LOC ** 2 * G2) * sfac
    v[G2 > gcut2] = 0.0
    return np.ascontiguousarray(v, dtype=np.complex128)


def projectors(cell, tau, channels, q: np.ndarray):
    """beta[P][npw], proj_offset[natom+1], D (concatenated per-atom symmetric blocks).
    beta_lm(q) = Omega^{-1/2} |q|^l exp(-r_c^2 q^2/2) Y_lm(q^) exp(-i q.tau_a); real harmonics,
    |q| Y_1m = sqrt(3/4pi) (q_y, q_z, q_x) for m=-1,0,1 (reading C8)."""
    omega = abs(np.linalg.det(np.asarray(cell)))
    q2 = np.einsum("ij,ij->i", q, q)
    y00 = 1.0 / math.sqrt(4 * math.pi)
    y1 = math.sqrt(3.0 / (4 * math.pi))
    per_atom = sum(2 * l + 1 for l, _, _ in channels)
    natom = len(tau)
    beta = np.empty((natom * per_atom, q.shape[0]), dtype=np.complex128)
    dvals = []
    for l, rc, d in channels:
        dvals += [d] * (2 * l + 1)
    Dblk = np.diag(np.array(dvals, dtype=np.float64))
    D = np.tile(Dblk.ravel(), natom)
    row = 0
    for a in range(natom):
        phase = np.exp(-1j * (q @ np.asarray(tau[a]))) / math.sqrt(omega)
        for l, rc, d in channels:
            rad = np.exp(-0.5 * rc * rc * q2)
            if l == 0:
                beta[row] = (y00 * rad) * phase
                row += 1
            else:
                for comp in (1, 2, 0):  # m = -1, 0, 1  ->  q_y, q_z, q_x
                    beta[row] = (y1 * rad * q[:, comp]) * phase
                    row += 1
    off = np.arange(natom + 1, dtype=np.int32) * per_atom
    return beta, off, D


def positions(cfg: Config, rng: np.random.Generator) -> np.ndarray:
    c = cfg.index
    if c == 0:
        return rng.uniform(0, 10.0, size=(2, 3))
    if c == 2:
        return _diamond_sites(1)
    rep = 3 if c == 3 else 2
    sites = _diamond_sites(rep)
    return sites + rng.uniform(-0.05, 0.05, size=sites.shape)


@dataclasses.dataclass
class Problem:
    cfg: Config
    k_index: int
    cell: np.ndarray
    k_frac: np.ndarray
    ecutwfc: float
    grid: np.ndarray          # int32[3]
    tau: np.ndarray
    miller: np.ndarray        # int32[npw][3]
    g2: np.ndarray
    vloc_g: np.ndarray        # complex128 [n1][n2][n3]
    beta: np.ndarray          # complex128 [P][npw]
    proj_offset: np.ndarray   # int32[natom+1]
    D: np.ndarray             # float64, concatenated blocks
    psi0: np.ndarray          # complex128 [nbands][npw]
    nbands: int

    @property
    def npw(self) -> int:
        return int(self.miller.shape[0])

    @property
    def nproj(self) -> int:
        return int(self.beta.shape[0])

    @property
    def natom(self) -> int:
        return int(self.tau.shape[0])


def make_problem(c: int, k_index: int = 0, *, ecutwfc: Optional[float] = None,
                 grid: Optional[Sequence[int]] = None, nbands: Optional[int] = None,
                 with_beta: bool = True, with_vloc: bool = True,
                 vloc_scale: float = 1.0) -> Problem:
    """Problem `k_index` of config `c`.  ecutwfc / grid / nbands override the config to give the
    *shrunk variants* (same cell, atoms, projector channels and k).  The
    generator stream is positions -> (re, im) for k=0 -> (re, im) for k=1 ..., so a problem's psi0
    depends on the sizes of the k-points before it, exactly as in the recipe."""
    cfg = config(c)
    ecut = cfg.ecutwfc if ecutwfc is None else float(ecutwfc)
    grd = tuple(cfg.grid if grid is None else grid)
    nb = cfg.nbands if nbands is None else int(nbands)
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    tau = positions(cfg, rng)
    psi0 = None
    for ik in range(k_index + 1):
        m, g2, q = pw_list(cfg.cell, cfg.kpts[ik], ecut)
        re = rng.standard_normal((nb, m.shape[0]))
        im = rng.standard_normal((nb, m.shape[0]))
        if ik == k_index:
            psi0 = (re + 1j * im) / (1.0 + g2)
    if with_vloc:
        v = vloc_g(cfg.cell, tau, grd, 4.0 * ecut) * vloc_scale
    else:
        v = np.zeros(grd, dtype=np.complex128)
    if with_beta:
        beta, off, D = projectors(cfg.cell, tau, cfg.channels, q)
    else:
        beta = np.zeros((0, m.shape[0]), dtype=np.complex128)
        off = np.zeros(1, dtype=np.int32)
        D = np.zeros(0, dtype=np.float64)
    return Problem(cfg, k_index, np.ascontiguousarray(cfg.cell, dtype=np.float64),
                   np.array(cfg.kpts[k_index], dtype=np.float64), ecut,
                   np.array(grd, dtype=np.int32), tau, m, g2, v, np.ascontiguousarray(beta),
                   off, D, np.ascontiguousarray(psi0), nb)


# Shrunk variants used by the brute-force Davidson pins and GPU parity tests: same cell, atoms,
# projectors, k as the parent config; ecutwfc lowered so npw <~ 1500; smallest supported
# alias-free grid (n_i > 2 m_psi,i + m_V,i and n_i > 2 m_V,i, m_V,i = floor(2 sqrt(ecut) |a_i| / 2 pi)).
SHRUNK = {
    "s1": dict(c=1, ecutwfc=4.7, grid=(32, 32, 32), nbands=23),
    "s2": dict(c=2, k_index=21, ecutwfc=18.0, grid=(32, 32, 32), nbands=10),   # k != 0
    "s3": dict(c=3, ecutwfc=2.1, grid=(32, 32, 32), nbands=19),
    "s4": dict(c=4, ecutwfc=1.85, grid=(18, 18, 64), nbands=22),               # non-cubic
}


def make_shrunk(name: str, **kw) -> Problem:
    d = dict(SHRUNK[name])
    d.update(kw)
    c = d.pop("c")
    k_index = d.pop("k_index", 0)
    return make_problem(c, k_index, **d)
