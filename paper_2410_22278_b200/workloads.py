"""Seeded synthetic workloads (BASELINE.json `configs`).

This module is shared by the oracle tests and by the CUDA harness.  It is DATA
only: geometry, exponents, coefficients, seeds.  It contains none of the
method's arithmetic (no integrals, no overlap matrix, no Ewald sums): anything
that needs the crystalline overlap S takes S as an argument.

The paper measures on def2-SVP ice XI / Si / ZnO / benzene cells (PAPER.md
L849, L880, L900).  Neither the basis tables nor the geometries are available
here, so the five seeded cells below stand in for them ("Input
recipe").
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional

import numpy as np

_DFACT = {0: 1.0, 1: 1.0, 2: 3.0}  # (2l-1)!!


@dataclasses.dataclass
class Workload:
    name: str
    cell: np.ndarray          # (3,3) rows a1,a2,a3 in bohr
    xyz: np.ndarray           # (natom,3) bohr
    sh_atom: np.ndarray       # (nshell,) int32
    sh_l: np.ndarray          # (nshell,) int32, 0/1/2
    sh_nprim: np.ndarray      # (nshell,) int32
    sh_off: np.ndarray        # (nshell,) int32 offset into exps/coefs
    exps: np.ndarray          # (nprim_total,)
    coefs: np.ndarray         # (nprim_total,) multiply eq-6-normalised primitives
    omega: float
    n_occ: int
    seed: int
    r_cut: float = 0.0        # 0 => derive from thresholds
    g_cut: float = 0.0
    tau_schwarz: float = 1e-13
    elements: Optional[List[str]] = None

    @property
    def nshell(self) -> int:
        return int(self.sh_l.shape[0])

    @property
    def natom(self) -> int:
        return int(self.xyz.shape[0])

    @property
    def nbf(self) -> int:
        return int(sum((l + 1) * (l + 2) // 2 for l in self.sh_l))

    def shell_offsets(self) -> np.ndarray:
        """AO offset of each shell (AO order = shells in input order, C-10)."""
        n = np.array([(l + 1) * (l + 2) // 2 for l in self.sh_l], dtype=np.int64)
        return np.concatenate([[0], np.cumsum(n)])[:-1]

    def orbitals_seed(self) -> np.ndarray:
        """C0 ~ N(0,1)^{N x n_occ} (C-19); orthonormalise with density_from_orbitals."""
        rng = np.random.default_rng(self.seed + 7919)
        return rng.standard_normal((self.nbf, self.n_occ))


def orthonormal_orbitals(C0: np.ndarray, S: np.ndarray) -> np.ndarray:
    """C = C0 (C0^T S C0)^(-1/2): seeded orbitals orthonormalised under the overlap matrix (SURVEY C-19)."""
    M = C0.T @ S @ C0
    M = 0.5 * (M + M.T)
    w, V = np.linalg.eigh(M)
    if w.min() <= 0:
        raise ValueError("C0^T S C0 is not positive definite")
    return C0 @ (V * (1.0 / np.sqrt(w))) @ V.T


def density_from_orbitals(C0: np.ndarray, S: np.ndarray) -> np.ndarray:
    """P = C C^T with C = C0 (C0^T S C0)^(-1/2)  (SURVEY C-19, tr(PS) = n_occ).

    Plain linear algebra on inputs; S comes from the caller (oracle S in the
    tests, the library's own S in bench.py).
    """
    C = orthonormal_orbitals(C0, S)
    P = C @ C.T
    return 0.5 * (P + P.T)


# ----------------------------------------------------------------------------
# basis helpers (data recipe only)
# ----------------------------------------------------------------------------

def _contracted_scale(l: int, exps: np.ndarray, coefs: np.ndarray) -> np.ndarray:
    """Scale coefficients so the axis-aligned component (s, p_x, d_xx) of the
    contracted shell has unit LOCAL self-overlap (C-9).  For unit-normalised
    primitives <i|j> = (2 sqrt(a_i a_j)/(a_i+a_j))^(l+3/2) (textbook)."""
    a = exps[:, None]
    b = exps[None, :]
    ov = (2.0 * np.sqrt(a * b) / (a + b)) ** (l + 1.5)
    nrm = float(coefs @ ov @ coefs)
    return coefs / math.sqrt(nrm)


def _log_uniform_sorted(rng, n: int, lo: float, hi: float, min_ratio: float) -> np.ndarray:
    """n exponents log-uniform in [lo,hi], descending, adjacent ratio >= min_ratio."""
    if n == 0:
        return np.zeros(0)
    span = math.log(hi / lo)
    max_ratio_feasible = math.exp(span / max(n - 1, 1)) if n > 1 else float("inf")
    ratio = min(min_ratio, 0.8 * max_ratio_feasible + 0.2) if n > 1 else min_ratio
    for _ in range(100000):
        e = np.sort(np.exp(rng.uniform(math.log(lo), math.log(hi), size=n)))[::-1]
        if n == 1 or np.all(e[:-1] / e[1:] >= ratio):
            return e
    raise RuntimeError("could not draw exponents")


class _Basis:
    """Per-element shell list: [(l, exps, coefs)]"""

    def __init__(self):
        self.shells: Dict[str, list] = {}

    def add(self, el: str, l: int, exps, coefs):
        exps = np.asarray(exps, dtype=np.float64)
        coefs = _contracted_scale(l, exps, np.asarray(coefs, dtype=np.float64))
        self.shells.setdefault(el, []).append((l, exps, coefs))


def _deal(rng, basis: _Basis, el: str, l: int, nprims: List[int], lo: float, hi: float,
          min_ratio: float):
    """Draw sum(nprims) exponents, sort descending and deal consecutive bands to
    the shells (tightest band first), coefficients uniform [0.2,1]."""
    e = _log_uniform_sorted(rng, int(sum(nprims)), lo, hi, min_ratio)
    k = 0
    for n in nprims:
        c = rng.uniform(0.2, 1.0, size=n)
        basis.add(el, l, e[k:k + n], c)
        k += n


def _assemble(name, cell, xyz, elements, basis: _Basis, **kw) -> Workload:
    sh_atom, sh_l, sh_nprim, sh_off, exps, coefs = [], [], [], [], [], []
    off = 0
    for ia, el in enumerate(elements):
        for (l, e, c) in basis.shells[el]:
            sh_atom.append(ia)
            sh_l.append(l)
            sh_nprim.append(len(e))
            sh_off.append(off)
            exps.extend(e.tolist())
            coefs.extend(c.tolist())
            off += len(e)
    return Workload(
        name=name, cell=np.asarray(cell, dtype=np.float64),
        xyz=np.ascontiguousarray(xyz, dtype=np.float64),
        sh_atom=np.asarray(sh_atom, dtype=np.int32), sh_l=np.asarray(sh_l, dtype=np.int32),
        sh_nprim=np.asarray(sh_nprim, dtype=np.int32), sh_off=np.asarray(sh_off, dtype=np.int32),
        exps=np.asarray(exps, dtype=np.float64), coefs=np.asarray(coefs, dtype=np.float64),
        elements=list(elements), **kw)


# ----------------------------------------------------------------------------
# geometry helpers
# ----------------------------------------------------------------------------

_SHIFTS = np.array([[i, j, k] for i in (-1, 0, 1) for j in (-1, 0, 1) for k in (-1, 0, 1)], dtype=np.float64)


def _min_image_dists(cell: np.ndarray, a: np.ndarray, pts: np.ndarray) -> np.ndarray:
    """Minimum-image distances (C-21) from point a to every row of pts."""
    if pts.shape[0] == 0:
        return np.zeros(0)
    inv = np.linalg.inv(cell)
    d = (a[None, :] - pts) @ inv
    d -= np.round(d)
    v = (d[:, None, :] + _SHIFTS[None, :, :]) @ cell            # (n, 27, 3)
    return np.sqrt((v * v).sum(-1)).min(axis=1)


def _min_image_dist(cell: np.ndarray, a: np.ndarray, b: np.ndarray) -> float:
    return float(_min_image_dists(cell, a, b[None, :])[0])


def _random_rotation(rng) -> np.ndarray:
    q = rng.standard_normal(4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def _water_box(rng, L: float, nmol: int, min_oo: float):
    """Rigid waters (O-H 1.81 bohr, H-O-H 104.5 deg), uniform random
    orientation, O positions by rejection on minimum-image O-O distance.
    Uses a jittered grid start when random insertion stalls (dense boxes)."""
    cell = np.eye(3) * L
    half = math.radians(104.5) / 2.0
    h1 = 1.81 * np.array([math.sin(half), 0.0, math.cos(half)])
    h2 = 1.81 * np.array([-math.sin(half), 0.0, math.cos(half)])
    O: List[np.ndarray] = []
    # jittered lattice sites guarantee termination for liquid-like densities
    ng = int(math.ceil(nmol ** (1.0 / 3.0)))
    sites = [(i, j, k) for i in range(ng) for j in range(ng) for k in range(ng)]
    order = rng.permutation(len(sites))
    a = L / ng
    max_jit = max(0.0, 0.5 * (a - min_oo))
    for idx in order[:nmol]:
        i, j, k = sites[idx]
        base = (np.array([i, j, k]) + 0.5) * a
        for _ in range(1000):
            pos = base + rng.uniform(-1, 1, size=3) * (max_jit + 0.35 * a)
            pos = pos % L
            if not O or _min_image_dists(cell, pos, np.array(O)).min() >= min_oo:
                O.append(pos)
                break
        else:
            pos = base % L
            O.append(pos)
    xyz, el = [], []
    for o in O:
        Rm = _random_rotation(rng)
        xyz += [o, o + Rm @ h1, o + Rm @ h2]
        el += ["O", "H", "H"]
    return cell, np.array(xyz), el


def _water_basis(rng, with_d: bool, with_hp: bool) -> _Basis:
    """Config-2 recipe (C-18): O 3 s shells x 3 prims in [0.2,5000]; O p shells
    3+1 prims in [0.15,30]; H s shells 3+1 prims in [0.12,20]; optional O d(0.8)
    and H p(0.8).  One exponent set per element."""
    b = _Basis()
    _deal(rng, b, "O", 0, [3, 3, 3], 0.2, 5000.0, 1.8)
    _deal(rng, b, "O", 1, [3, 1], 0.15, 30.0, 1.8)
    if with_d:
        b.add("O", 2, [0.8], [1.0])
    _deal(rng, b, "H", 0, [3, 1], 0.12, 20.0, 1.8)
    if with_hp:
        b.add("H", 1, [0.8], [1.0])
    return b


# ----------------------------------------------------------------------------
# the five configs
# ----------------------------------------------------------------------------

SEEDS = {"tiny": 1001, "water8": 1002, "si64": 1003, "water64": 1004, "water343": 1005}


def tiny(seed: int = SEEDS["tiny"], omega: float = 0.4) -> Workload:
    """Config 1: cubic L=8, 4 centres (min sep 1.5), two uncontracted s (3.0, 0.5)."""
    rng = np.random.default_rng(seed)
    L = 8.0
    cell = np.eye(3) * L
    pts: List[np.ndarray] = []
    while len(pts) < 4:
        p = rng.uniform(0, L, size=3)
        if all(_min_image_dist(cell, p, q) >= 1.5 for q in pts):
            pts.append(p)
    b = _Basis()
    b.add("X", 0, [3.0], [1.0])
    b.add("X", 0, [0.5], [1.0])
    return _assemble("tiny", cell, np.array(pts), ["X"] * 4, b, omega=omega, n_occ=2,
                     seed=seed, r_cut=30.0, g_cut=6.0)


def water8(seed: int = SEEDS["water8"], omega: float = 0.35) -> Workload:
    """Config 2: cubic L=18.6, 8 waters (min O-O 4.5), s,p basis, n_occ=40."""
    rng = np.random.default_rng(seed)
    cell, xyz, el = _water_box(rng, 18.6, 8, 4.5)
    b = _water_basis(rng, with_d=False, with_hp=False)
    return _assemble("water8", cell, xyz, el, b, omega=omega, n_occ=40, seed=seed)


def si64(seed: int = SEEDS["si64"], omega: float = 0.3) -> Workload:
    """Config 3: diamond lattice, 2x2x2 conventional cells (a=10.26), ideal
    positions; 3s 2p 1d per atom, exponents in [0.1,1500], 1-6 prims/shell."""
    rng = np.random.default_rng(seed)
    a = 10.26
    fcc = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]])
    basis8 = np.concatenate([fcc, fcc + 0.25])
    xyz = []
    for i in range(2):
        for j in range(2):
            for k in range(2):
                xyz.append((basis8 + np.array([i, j, k])) * a)
    xyz = np.concatenate(xyz)
    cell = np.eye(3) * (2 * a)
    b = _Basis()
    ns = [int(rng.integers(1, 7)) for _ in range(3)]
    np_ = [int(rng.integers(1, 7)) for _ in range(2)]
    nd = [int(rng.integers(1, 7))]
    ns.sort(reverse=True); np_.sort(reverse=True)
    _deal(rng, b, "Si", 0, ns, 0.1, 1500.0, 2.0)
    _deal(rng, b, "Si", 1, np_, 0.1, 1500.0, 2.0)
    _deal(rng, b, "Si", 2, nd, 0.1, 1500.0, 2.0)
    return _assemble("si64", cell, xyz, ["Si"] * 64, b, omega=omega, n_occ=128, seed=seed)


def water64(seed: int = SEEDS["water64"], omega: float = 0.3) -> Workload:
    """Config 4 (192 atoms; the ncu / bench config): cubic L=23.46, 64 waters
    (min O-O 4.8), O s/s/s/p/p/d, H s/s/p, n_occ=256."""
    rng = np.random.default_rng(seed)
    cell, xyz, el = _water_box(rng, 23.46, 64, 4.8)
    b = _water_basis(rng, with_d=True, with_hp=True)
    return _assemble("water64", cell, xyz, el, b, omega=omega, n_occ=256, seed=seed)


def water343(seed: int = SEEDS["water343"], omega: float = 0.25) -> Workload:
    """Config 5: cubic L=41.9, 343 waters, O s/s/s/p/p, H s/s, n_occ=1372,
    Schwarz threshold 1e-11."""
    rng = np.random.default_rng(seed)
    cell, xyz, el = _water_box(rng, 41.9, 343, 4.8)
    b = _water_basis(rng, with_d=False, with_hp=False)
    return _assemble("water343", cell, xyz, el, b, omega=omega, n_occ=1372, seed=seed,
                     tau_schwarz=1e-11)


def pd_test_cell(seed: int = 77, omega: float = 0.45, L: float = 6.0) -> Workload:
    """Extra tiny s/p/d cell: 2 centres in a slightly sheared
    cell, modest exponents so the pure reciprocal-space sum converges."""
    rng = np.random.default_rng(seed)
    cell = np.array([[L, 0.0, 0.0], [0.4, L * 1.05, 0.0], [-0.3, 0.5, L * 0.95]])
    pts: List[np.ndarray] = []
    while len(pts) < 2:
        f = rng.uniform(0, 1, size=3)
        p = f @ cell
        if all(_min_image_dist(cell, p, q) >= 1.6 for q in pts):
            pts.append(p)
    b = _Basis()
    b.add("A", 0, [1.8, 0.7], [0.6, 0.5])
    b.add("A", 1, [1.3], [1.0])
    b.add("A", 2, [1.1], [1.0])
    b.add("B", 0, [1.6], [1.0])
    b.add("B", 1, [1.7, 0.8], [0.4, 0.7])
    return _assemble("pd_test", cell, np.array(pts), ["A", "B"], b, omega=omega, n_occ=3,
                     seed=seed)


CONFIGS = {"tiny": tiny, "water8": water8, "si64": si64, "water64": water64,
           "water343": water343, "pd_test": pd_test_cell}


def get(name: str, **kw) -> Workload:
    return CONFIGS[name](**kw)
