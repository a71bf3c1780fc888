"""ctypes front end of the fp64 CPU oracle (oracle/pbc_jk_oracle.c).

TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It never imports
the CUDA package and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pbc_jk_oracle.c")
_LIB = os.path.join(_HERE, "libpbc_jk_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


class _System(C.Structure):
    _fields_ = [("cell", C.c_double * 9), ("natom", C.c_int32), ("xyz", C.POINTER(C.c_double)),
                ("nshell", C.c_int32), ("sh_atom", C.POINTER(C.c_int32)), ("sh_l", C.POINTER(C.c_int32)),
                ("sh_nprim", C.POINTER(C.c_int32)), ("sh_off", C.POINTER(C.c_int32)),
                ("exps", C.POINTER(C.c_double)), ("coefs", C.POINTER(C.c_double))]


class _Opts(C.Structure):
    _fields_ = [("delta_o", C.c_double), ("r_cut", C.c_double), ("g_cut", C.c_double),
                ("which", C.c_int32), ("parts", C.c_int32), ("g_min", C.c_double)]


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_boys.argtypes = [C.c_int, C.c_double, C.POINTER(C.c_double)]
        _lib.orc_prim_eri.restype = None
        _lib.orc_overlap.restype = C.c_int
        _lib.orc_jk.restype = C.c_int
        _lib.orc_nbf.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_one_electron.restype = C.c_int
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


class _Sys:
    """Keeps the numpy buffers alive next to the C struct."""

    def __init__(self, wl):
        self.bufs = dict(
            xyz=np.ascontiguousarray(wl.xyz, dtype=np.float64),
            sh_atom=np.ascontiguousarray(wl.sh_atom, dtype=np.int32),
            sh_l=np.ascontiguousarray(wl.sh_l, dtype=np.int32),
            sh_nprim=np.ascontiguousarray(wl.sh_nprim, dtype=np.int32),
            sh_off=np.ascontiguousarray(wl.sh_off, dtype=np.int32),
            exps=np.ascontiguousarray(wl.exps, dtype=np.float64),
            coefs=np.ascontiguousarray(wl.coefs, dtype=np.float64))
        s = _System()
        cell = np.ascontiguousarray(wl.cell, dtype=np.float64).ravel()
        for i in range(9):
            s.cell[i] = float(cell[i])
        b = self.bufs
        s.natom = b["xyz"].shape[0]
        s.xyz = _dp(b["xyz"])
        s.nshell = b["sh_l"].shape[0]
        s.sh_atom, s.sh_l, s.sh_nprim, s.sh_off = _ip(b["sh_atom"]), _ip(b["sh_l"]), _ip(b["sh_nprim"]), _ip(b["sh_off"])
        s.exps, s.coefs = _dp(b["exps"]), _dp(b["coefs"])
        self.c = s


def num_threads() -> int:
    return int(_load().orc_num_threads())


def boys(mmax: int, x: float) -> np.ndarray:
    out = np.zeros(mmax + 1)
    _load().orc_boys(int(mmax), float(x), _dp(out))
    return out


def prim_eri(kernel: int, omega: float, la, a, A, lb, b, B, lc, c, Cc, ld, d, D) -> np.ndarray:
    """Non-periodic primitive quartet over eq-6-normalised Cartesian Gaussians.
    kernel 0: 1/r, 1: erfc(w r)/r, 2: erf(w r)/r.  Shape (na, nb, nc, nd)."""
    nc = lambda l: (l + 1) * (l + 2) // 2
    out = np.zeros((nc(la), nc(lb), nc(lc), nc(ld)))
    A, B, Cc, D = (np.ascontiguousarray(v, dtype=np.float64) for v in (A, B, Cc, D))
    _load().orc_prim_eri(C.c_int(kernel), C.c_double(omega),
                         C.c_int(la), C.c_double(a), _dp(A), C.c_int(lb), C.c_double(b), _dp(B),
                         C.c_int(lc), C.c_double(c), _dp(Cc), C.c_int(ld), C.c_double(d), _dp(D), _dp(out))
    return out


def overlap(wl, delta_o: float = 1e-18, r_cut: float = 0.0) -> np.ndarray:
    """Crystalline overlap S (PAPER eq 21)."""
    lib = _load()
    s = _Sys(wl)
    n = lib.orc_nbf(C.byref(s.c))
    S = np.zeros((n, n))
    lib.orc_overlap(C.byref(s.c), C.c_double(delta_o), C.c_double(r_cut), _dp(S))
    return S


def jk(wl, P: np.ndarray, omega: Optional[float] = None, blocks: Optional[Sequence[Tuple[int, int]]] = None,
       delta_o: float = 1e-18, r_cut: Optional[float] = None, g_cut: Optional[float] = None,
       which: str = "jk", parts: str = "sr+lr+self", g_min: float = 0.0) -> dict:
    """J and K with their SR / LR / SELF parts.

    blocks=None: the full matrices.  blocks=[(shell_mu, shell_nu), ...]: only those
    shell blocks are computed (sampled mode); everything else is left 0.
    Returns dict with J, K (sums of the requested parts), the parts, S, counts.
    """
    lib = _load()
    s = _Sys(wl)
    n = lib.orc_nbf(C.byref(s.c))
    P = np.ascontiguousarray(P, dtype=np.float64)
    assert P.shape == (n, n)
    o = _Opts()
    o.delta_o = delta_o
    o.r_cut = float(wl.r_cut if r_cut is None else r_cut)
    o.g_cut = float(wl.g_cut if g_cut is None else g_cut)
    o.g_min = float(g_min)
    o.which = (1 if "j" in which else 0) | (2 if "k" in which else 0)
    o.parts = (1 if "sr" in parts else 0) | (2 if "lr" in parts else 0) | (4 if "self" in parts else 0)
    om = float(wl.omega if omega is None else omega)
    z = lambda: np.zeros((n, n))
    Jsr, Jlr, Jself, Ksr, Klr, Kself, S = z(), z(), z(), z(), z(), z(), z()
    counts = (C.c_longlong * 4)()
    if blocks is None:
        nblk, bm, bn = -1, np.zeros(1, np.int32), np.zeros(1, np.int32)
    else:
        nblk = len(blocks)
        bm = np.ascontiguousarray([b[0] for b in blocks], dtype=np.int32)
        bn = np.ascontiguousarray([b[1] for b in blocks], dtype=np.int32)
        if nblk == 0:
            bm, bn = np.zeros(1, np.int32), np.zeros(1, np.int32)
    rc = lib.orc_jk(C.byref(s.c), C.c_double(om), C.byref(o), _dp(P), C.c_int(nblk), _ip(bm), _ip(bn),
                    _dp(Jsr), _dp(Jlr), _dp(Jself), _dp(Ksr), _dp(Klr), _dp(Kself), _dp(S), counts)
    if rc != 0:
        raise RuntimeError("oracle failed")
    return dict(J=Jsr + Jlr + Jself, K=Ksr + Klr + Kself, J_sr=Jsr, J_lr=Jlr, J_self=Jself,
                K_sr=Ksr, K_lr=Klr, K_self=Kself, S=S,
                counts=dict(quartets_J=int(counts[0]), quartets_K=int(counts[1]),
                            pair_images=int(counts[2]), n_G=int(counts[3])))


def one_electron(wl, charges, omega: Optional[float] = None, delta_o: float = 1e-18, r_cut: Optional[float] = None,
                 g_cut: Optional[float] = None) -> dict:
    """One-electron Ewald terms: kinetic matrix T (SI eq S1), the interaction V of every pair density
    with the point charges `charges` (one per atom; PAPER eq 52, SR / LR / SELF parts) under the zero-mean periodic
    kernel, and the Ewald energy E_nuc of the point charges themselves (eq 91)."""
    lib = _load()
    s = _Sys(wl)
    n = lib.orc_nbf(C.byref(s.c))
    q = np.ascontiguousarray(charges, dtype=np.float64)
    assert q.shape == (s.c.natom,)
    o = _Opts()
    o.delta_o = delta_o
    o.r_cut = float(wl.r_cut if r_cut is None else r_cut)
    o.g_cut = float(wl.g_cut if g_cut is None else g_cut)
    o.which, o.parts, o.g_min = 3, 7, 0.0
    om = float(wl.omega if omega is None else omega)
    z = lambda: np.zeros((n, n))
    T, Vsr, Vlr, Vself = z(), z(), z(), z()
    e = np.zeros(4)
    rc = lib.orc_one_electron(C.byref(s.c), C.c_double(om), C.byref(o), _dp(q), _dp(T), _dp(Vsr), _dp(Vlr), _dp(Vself), _dp(e))
    if rc != 0:
        raise RuntimeError("oracle failed")
    return dict(T=T, V=Vsr + Vlr + Vself, V_sr=Vsr, V_lr=Vlr, V_self=Vself, E_nuc=float(e[3]),
                E_nuc_parts=dict(lr=float(e[0]), sr=float(e[1]), const=float(e[2])))


def block_mask(wl, blocks: Sequence[Tuple[int, int]]) -> np.ndarray:
    """Boolean N x N mask of the AO entries covered by the listed shell blocks."""
    off = np.concatenate([wl.shell_offsets(), [wl.nbf]])
    m = np.zeros((wl.nbf, wl.nbf), dtype=bool)
    for (a, b) in blocks:
        m[off[a]:off[a + 1], off[b]:off[b + 1]] = True
    return m
