"""Pin P3: pure reciprocal-space evaluation of J and K from the
plain definition

    (mn|ls) = (1/Omega) sum_{G != 0} (4 pi / G^2) conj(rho_mn(G)) rho_ls(G)

(PAPER eq 54 L408 at Gamma with the divergent K=0 term dropped, L253).  Uses no
Boys function, no Hermite E/R recursion and no Ewald split: the 1-D Fourier
integrals of Cartesian Gaussian products are written with binomial expansions
about the product centre and physicists' Hermite polynomials,

    int y^n e^{-p y^2 - i G y} dy = sqrt(pi/p) e^{-G^2/4p} (-i)^n (2 sqrt p)^{-n} H_n(G / (2 sqrt p)).

Independent of oracle/ (numpy only).  Converges only for modest exponents on
small cells, which is what the pin uses it on.
"""
from __future__ import annotations

import itertools
import math

import numpy as np
from numpy.polynomial import hermite as _H
from numpy.polynomial import polynomial as _P


def cart_components(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def _norm(a, ix, iy, iz):
    # PAPER eq 6 (reading C-1), retyped here on purpose
    l = ix + iy + iz
    f = math.factorial
    return (2 * a / math.pi) ** 0.75 * math.sqrt((8 * a) ** l * f(ix) * f(iy) * f(iz) / (f(2 * ix) * f(2 * iy) * f(2 * iz)))


def g_vectors(cell, gmax):
    b = 2 * math.pi * np.linalg.inv(cell).T          # rows b_i
    nmax = [int(math.ceil(gmax * np.linalg.norm(cell[i]) / (2 * math.pi))) + 1 for i in range(3)]
    rng = [np.arange(-n, n + 1) for n in nmax]
    m = np.array(list(itertools.product(*rng)))
    G = m @ b
    g2 = (G * G).sum(1)
    keep = (g2 > 1e-12) & (g2 <= gmax * gmax)
    return G[keep]


def _poly_coeffs(i, j, PA, PB):
    """Coefficients c_n (arrays over images) of (y+PA)^i (y+PB)^j = sum_n c_n y^n."""
    poly = [np.ones_like(PA)]
    for (k, sh) in ((i, PA), (j, PB)):
        for _ in range(k):
            new = [np.zeros_like(PA) for _ in range(len(poly) + 1)]
            for n, c in enumerate(poly):
                new[n] = new[n] + c * sh
                new[n + 1] = new[n + 1] + c
            poly = new
    return poly


def pair_density_ft(wl, G, tail=1e-22):
    """rho_mn(G) for all ordered AO pairs, image-summed: array (N, N, nG) complex."""
    N = wl.nbf
    off = wl.shell_offsets()
    out = np.zeros((N, N, G.shape[0]), dtype=complex)
    cell = wl.cell
    inv = np.linalg.inv(cell)
    for A in range(wl.nshell):
        for B in range(wl.nshell):
            RA, RB = wl.xyz[wl.sh_atom[A]], wl.xyz[wl.sh_atom[B]]
            la, lb = int(wl.sh_l[A]), int(wl.sh_l[B])
            for ia in range(wl.sh_nprim[A]):
                for ib in range(wl.sh_nprim[B]):
                    a = wl.exps[wl.sh_off[A] + ia]; b = wl.exps[wl.sh_off[B] + ib]
                    ca = wl.coefs[wl.sh_off[A] + ia]; cb = wl.coefs[wl.sh_off[B] + ib]
                    p = a + b
                    mu = a * b / p
                    R = math.sqrt(math.log(1 / tail) / mu) + 2.0
                    nmax = [int(math.ceil((R + np.linalg.norm(RA - RB)) * np.linalg.norm(inv[:, k]))) + 1 for k in range(3)]
                    n = np.array(list(itertools.product(*[range(-m, m + 1) for m in nmax])))
                    Bt = RB[None, :] + n @ cell                                   # (img, 3)
                    Bt = Bt[np.linalg.norm(RA[None, :] - Bt, axis=1) <= R]
                    one = {}
                    for d in range(3):
                        Gd = G[:, d]
                        Px = (a * RA[d] + b * Bt[:, d]) / p                       # (img,)
                        pref = np.exp(-mu * (RA[d] - Bt[:, d]) ** 2)
                        base = (pref[:, None] * (math.sqrt(math.pi / p) * np.exp(-Gd * Gd / (4 * p)))[None, :]
                                * np.exp(-1j * Px[:, None] * Gd[None, :]))        # (img, g)
                        g = Gd / (2 * math.sqrt(p))
                        herm = []
                        for k in range(la + lb + 1):
                            c = np.zeros(k + 1); c[k] = 1.0
                            herm.append(((-1j) ** k) * (2 * math.sqrt(p)) ** (-k) * _H.hermval(g, c))
                        for i in range(la + 1):
                            for j in range(lb + 1):
                                cs = _poly_coeffs(i, j, Px - RA[d], Px - Bt[:, d])
                                fac = sum(c[:, None] * herm[k][None, :] for k, c in enumerate(cs))
                                one[(d, i, j)] = base * fac
                    for ka, (ix, iy, iz) in enumerate(cart_components(la)):
                        for kb, (jx, jy, jz) in enumerate(cart_components(lb)):
                            c = ca * cb * _norm(a, ix, iy, iz) * _norm(b, jx, jy, jz)
                            out[off[A] + ka, off[B] + kb] += c * np.einsum(
                                "ig,ig,ig->g", one[(0, ix, jx)], one[(1, iy, jy)], one[(2, iz, jz)])
    return out


def jk_pure_g(wl, P, gmax, chunk=4096):
    """J and K straight from the definition, all in reciprocal space."""
    G = g_vectors(wl.cell, gmax)
    vol = abs(np.linalg.det(wl.cell))
    N = wl.nbf
    J = np.zeros((N, N)); K = np.zeros((N, N))
    for s in range(0, G.shape[0], chunk):
        Gc = G[s:s + chunk]
        rho = pair_density_ft(wl, Gc)                       # (N,N,g)
        w = 4 * math.pi / (vol * (Gc * Gc).sum(1))
        tot = np.einsum("ls,lsg->g", P, rho)
        J += np.einsum("g,mng,g->mn", w, rho.conj(), tot).real
        K += np.einsum("g,mlg,ls,sng->mn", w, rho.conj(), P, rho, optimize=True).real
    return J, K, G.shape[0]
