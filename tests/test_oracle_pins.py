"""Pins for the CPU oracle.  No GPU, no CUDA package.

Each test checks oracle/ against something that is not the oracle: a closed
form, a library special function, a textbook constant, the plain
reciprocal-space definition, or an exact invariance of the definition.
The paper prints no worked numeric example for this path (SURVEY 8(c) last row),
so there is no cited golden value from the paper itself.
"""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy.special import erfc, hyp1f1

from paper_2410_22278_b200 import workloads as W

import pure_g

XI_CUBIC = -2.837297479480619        # Madelung constant of a point charge in a cubic cell (textbook)
M_NACL = 1.7475645946331822          # NaCl Madelung constant w.r.t. nearest-neighbour distance (textbook)


def _dens(oracle, wl):
    S = oracle.overlap(wl)
    return W.density_from_orbitals(wl.orbitals_seed(), S), S


@pytest.fixture(scope="module")
def tiny_ref(oracle_mod):
    wl = W.tiny()
    P, S = _dens(oracle_mod, wl)
    return wl, P, S, oracle_mod.jk(wl, P)


@pytest.fixture(scope="module")
def pd_ref(oracle_mod):
    wl = W.pd_test_cell()
    P, S = _dens(oracle_mod, wl)
    return wl, P, S, oracle_mod.jk(wl, P)


# ---------------------------------------------------------------- P2: Boys
@pytest.mark.parametrize("x", [0.0, 1e-12, 1e-3, 0.7, 4.0, 17.3, 34.999, 35.001, 60.0, 1e4])
def test_boys_against_1f1(oracle_mod, x):
    """F_m(x) = 1F1(m+1/2; m+3/2; -x)/(2m+1), m <= 8 (SciPy); PAPER eq 28 is m = 0."""
    F = oracle_mod.boys(8, x)
    ref = np.array([hyp1f1(m + 0.5, m + 1.5, -x) / (2 * m + 1) for m in range(9)])
    assert np.max(np.abs(F - ref) / ref) < 5e-14
    if x > 0:
        f0 = 0.5 * math.sqrt(math.pi / x) * math.erf(math.sqrt(x))      # eq 28
        assert abs(F[0] - f0) / f0 < 5e-14 or x < 1e-6


# ---------------------------------------------------------------- P1: closed-form (ss|ss)
def _ssss_closed(kernel, omega, a, A, b, B, c, C, d, D, mpf=False):
    """PAPER eq 55/56 (L429, L439) for normalised s primitives, non-periodic, one image."""
    if mpf:
        sqrt, exp, erf, pi = mp.sqrt, mp.exp, mp.erf, mp.pi
    else:
        sqrt, exp, erf, pi = math.sqrt, math.exp, math.erf, math.pi
    p, q = a + b, c + d
    P = [(a * A[k] + b * B[k]) / p for k in range(3)]
    Q = [(c * C[k] + d * D[k]) / q for k in range(3)]
    ab2 = sum((A[k] - B[k]) ** 2 for k in range(3))
    cd2 = sum((C[k] - D[k]) ** 2 for k in range(3))
    pq2 = sum((P[k] - Q[k]) ** 2 for k in range(3))
    nrm = 1
    for e in (a, b, c, d):
        nrm = nrm * (2 * e / pi) ** 0.75 if not mpf else nrm * (2 * e / pi) ** mp.mpf("0.75")

    def F0(x):
        if x == 0:
            return 1
        return sqrt(pi) / 2 * erf(sqrt(x)) / sqrt(x)                    # eq 28

    alpha = p * q / (p + q)
    aw = 1 / (1 / p + 1 / q + 1 / omega ** 2)
    theta = omega * sqrt(p + q) / sqrt(p * q + omega ** 2 * (p + q))
    full = F0(alpha * pq2)
    lr = theta * F0(aw * pq2)
    val = {0: full, 1: full - lr, 2: lr}[kernel]
    return nrm * exp(-a * b / p * ab2) * exp(-c * d / q * cd2) * 2 * pi ** 2.5 / (p * q * sqrt(p + q)) * val \
        if not mpf else nrm * exp(-a * b / p * ab2) * exp(-c * d / q * cd2) * 2 * pi ** mp.mpf("2.5") / (p * q * sqrt(p + q)) * val


def test_ssss_closed_form(oracle_mod):
    rng = np.random.default_rng(5)
    for trial in range(40):
        a, b, c, d = np.exp(rng.uniform(math.log(0.1), math.log(50), 4))
        A, B, C, D = rng.uniform(-1.5, 1.5, (4, 3))
        if trial == 0:
            B, C, D = A.copy(), A.copy(), A.copy()      # coincident centres: x -> 0 branch
        omega = float(np.exp(rng.uniform(math.log(0.1), math.log(2.0))))
        for kernel in (0, 1, 2):
            ref = _ssss_closed(kernel, omega, a, A, b, B, c, C, d, D)
            got = oracle_mod.prim_eri(kernel, omega, 0, a, A, 0, b, B, 0, c, C, 0, d, D)[0, 0, 0, 0]
            assert abs(got - ref) <= 2e-13 * max(abs(ref), 1e-3), (trial, kernel)


# ---------------------------------------------------------------- P11: p/d classes by differentiating P1
def _unnorm_ratio(a, comp):
    """N(a;comp)/N(a;s): eq 6 ratio, retyped."""
    l = sum(comp)
    f = math.factorial
    return math.sqrt((8 * a) ** l * f(comp[0]) * f(comp[1]) * f(comp[2]) / (f(2 * comp[0]) * f(2 * comp[1]) * f(2 * comp[2])))


def _cart_from_derivs(a, comp):
    """(x-A)^i e^{-a(x-A)^2} as a combination of d^k/dA^k of e^{-a(x-A)^2}, per axis:
    i=0: [1]; i=1: (1/2a) d; i=2: (1/4a^2) d^2 + (1/2a)."""
    table = {0: {0: 1.0}, 1: {1: 1.0 / (2 * a)}, 2: {2: 1.0 / (4 * a * a), 0: 1.0 / (2 * a)}}
    terms = {(): 1.0}
    out = {}
    for kx, cx in table[comp[0]].items():
        for ky, cy in table[comp[1]].items():
            for kz, cz in table[comp[2]].items():
                out[(kx, ky, kz)] = cx * cy * cz
    return out


def _fd(f, x0, order, h):
    """Tensor-product central differences (order 1: (f+ - f-)/2h, order 2: (f+ - 2f0 + f-)/h^2)
    in multiprecision; truncation error O(h^2)."""
    sten = {0: [(0, 1)], 1: [(1, mp.mpf(1) / (2 * h)), (-1, mp.mpf(-1) / (2 * h))],
            2: [(1, 1 / h ** 2), (0, -2 / h ** 2), (-1, 1 / h ** 2)]}
    pts = [(list(x0), mp.mpf(1))]
    for n, o in enumerate(order):
        if o == 0:
            continue
        new = []
        for (x, w) in pts:
            for (k, c) in sten[o]:
                y = list(x); y[n] = y[n] + k * h
                new.append((y, w * c))
        pts = new
    return mp.fsum(w * f(x) for (x, w) in pts)


def _pick_components(ls):
    """Two component quadruples per class: the axis-aligned one (x, xx) and a mixed one
    (y / xy / yz ...), chosen so that the number of differentiated variables stays small."""
    first = tuple(0 for _ in ls)
    mixed = []
    for n, l in enumerate(ls):
        if l == 0:
            mixed.append(0)
        elif l == 1:
            mixed.append(1 + (n % 2))            # y or z
        else:
            mixed.append([1, 4, 2, 1][n])        # xy, yz, xz, xy
    return [first, tuple(mixed)]


@pytest.mark.parametrize("ls", [(1, 0, 0, 0), (0, 1, 1, 0), (2, 0, 0, 0), (1, 1, 0, 1), (2, 0, 1, 0),
                                (0, 2, 0, 2), (2, 1, 0, 0), (2, 2, 0, 0), (1, 0, 2, 1), (2, 1, 2, 1),
                                (2, 2, 2, 2)])
def test_higher_l_from_derivatives_of_closed_form(oracle_mod, ls):
    """p and d integrals are centre-derivatives of the s closed form (P11), taken here by
    mpmath high-precision numerical differentiation of eq 55/56: independent of the
    oracle's E and R recursions."""
    mp.mp.dps = 110
    rng = np.random.default_rng(100 + sum(l * 3 ** i for i, l in enumerate(ls)))
    exps = [float(v) for v in np.exp(rng.uniform(math.log(0.3), math.log(3.0), 4))]
    cen = rng.uniform(-1.0, 1.0, (4, 3))
    omega = 0.6
    kernel = 1
    got = oracle_mod.prim_eri(kernel, omega, ls[0], exps[0], cen[0], ls[1], exps[1], cen[1],
                              ls[2], exps[2], cen[2], ls[3], exps[3], cen[3])
    comps = [pure_g.cart_components(l) for l in ls]
    x0 = [mp.mpf(float(v)) for v in cen.ravel()]
    mexps = [mp.mpf(e) for e in exps]

    def f_full(x):
        c = [x[0:3], x[3:6], x[6:9], x[9:12]]
        return _ssss_closed(kernel, mp.mpf(omega), mexps[0], c[0], mexps[1], c[1], mexps[2], c[2],
                            mexps[3], c[3], mpf=True)

    for (i, j, k, l) in _pick_components(ls):
        cc = [comps[0][i], comps[1][j], comps[2][k], comps[3][l]]
        combos = [_cart_from_derivs(exps[n], cc[n]) for n in range(4)]
        ref = mp.mpf(0)
        for d0, c0 in combos[0].items():
            for d1, c1 in combos[1].items():
                for d2, c2 in combos[2].items():
                    for d3, c3 in combos[3].items():
                        order = tuple(d0) + tuple(d1) + tuple(d2) + tuple(d3)
                        val = _fd(f_full, x0, order, mp.mpf(10) ** -10)
                        ref += c0 * c1 * c2 * c3 * val
        for n in range(4):
            ref *= _unnorm_ratio(exps[n], cc[n])
        ref = float(ref)
        assert abs(got[i, j, k, l] - ref) <= 1e-11 * max(abs(ref), 1e-2), (ls, (i, j, k, l), got[i, j, k, l], ref)


# ---------------------------------------------------------------- P3: pure reciprocal-space brute force
def test_tiny_vs_pure_reciprocal_sum(oracle_mod, tiny_ref):
    wl, P, S, r = tiny_ref
    J, K, nG = pure_g.jk_pure_g(wl, P, gmax=24.0, chunk=16384)
    assert nG > 1e5
    assert np.max(np.abs(J - r["J"])) < 1e-12
    assert np.max(np.abs(K - r["K"])) < 1e-12


def test_pd_cell_vs_pure_reciprocal_sum(oracle_mod, pd_ref):
    """s, p, d shells, contracted, sheared cell: pins E/R recursions, the sign reading C-4,
    normalisation C-1, component order C-10 and SELF (C-6) at once."""
    wl, P, S, r = pd_ref
    J, K, nG = pure_g.jk_pure_g(wl, P, gmax=21.0, chunk=16384)
    assert np.max(np.abs(J - r["J"])) < 1e-12
    assert np.max(np.abs(K - r["K"])) < 1e-12
    # the overlap is the G = 0 coefficient of the same pair densities
    S0 = pure_g.pair_density_ft(wl, np.zeros((1, 3)))[:, :, 0].real
    assert np.max(np.abs(S0 - S)) < 1e-13


# ---------------------------------------------------------------- P5: omega invariance
def test_omega_invariance_tiny(oracle_mod, tiny_ref):
    wl, P, S, r = tiny_ref
    EJ, EK = 0.5 * np.trace(P @ r["J"]), 0.5 * np.trace(P @ r["K"])
    for om in (0.25, 0.6, 0.9):
        r2 = oracle_mod.jk(wl, P, omega=om, r_cut=0.0, g_cut=0.0)
        assert np.max(np.abs(r2["J"] - r["J"])) < 1e-12
        assert np.max(np.abs(r2["K"] - r["K"])) < 1e-12
        assert abs(0.5 * np.trace(P @ r2["J"]) - EJ) < 1e-9       # north_star bound
        assert abs(0.5 * np.trace(P @ r2["K"]) - EK) < 1e-9
        # the parts themselves do change: the test would be vacuous otherwise
        assert np.max(np.abs(r2["J_sr"] - r["J_sr"])) > 1e-3


def test_omega_invariance_pd(oracle_mod, pd_ref):
    wl, P, S, r = pd_ref
    for om in (0.3, 0.7):
        r2 = oracle_mod.jk(wl, P, omega=om)
        assert np.max(np.abs(r2["J"] - r["J"])) < 1e-12
        assert np.max(np.abs(r2["K"] - r["K"])) < 1e-12


# ---------------------------------------------------------------- P4: truncation
def test_truncation_converged(oracle_mod, tiny_ref):
    """Looser pair threshold / explicit cutoffs of config 1 agree with the unscreened run."""
    wl, P, S, r = tiny_ref
    r2 = oracle_mod.jk(wl, P, delta_o=1e-15, r_cut=0.0, g_cut=0.0)
    assert np.max(np.abs(r2["J"] - r["J"])) < 1e-12
    assert np.max(np.abs(r2["K"] - r["K"])) < 1e-12


# ---------------------------------------------------------------- P6: Madelung constants
def _single_s(L, a):
    return W.Workload(name="one_s", cell=np.eye(3) * L, xyz=np.array([[0.3, -0.2, 0.1]]),
                      sh_atom=np.array([0], np.int32), sh_l=np.array([0], np.int32),
                      sh_nprim=np.array([1], np.int32), sh_off=np.array([0], np.int32),
                      exps=np.array([a]), coefs=np.array([1.0]), omega=0.5, n_occ=1, seed=0)


def test_madelung_point_charge_cubic(oracle_mod):
    """(mm|mm) of one normalised s primitive with a L^2 >> 1 equals
    xi/L + 2 sqrt(a/pi) + pi/(Omega a) - sum_{T != 0} erfc(sqrt(a)|T|)/|T|."""
    L, a = 5.0, 2.5
    wl = _single_s(L, a)
    P = np.array([[1.0]])
    tail = 0.0
    for n in np.ndindex(9, 9, 9):
        t = (np.array(n) - 4) * L
        d = np.linalg.norm(t)
        if d > 0:
            tail += erfc(math.sqrt(a) * d) / d
    ref = XI_CUBIC / L + 2 * math.sqrt(a / math.pi) + math.pi / (L ** 3 * a) - tail
    for om in (0.5, 0.9):
        r = oracle_mod.jk(wl, P, omega=om)
        assert abs(r["J"][0, 0] - ref) < 1e-9
        assert abs(r["K"][0, 0] - ref) < 1e-9          # one function: J = K


def test_madelung_nacl(oracle_mod):
    """8 tight s primitives on rock-salt sites, P = diag(+-1): 1/2 tr(PJ) = -8 M/L + 8 sqrt(a/pi)."""
    L, a = 8.0, 6.0
    sites, q = [], []
    for i in range(2):
        for j in range(2):
            for k in range(2):
                sites.append(np.array([i, j, k]) * L / 2)
                q.append(1.0 if (i + j + k) % 2 == 0 else -1.0)
    n = 8
    wl = W.Workload(name="nacl", cell=np.eye(3) * L, xyz=np.array(sites),
                    sh_atom=np.arange(n, dtype=np.int32), sh_l=np.zeros(n, np.int32),
                    sh_nprim=np.ones(n, np.int32), sh_off=np.arange(n, dtype=np.int32),
                    exps=np.full(n, a), coefs=np.ones(n), omega=0.45, n_occ=1, seed=0)
    P = np.diag(q)
    r = oracle_mod.jk(wl, P, which="j")
    E = 0.5 * np.trace(P @ r["J"])
    ref = -8 * M_NACL / L + 8 * math.sqrt(a / math.pi)
    assert abs(E - ref) < 1e-9


# ---------------------------------------------------------------- P7: symmetry, ERI permutations
def test_symmetry_and_eri_permutations(oracle_mod, tiny_ref, pd_ref):
    for (wl, P, S, r) in (tiny_ref, pd_ref):
        assert np.max(np.abs(r["J"] - r["J"].T)) < 1e-12
        assert np.max(np.abs(r["K"] - r["K"].T)) < 1e-12
        assert np.max(np.abs(S - S.T)) < 1e-13
    wl, P, S, r = pd_ref
    N = wl.nbf
    # (mn|ls) for fixed (l,s) from J with a unit density (J is linear in P; the oracle
    # does not assume P symmetric)
    rng = np.random.default_rng(3)
    for _ in range(2):
        l, s = rng.integers(0, N, 2)
        E = np.zeros((N, N)); E[l, s] = 1.0
        Et = np.zeros((N, N)); Et[s, l] = 1.0
        J1 = oracle_mod.jk(wl, E, which="j")["J"]
        J2 = oracle_mod.jk(wl, Et, which="j")["J"]
        assert np.max(np.abs(J1 - J1.T)) < 1e-12          # (mn|ls) = (nm|ls)
        assert np.max(np.abs(J1 - J2)) < 1e-12            # (mn|ls) = (mn|sl)
        m, n = rng.integers(0, N, 2)
        E2 = np.zeros((N, N)); E2[m, n] = 1.0
        J3 = oracle_mod.jk(wl, E2, which="j")["J"]
        assert abs(J1[m, n] - J3[l, s]) < 1e-12           # (mn|ls) = (ls|mn)
        # K from the same tensor: K_mn[E_ls] = (ml|sn)
        K1 = oracle_mod.jk(wl, E, which="k")["K"]
        E3 = np.zeros((N, N)); E3[n, s] = 1.0             # J_ml[E_ns] = (ml|ns)
        J4 = oracle_mod.jk(wl, E3, which="j")["J"]
        assert abs(K1[m, n] - J4[m, l]) < 1e-12


# ---------------------------------------------------------------- P8 / P9
def test_rank1_identity_and_positivity(oracle_mod, tiny_ref, pd_ref):
    wl, P, S, r = pd_ref
    rng = np.random.default_rng(11)
    c = rng.standard_normal(wl.nbf)
    P1 = np.outer(c, c)
    r1 = oracle_mod.jk(wl, P1)
    assert np.max(np.abs(r1["J"] @ c - r1["K"] @ c)) < 1e-11 * np.max(np.abs(r1["J"] @ c))
    for (wl, P, S, r) in (tiny_ref, pd_ref):
        assert 0.5 * np.trace(P @ r["J"]) > 0
        assert np.linalg.eigvalsh(0.5 * (r["K"] + r["K"].T)).min() > -1e-12


# ---------------------------------------------------------------- P10: geometric invariances
def test_translation_and_image_invariance(oracle_mod, pd_ref):
    wl, P, S, r = pd_ref
    import dataclasses
    shift = np.array([0.37, -1.21, 2.05])
    xyz = wl.xyz + shift
    xyz[1] = xyz[1] + 2 * wl.cell[0] - 1 * wl.cell[2]       # one atom in another lattice image (L781)
    wl2 = dataclasses.replace(wl, xyz=xyz)
    r2 = oracle_mod.jk(wl2, P)
    assert np.max(np.abs(r2["J"] - r["J"])) < 1e-12
    assert np.max(np.abs(r2["K"] - r["K"])) < 1e-12
    assert np.max(np.abs(r2["S"] - S)) < 1e-13


def test_axis_permutation(oracle_mod, pd_ref):
    """x->y->z->x of cell and coordinates permutes p and d components in a known way."""
    wl, P, S, r = pd_ref
    import dataclasses
    perm = [2, 0, 1]                     # new (x,y,z) = old (z,x,y)
    wl2 = dataclasses.replace(wl, cell=wl.cell[:, perm], xyz=wl.xyz[:, perm])
    # AO permutation: component (ix,iy,iz) of the old frame becomes (iz,ix,iy) in the new frame
    off = wl.shell_offsets()
    idx = np.zeros(wl.nbf, dtype=int)
    for sh in range(wl.nshell):
        comps = pure_g.cart_components(int(wl.sh_l[sh]))
        for k, (ix, iy, iz) in enumerate(comps):
            idx[off[sh] + comps.index((iz, ix, iy))] = off[sh] + k      # new index <- old index
    P2 = P[np.ix_(idx, idx)]
    r2 = oracle_mod.jk(wl2, P2)
    assert np.max(np.abs(r2["J"] - r["J"][np.ix_(idx, idx)])) < 1e-12
    assert np.max(np.abs(r2["K"] - r["K"][np.ix_(idx, idx)])) < 1e-12


# ---------------------------------------------------------------- sampled mode = full mode on its blocks
def test_sampled_blocks_equal_full(oracle_mod, pd_ref):
    wl, P, S, r = pd_ref
    blocks = [(0, 0), (1, 2), (2, 2), (4, 1), (3, 0)]
    rs = oracle_mod.jk(wl, P, blocks=blocks)
    m = oracle_mod.block_mask(wl, blocks)
    for key in ("J", "K", "J_sr", "K_sr", "J_lr", "K_lr", "J_self", "K_self"):
        assert np.max(np.abs(rs[key][m] - r[key][m])) < 1e-13, key
        assert np.all(rs[key][~m] == 0.0)


# ---------------------------------------------------------------- P13: eq 5-6 normalisation of p and d components
def _quad_1d(m, c):
    """int_{-inf}^{inf} x^m e^{-c x^2} dx by adaptive quadrature (no closed form typed in)"""
    return mp.quad(lambda x: x ** m * mp.exp(-c * x * x), [-mp.inf, 0, mp.inf])


def test_prim_norm_by_quadrature(oracle_mod):
    """prim_norm (eq 5-6, reading C-1) pinned without retyping eq 6: a primitive is "normalised" iff
    int phi^2 = 1, so N = (int [x^i y^j z^k e^{-a r^2}]^2)^{-1/2} with the integral taken by mpmath quadrature.
    One centre with uncontracted s, p and d shells (coefficient 1) in a 40-bohr cube, where lattice images do not
    overlap (e^{-0.45 * 40^2} underflows): the oracle's crystalline S (eq 21) must equal the matrix of quadrature
    overlaps of the quadrature-normalised functions, for every one of the 10 components incl. d_xy, d_xz, d_yz."""
    mp.mp.dps = 30
    exps = {0: 1.3, 1: 0.9, 2: 1.1}
    wl = W.Workload(name="norm_pin", cell=np.eye(3) * 40.0, xyz=np.array([[1.0, -2.0, 0.5]]),
                    sh_atom=np.zeros(3, np.int32), sh_l=np.array([0, 1, 2], np.int32), sh_nprim=np.ones(3, np.int32),
                    sh_off=np.arange(3, dtype=np.int32), exps=np.array([exps[0], exps[1], exps[2]]),
                    coefs=np.ones(3), omega=0.3, n_occ=1, seed=1)
    S = oracle_mod.overlap(wl)
    comps = [(0, (0, 0, 0))] + [(1, c) for c in [(1, 0, 0), (0, 1, 0), (0, 0, 1)]] + \
            [(2, c) for c in [(2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 2, 0), (0, 1, 1), (0, 0, 2)]]     # C-10 order
    assert S.shape == (10, 10)

    def raw(ci, cj):
        (li, pi), (lj, pj) = ci, cj
        c = exps[li] + exps[lj]
        return _quad_1d(pi[0] + pj[0], c) * _quad_1d(pi[1] + pj[1], c) * _quad_1d(pi[2] + pj[2], c)

    nrm = [1 / mp.sqrt(raw(c, c)) for c in comps]
    for i, ci in enumerate(comps):
        for j, cj in enumerate(comps):
            ref = float(nrm[i] * nrm[j] * raw(ci, cj))
            assert abs(S[i, j] - ref) < 2e-14, (ci, cj, S[i, j], ref)
    assert np.abs(np.diag(S) - 1.0).max() < 2e-14
    # two values the quadrature must have produced (textbook): <d_xx|d_yy> = 1/3, <d_xy|d_xy> = 1
    assert abs(S[4, 7] - 1.0 / 3.0) < 1e-14 and abs(S[5, 5] - 1.0) < 2e-14


def test_pd_test_unit_diagonal_in_scaled_cell(oracle_mod):
    """Every component of the s/p/d test cell has unit crystalline self-overlap once the cell is scaled (x6) so that
    images do not overlap -- for the uncontracted shells directly by eq 5-6, for the contracted ones through C-9
    (axis-aligned component scaled to unit local self-overlap; d_xy... follow from the per-component norm)."""
    wl = W.pd_test_cell(L=36.0)
    S = oracle_mod.overlap(wl)
    assert wl.nbf == 14
    assert np.abs(np.diag(S) - 1.0).max() < 1e-13


# ---------------------------------------------------------------- P14-P16: one-electron Ewald terms
def test_kinetic_by_quadrature(oracle_mod):
    """Kinetic matrix (SI eq S1, reading C-27) without the E recursion: one s, one p and one d primitive on
    two centres 1.1 bohr apart in a 40-bohr cube (no image overlap); T_mn = -1/2 int phi_m phi_n'' separates into 1-D
    integrals taken by mpmath quadrature, with the functions normalised by quadrature as well."""
    mp.mp.dps = 30
    exps = [1.3, 0.9, 1.1, 0.7]
    ls = [0, 1, 2, 1]
    cen = np.array([[0.3, -0.2, 0.1], [0.3 + 0.7, -0.2 + 0.6, 0.1 - 0.6]])
    at = [0, 0, 1, 1]
    wl = W.Workload(name="kin_pin", cell=np.eye(3) * 40.0, xyz=cen, sh_atom=np.array(at, np.int32),
                    sh_l=np.array(ls, np.int32), sh_nprim=np.ones(4, np.int32), sh_off=np.arange(4, dtype=np.int32),
                    exps=np.array(exps), coefs=np.ones(4), omega=0.3, n_occ=1, seed=1)
    T = oracle_mod.one_electron(wl, np.zeros(2))["T"]
    funcs = []                                      # (exponent, centre, (ix, iy, iz))
    for sh in range(4):
        for comp in pure_g.cart_components(ls[sh]):
            funcs.append((exps[sh], cen[at[sh]], comp))
    assert T.shape == (len(funcs), len(funcs))

    def g1(x, a, c, i):
        return (x - c) ** i * mp.exp(-a * (x - c) ** 2)

    def ov(f, g, d):
        return mp.quad(lambda x: g1(x, f[0], f[1][d], f[2][d]) * g1(x, g[0], g[1][d], g[2][d]), [-mp.inf, 0, mp.inf])

    def kin(f, g, d):
        return mp.quad(lambda x: -0.5 * g1(x, f[0], f[1][d], f[2][d]) * mp.diff(lambda y: g1(y, g[0], g[1][d], g[2][d]), x, 2),
                       [-mp.inf, 0, mp.inf])

    nrm = [1 / mp.sqrt(ov(f, f, 0) * ov(f, f, 1) * ov(f, f, 2)) for f in funcs]
    rng = np.random.default_rng(0)
    pairs = [(i, i) for i in range(len(funcs))] + [tuple(p) for p in rng.integers(0, len(funcs), (14, 2))]
    for (i, j) in pairs:
        f, g = funcs[i], funcs[j]
        s = [ov(f, g, d) for d in range(3)]
        k = [kin(f, g, d) for d in range(3)]
        ref = float(nrm[i] * nrm[j] * (k[0] * s[1] * s[2] + s[0] * k[1] * s[2] + s[0] * s[1] * k[2]))
        assert abs(T[i, j] - ref) < 1e-11 * max(1.0, abs(ref)), (i, j, T[i, j], ref)
    assert np.abs(T - T.T).max() < 1e-13          # hermiticity: the Laplacian acts on the second function only


def test_nuclear_attraction_pure_g_and_omega(oracle_mod):
    """V of eq 52 (point charges under the zero-mean periodic kernel) against the plain reciprocal-space definition
    V_mn = sum_C q_C (1/Omega) sum_{G != 0} (4 pi/G^2) Re[conj(rho_mn(G)) e^{-iG.C}] -- no Boys function, no E or R
    recursion, no Ewald split (tests/pure_g.py) -- and its independence of the Ewald parameter."""
    wl = W.pd_test_cell()
    q = np.array([1.5, -0.7])                       # a charged cell on purpose: the SELF term matters
    ref = oracle_mod.one_electron(wl, q)
    G = pure_g.g_vectors(wl.cell, 24.0)
    vol = abs(np.linalg.det(wl.cell))
    V = np.zeros((wl.nbf, wl.nbf))
    for s in range(0, G.shape[0], 16384):
        Gc = G[s:s + 16384]
        rho = pure_g.pair_density_ft(wl, Gc)
        nuc = (q[None, :] * np.exp(-1j * Gc @ wl.xyz.T)).sum(1)
        V += np.einsum("g,mng,g->mn", 4 * math.pi / (vol * (Gc * Gc).sum(1)), rho.conj(), nuc).real
    assert np.abs(ref["V"] - V).max() < 1e-9
    assert np.abs(ref["V"]).max() > 0.05 and np.abs(ref["V_self"]).max() > 1e-3
    for om in (0.3, 0.9):
        r2 = oracle_mod.one_electron(wl, q, omega=om)
        assert np.abs(r2["V"] - ref["V"]).max() < 1e-10
        assert abs(r2["E_nuc"] - ref["E_nuc"]) < 1e-10
    assert np.abs(ref["V"] - ref["V"].T).max() < 1e-13


def test_nuclear_repulsion_madelung(oracle_mod):
    """E_nuc of eq 91 against textbook constants: one unit charge in a cube (charged cell: 1/2 xi / L) and the rock-salt
    arrangement of +-1 charges (-8 M / L per conventional cell)."""
    L = 7.0
    one = W.Workload(name="q1", cell=np.eye(3) * L, xyz=np.array([[0.4, 0.1, -0.3]]), sh_atom=np.zeros(1, np.int32),
                     sh_l=np.zeros(1, np.int32), sh_nprim=np.ones(1, np.int32), sh_off=np.zeros(1, np.int32),
                     exps=np.array([1.0]), coefs=np.ones(1), omega=0.5, n_occ=1, seed=1)
    e = oracle_mod.one_electron(one, np.array([1.0]))["E_nuc"]
    assert abs(e - 0.5 * XI_CUBIC / L) < 1e-11
    sites, ch = [], []
    for i in range(2):
        for j in range(2):
            for k in range(2):
                sites.append([i * L / 2, j * L / 2, k * L / 2]); ch.append(1.0 if (i + j + k) % 2 == 0 else -1.0)
    n = len(sites)
    nacl = W.Workload(name="nacl", cell=np.eye(3) * L, xyz=np.array(sites), sh_atom=np.arange(n, dtype=np.int32),
                      sh_l=np.zeros(n, np.int32), sh_nprim=np.ones(n, np.int32), sh_off=np.arange(n, dtype=np.int32),
                      exps=np.full(n, 2.0), coefs=np.ones(n), omega=0.45, n_occ=1, seed=1)
    for om in (0.45, 0.8):
        e = oracle_mod.one_electron(nacl, np.array(ch), omega=om)["E_nuc"]
        assert abs(e - (-8.0 * M_NACL / L)) < 1e-10, (om, e)
