"""Generator of the straight-line quartet evaluators of the real-space K kernels.

    python gen_sr_k.py OUTDIR            -> OUTDIR/k_eval_{la}{lb}{ld}.cuh for every unit of build.py

One specialisation KEval<LA,LB,LC,LD>::run per angular-momentum class (mu:LA lambda:LB | sigma:LC nu:LD).
Everything is emitted with literal indices (no loops, no index arithmetic at run time), so that every
array element is a register or a shared-memory word with an immediate offset:

  1. Hermite Coulomb integrals R^0_tuv, t+u+v <= L, from the merged Boys values Rm[m] = R^m_000
     (PAPER eq 47-51), in place; registers for L <= 4, shared memory (one column per
     thread, Rs[i*RS]) above.
  2. per ket component pair (d, c):  X_T = sum_S E^{nu sigma}_S R_{T+S}                 (eq 16, 56)
     per bra component pair (a, b):  I_ab = sum_T (-1)^{|T|} E^{mu lambda}_T X_T       (reading C-4)
     K_ad += P'_bc I_ab                                                                 (eq 74)
     The E products come from the per-pair tables built at create (etab_kernel), one row per lane for the bra and
     one for the ket, read through L1 (the lanes of a pass mostly share a bra).  The loads of a ket component
     pair's E terms and density elements are issued one block ahead of their use (software pipelining).

The evaluator is a template over the scalar type T: double, or float for the mixed-precision mode (PAPER 3.5
L817-821), where the tables and the density are read from their fp32 copies.

Table order (same for bra and ket rows; first index = the shell at home, second = the translated one):
  n runs over i1 in cart(l1), i2 in cart(l2), tx <= x1+x2, ty <= y1+y2, tz <= z1+z2 (nested in that order).
"""
from __future__ import annotations

import os
import sys


def cart(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def nherm(L):
    return (L + 1) * (L + 2) * (L + 3) // 6


def hidx(t, u, v):
    n = t + u + v
    return n * (n + 1) * (n + 2) // 6 + (n - t) * (n - t + 1) // 2 + (n - t - u)


def eterm_table(l1, l2):
    """[(i1, i2, [(tx,ty,tz, n), ...]), ...] with n the running table index"""
    out, n = [], 0
    for i1, a in enumerate(cart(l1)):
        for i2, b in enumerate(cart(l2)):
            terms = []
            for tx in range(a[0] + b[0] + 1):
                for ty in range(a[1] + b[1] + 1):
                    for tz in range(a[2] + b[2] + 1):
                        terms.append((tx, ty, tz, n))
                        n += 1
            out.append((i1, i2, terms))
    return out, n


def emit_R(L, smem):
    """statements forming R^0_tuv in place (same visiting order as hermite_R in pbcjk_md.cuh)"""
    def R(i, write=False):
        if not smem:
            return f"R{i}"
        return f"Rs[{i} * RS]" if write else f"LDV(Rs + {i} * RS)"
    o = []
    if not smem:
        o.append("T " + ", ".join(f"R{i}" for i in range(nherm(L))) + ";")
    o.append(f"{R(0, True)} = Rm[{L}];")
    for m in range(L - 1, -1, -1):
        for n in range(L - m, 0, -1):
            for t in range(n, -1, -1):
                for u in range(n - t, -1, -1):
                    v = n - t - u
                    if t > 0:
                        ax, k, lo1, lo2 = "X", t, hidx(t - 1, u, v), hidx(t - 2, u, v) if t > 1 else -1
                    elif u > 0:
                        ax, k, lo1, lo2 = "Y", u, hidx(t, u - 1, v), hidx(t, u - 2, v) if u > 1 else -1
                    else:
                        ax, k, lo1, lo2 = "Z", v, hidx(t, u, v - 1), hidx(t, u, v - 2) if v > 1 else -1
                    if k == 1:
                        e = f"{ax} * {R(lo1)}"
                    elif k == 2:
                        e = f"fma({ax}, {R(lo1)}, {R(lo2)})"
                    else:
                        e = f"fma(T({float(k - 1)}), {R(lo2)}, {ax} * {R(lo1)})"
                    o.append(f"{R(hidx(t, u, v), True)} = {e};")
        o.append(f"{R(0, True)} = Rm[{m}];")
    return o, R


def emit_class(la, lb, lc, ld):
    LBRA, LKET = la + lb, lc + ld
    L = LBRA + LKET
    smem = L > 4
    NA, NB, NC, ND = (len(cart(x)) for x in (la, lb, lc, ld))
    bra, nbra = eterm_table(la, lb)           # rows (a, b)
    ket, nket = eterm_table(ld, lc)           # rows (d, c): first index = nu (home shell), second = sigma
    Tlist = [(tx, ty, tz) for tx in range(LBRA + 1) for ty in range(LBRA + 1 - tx) for tz in range(LBRA + 1 - tx - ty)]
    o = []
    w = o.append
    w(f"// ({'spd'[la]}{'spd'[lb]}|{'spd'[lc]}{'spd'[ld]}): L = {L}, {nherm(L)} Hermite integrals "
      f"({'shared memory' if smem else 'registers'}), {nbra} bra and {nket} ket E terms")
    w(f"template <> struct KEval<{la}, {lb}, {lc}, {ld}> {{")
    w(f"    static constexpr int NBRA = {nbra}, NKET = {nket};")
    w("    template <int RS, typename T>")
    w("    static __device__ __forceinline__ void run(const T *__restrict__ bE, const T *__restrict__ kE,")
    w("                                               const T *__restrict__ Pb, const int ldP,")
    w(f"                                               const T (&Rm)[{L + 1}], const T X, const T Y,")
    w(f"                                               const T Z, T *__restrict__ Rs, T (&K)[{NA * ND}])")
    w("    {")
    body, R = emit_R(L, smem)
    for s in body:
        w("        " + s)
    # one basic block per (d, c): a rolled loop over a switch.  ptxas schedules block by block (its time grows
    # faster than linearly with the block length: 7 min for (dd|dp) as one block); every lane takes the same
    # case, so the branch is uniform.  The ket E terms and density elements of block dc + 1 are loaded while
    # block dc computes (registers en*/pn* -> ec*/pc* at the end of the block).
    nblk = ND * NC
    kmax = max(len(k[2]) for k in ket) if LKET > 0 else 0
    # the one-block-ahead loads cost kmax + NB extra live doubles: worth it only where registers are not the limit
    prefetch = True      # measured on water64: on in every class beats off in the L >= 5 classes by 10-15 %

    def loads(blk, dst_e, dst_p):
        d, c = divmod(blk, NC)
        terms = ket[d * NC + c][2]
        out = []
        if LKET > 0:
            out += [f"{dst_e}{k} = __ldg(kE + {t[3]});" for k, t in enumerate(terms)]
        out += [f"{dst_p}{b} = __ldg(Pb + {b} * ldP + {c});" for b in range(NB)]
        return out

    if prefetch:
        if kmax:
            w("        T " + ", ".join(f"ec{k} = T(0)" for k in range(kmax)) + ";")
        w("        T " + ", ".join(f"pc{b}" for b in range(NB)) + ";")
        for s in loads(0, "ec", "pc"):
            w("        " + s)
    if nblk > 1:
        w("#pragma unroll 1")
        w(f"        for (int dc = 0; dc < {nblk}; ++dc) {{")
        w("        switch (dc) {")
    for d in range(ND):
        for c in range(NC):
            blk = d * NC + c
            terms = ket[blk][2]
            if nblk > 1:
                w(f"        case {blk}:")
            w(f"        {{   // nu component {d}, sigma component {c}")
            if prefetch and blk + 1 < nblk:
                if kmax:
                    w("            T " + ", ".join(f"en{k} = T(0)" for k in range(kmax)) + ";")
                w("            T " + ", ".join(f"pn{b}" for b in range(NB)) + ";")
                for s in loads(blk + 1, "en", "pn"):
                    w("            " + s)
            if not prefetch:
                if LKET > 0:
                    w("            const T " + ", ".join(f"ec{k} = __ldg(kE + {t[3]})" for k, t in enumerate(terms)) + ";")
                w("            const T " + ", ".join(f"pc{b} = __ldg(Pb + {b} * ldP + {c})" for b in range(NB)) + ";")
            ev = ["1.0"] if LKET == 0 else [f"ec{k}" for k in range(len(terms))]
            # X_T = sum_S E_S R_{T+S}
            for (tx, ty, tz) in Tlist:
                e = None
                for k, (sx, sy, sz, _) in enumerate(terms):
                    r = R(hidx(tx + sx, ty + sy, tz + sz))
                    if e is None:
                        e = r if ev[k] == "1.0" else f"{ev[k]} * {r}"
                    else:
                        e = f"fma({ev[k]}, {r}, {e})"
                w(f"            const T x{hidx(tx, ty, tz)} = {e};")
            # I_ab = sum_T (-1)^|T| E_T X_T ; K_ad += P_bc I_ab
            for a in range(NA):
                acc = f"K[{a * ND + d}]"
                w(f"            {{ T k = {acc};")
                for b in range(NB):
                    bt = bra[a * NB + b][2]
                    e = None
                    for (tx, ty, tz, n) in bt:
                        odd = (tx + ty + tz) & 1
                        x = f"x{hidx(tx, ty, tz)}"
                        if LBRA == 0:
                            e = x
                        elif e is None:
                            e = f"{'-' if odd else ''}LDGV(bE + {n}) * {x}"
                        else:
                            e = f"fma({'-' if odd else ''}LDGV(bE + {n}), {x}, {e})"
                    w(f"              k = fma(pc{b}, {e}, k);")
                w(f"              {acc} = k; }}")
            if prefetch and blk + 1 < nblk:
                mv = [f"ec{k} = en{k};" for k in range(kmax)] + [f"pc{b} = pn{b};" for b in range(NB)]
                w("            " + " ".join(mv))
            w("        }")
            if nblk > 1:
                w("        break;")
    if nblk > 1:
        w("        }")
        w("        }")
    w("    }")
    w("};")
    return "\n".join(o)


def units():
    return [(la, lb, ld) for la in range(3) for ld in range(la + 1) for lb in range(3)]


def main(outdir):
    os.makedirs(outdir, exist_ok=True)
    for (la, lb, ld) in units():
        txt = ["// GENERATED by gen_sr_k.py -- do not edit.", "#pragma once",
               "// shared-memory R columns and the bra's E terms are read where they are used: a volatile load is neither",
               "// hoisted nor kept live across blocks (NVVM would otherwise hold the whole bra table and all R_tuv in",
               "// registers and spill them).  LDGV = volatile ld.global.nc (pbcjk_srk.cuh).",
               "#define LDV(p) (*(const volatile T *)(p))", "#define LDGV(p) ldg_volatile(p)", "namespace pbcjk {", ""]
        for lc in range(3):
            txt.append(emit_class(la, lb, lc, ld))
            txt.append("")
        txt.append("}  // namespace pbcjk")
        txt.append("#undef LDV")
        txt.append("#undef LDGV")
        path = os.path.join(outdir, f"k_eval_{la}{lb}{ld}.cuh")
        new = "\n".join(txt) + "\n"
        if not os.path.exists(path) or open(path).read() != new:
            with open(path, "w") as fh:
                fh.write(new)


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else os.path.join(os.path.dirname(os.path.abspath(__file__)), "build", "gen"))
