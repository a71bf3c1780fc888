/*
 * oracle/pbc_jk_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU oracle for the Gamma-point, Ewald-split periodic
 * Coulomb (J) and exact-exchange (K) matrices over contracted Cartesian
 * Gaussian shells (s, p, d), written from /root/reference/PAPER.md
 * (arxiv 2410.22278).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code,
 * header, table or helper with the CUDA path under paper_2410_22278_b200/csrc.
 *
 * What it evaluates ("Ewald form"; PAPER eq 56 L439 generalised
 * by eq 69 L518 and eq 98), for every primitive quartet and every
 * pair of pair-images T2, T3:
 *
 *   SR   = 2 pi^{5/2}/(p q sqrt(p+q)) sum_{T1} sum_t E^{ab}_t sum_s E^{cd}_s (-1)^{|t|}
 *          [ R^0_{t+s}(alpha, L) - theta R^0_{t+s}(alpha_w, L) ],  L = Q(T3) - P(T2) + T1
 *   LR   = sum_{G != 0} 4 pi/(Omega G^2) e^{-G^2/4w^2} Re[ conj(rho_ab(G)) rho_cd(G) ]
 *   SELF = -pi/(Omega w^2) S_ab S_cd
 *
 * with alpha = pq/(p+q), alpha_w = 1/(1/p+1/q+1/w^2), theta = w sqrt(p+q)/sqrt(pq+w^2(p+q)),
 * J_mn = sum_ls P_ls (mn|ls) (eq 73), K_mn = sum_ls P_ls (ml|sn) (eq 74), Gamma point.
 *
 * Readings of garbled / silent passages: C-1 (eq 6),
 * C-4 (sign and s-index of eq 98's real-space term), C-6 (SELF kept), C-10
 * (component order p: x,y,z; d: xx,xy,xz,yy,yz,zz).
 *
 * One-electron Ewald terms (orc_one_electron below): kinetic matrix (SI eq S1), nuclear
 * attraction matrix (eq 52), nuclear repulsion energy (eq 91); reading C-27 for the garbled eq S1.
 *
 * Pins (tests/test_oracle_pins.py): closed-form attenuated (ss|ss) with erf,
 * 1F1 Boys values, pure reciprocal-space brute force, omega invariance,
 * Madelung constants, symmetry, rank-1 J/K identity, positivity, geometric
 * invariances, finite differences for p/d.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

#define LMAX 2
#define LTOT (4 * LMAX)

typedef struct {
    double cell[9];          /* rows a1, a2, a3 (bohr) */
    int32_t natom;
    const double *xyz;       /* 3*natom */
    int32_t nshell;
    const int32_t *sh_atom, *sh_l, *sh_nprim, *sh_off;
    const double *exps, *coefs;
} orc_system;

static int ncart(int l) { return (l + 1) * (l + 2) / 2; }

/* Cartesian components in the order of C-10 (PAPER L721 example list). */
static void cart_comp(int l, int k, int *ix, int *iy, int *iz)
{
    int n = 0;
    for (int x = l; x >= 0; --x)
        for (int y = l - x; y >= 0; --y) {
            if (n == k) { *ix = x; *iy = y; *iz = l - x - y; return; }
            ++n;
        }
    *ix = *iy = *iz = 0;
}

static double fact(int n) { double f = 1; for (int i = 2; i <= n; ++i) f *= i; return f; }

/* PAPER eq 6 (L72), reading C-1: each Cartesian component normalised on its own. */
static double prim_norm(double a, int ix, int iy, int iz)
{
    int l = ix + iy + iz;
    double num = pow(8.0 * a, l) * fact(ix) * fact(iy) * fact(iz);
    double den = fact(2 * ix) * fact(2 * iy) * fact(2 * iz);
    return pow(2.0 * a / M_PI, 0.75) * sqrt(num / den);
}

/* ------------------------------------------------------------------ */
/* Boys function F_m(x), m = 0..mmax (eq 28 L209 is m = 0).            */
/* x < 35: ascending series for F_mmax, downward recursion;            */
/* x >= 35: F_0 from erf, upward recursion (textbook).      */
/* ------------------------------------------------------------------ */
void orc_boys(int mmax, double x, double *F)
{
    if (x < 35.0) {
        double ex = exp(-x);
        double term = 1.0 / (2.0 * mmax + 1.0);
        double sum = term;
        for (int k = 1; k < 400; ++k) {
            term *= 2.0 * x / (2.0 * mmax + 2.0 * k + 1.0);
            sum += term;
            if (term < 1e-17 * sum) break;
        }
        F[mmax] = ex * sum;
        for (int m = mmax; m > 0; --m)
            F[m - 1] = (2.0 * x * F[m] + ex) / (2.0 * m - 1.0);
    } else {
        double ex = exp(-x);
        double sx = sqrt(x);
        F[0] = 0.5 * sqrt(M_PI) * erf(sx) / sx;
        for (int m = 0; m < mmax; ++m)
            F[m + 1] = ((2.0 * m + 1.0) * F[m] - ex) / (2.0 * x);
    }
}

/* ------------------------------------------------------------------ */
/* E coefficients, one direction (eq 17-20).                 */
/* E[i][j][t], i <= la, j <= lb, t <= i+j; includes eq 19's Gaussian.  */
/* ------------------------------------------------------------------ */
static void hermite_E(int la, int lb, double a, double b, double Ax, double Bx,
                      double E[LMAX + 1][LMAX + 1][2 * LMAX + 1])
{
    double p = a + b, mu = a * b / p;
    double Px = (a * Ax + b * Bx) / p;
    double XPA = Px - Ax, XPB = Px - Bx;
    memset(E, 0, sizeof(double) * (LMAX + 1) * (LMAX + 1) * (2 * LMAX + 1));
    E[0][0][0] = exp(-mu * (Ax - Bx) * (Ax - Bx));          /* eq 19 */
    for (int i = 0; i < la; ++i)                            /* eq 17 */
        for (int t = 0; t <= i + 1; ++t) {
            double v = XPA * (t <= i ? E[i][0][t] : 0.0);
            if (t > 0) v += E[i][0][t - 1] / (2.0 * p);
            if (t + 1 <= i) v += (t + 1) * E[i][0][t + 1];
            E[i + 1][0][t] = v;
        }
    for (int i = 0; i <= la; ++i)                           /* eq 18 */
        for (int j = 0; j < lb; ++j)
            for (int t = 0; t <= i + j + 1; ++t) {
                double v = XPB * (t <= i + j ? E[i][j][t] : 0.0);
                if (t > 0) v += E[i][j][t - 1] / (2.0 * p);
                if (t + 1 <= i + j) v += (t + 1) * E[i][j][t + 1];
                E[i][j + 1][t] = v;
            }
}

/* ------------------------------------------------------------------ */
/* Hermite Coulomb integrals R^0_{tuv}(beta, L), t+u+v <= N            */
/* (eq 46-51).  Adds scale * R^0 into out[t][u][v].          */
/* ------------------------------------------------------------------ */
typedef double rtab[LTOT + 1][LTOT + 1][LTOT + 1];

static void hermite_R_add(int N, double beta, const double Lv[3], double scale, rtab out)
{
    double F[LTOT + 1];
    double r2 = Lv[0] * Lv[0] + Lv[1] * Lv[1] + Lv[2] * Lv[2];
    orc_boys(N, beta * r2, F);
    /* Rm[m][t][u][v], sized by the order actually needed */
    double Rm[N + 1][N + 1][N + 1][N + 1];
    memset(Rm, 0, sizeof(Rm));
    double f = 1.0;
    for (int m = 0; m <= N; ++m) { Rm[m][0][0][0] = f * F[m]; f *= -2.0 * beta; }   /* eq 50 */
    for (int n = 1; n <= N; ++n)                      /* total order t+u+v = n */
        for (int m = 0; m <= N - n; ++m)
            for (int t = 0; t <= n; ++t)
                for (int u = 0; u <= n - t; ++u) {
                    int v = n - t - u;
                    double val;
                    if (t > 0) {                                                   /* eq 47 */
                        val = Lv[0] * Rm[m + 1][t - 1][u][v];
                        if (t > 1) val += (t - 1) * Rm[m + 1][t - 2][u][v];
                    } else if (u > 0) {                                            /* eq 48 */
                        val = Lv[1] * Rm[m + 1][t][u - 1][v];
                        if (u > 1) val += (u - 1) * Rm[m + 1][t][u - 2][v];
                    } else {                                                       /* eq 49 */
                        val = Lv[2] * Rm[m + 1][t][u][v - 1];
                        if (v > 1) val += (v - 1) * Rm[m + 1][t][u][v - 2];
                    }
                    Rm[m][t][u][v] = val;
                }
    for (int t = 0; t <= N; ++t)
        for (int u = 0; u <= N - t; ++u)
            for (int v = 0; v <= N - t - u; ++v)
                out[t][u][v] += scale * Rm[0][t][u][v];
}

/* ------------------------------------------------------------------ */
/* One primitive pair distribution (bra or ket), local (one image).    */
/* ------------------------------------------------------------------ */
typedef struct {
    int la, lb;
    double a, b, p;
    double A[3], B[3], P[3];
    double E[3][LMAX + 1][LMAX + 1][2 * LMAX + 1];
} prim_pair;

static void make_prim_pair(prim_pair *pp, int la, int lb, double a, double b,
                           const double A[3], const double B[3])
{
    pp->la = la; pp->lb = lb; pp->a = a; pp->b = b; pp->p = a + b;
    for (int k = 0; k < 3; ++k) {
        pp->A[k] = A[k]; pp->B[k] = B[k];
        pp->P[k] = (a * A[k] + b * B[k]) / (a + b);     /* L131 */
        hermite_E(la, lb, a, b, A[k], B[k], pp->E[k]);
    }
}

/* E^{ab}_t for Cartesian components (ia of shell a, ib of shell b): product of the three
 * directions (eq 16).  Returns 0 outside the range (eq 20). */
static inline double E3(const prim_pair *pp, const int ca[3], const int cb[3], int t, int u, int v)
{
    if (t > ca[0] + cb[0] || u > ca[1] + cb[1] || v > ca[2] + cb[2]) return 0.0;
    return pp->E[0][ca[0]][cb[0]][t] * pp->E[1][ca[1]][cb[1]][u] * pp->E[2][ca[2]][cb[2]][v];
}

/*
 * Real-space primitive quartet block for one separation vector L = Q - P (+T1):
 *   out[ia][ib][ic][id] += 2 pi^{5/2}/(pq sqrt(p+q)) sum_t E^{ab}_t sum_s E^{cd}_s (-1)^{|t|} Rk_{t+s}(L)
 * kernel: 0 = 1/r ; 1 = erfc(w r)/r (full minus theta*attenuated) ; 2 = erf(w r)/r.
 * Unnormalised primitives (norms and contraction coefficients applied by the caller).
 */
static void prim_quartet_block(const prim_pair *bra, const prim_pair *ket, const double Lv[3],
                               int kernel, double omega, double *out /* na*nb*nc*nd */)
{
    int la = bra->la, lb = bra->lb, lc = ket->la, ld = ket->lb;
    int Lb = la + lb, Lk = lc + ld, N = Lb + Lk;
    double p = bra->p, q = ket->p;
    double alpha = p * q / (p + q);
    rtab R;
    for (int t = 0; t <= N; ++t)
        for (int u = 0; u <= N; ++u)
            for (int v = 0; v <= N; ++v) R[t][u][v] = 0.0;
    if (kernel == 0 || kernel == 1) hermite_R_add(N, alpha, Lv, 1.0, R);
    if (kernel == 1 || kernel == 2) {
        double aw = 1.0 / (1.0 / p + 1.0 / q + 1.0 / (omega * omega));
        double theta = omega * sqrt(p + q) / sqrt(p * q + omega * omega * (p + q));   /* eq 56 */
        hermite_R_add(N, aw, Lv, kernel == 1 ? -theta : theta, R);
    }
    double pref = 2.0 * pow(M_PI, 2.5) / (p * q * sqrt(p + q));                       /* eq 55 */
    int na = ncart(la), nb = ncart(lb), nc = ncart(lc), nd = ncart(ld);
    /* X[t][u][v] for a fixed ket component pair, then sum over t with the bra E */
    for (int ic = 0; ic < nc; ++ic)
        for (int id = 0; id < nd; ++id) {
            int cc[3], cd[3];
            cart_comp(lc, ic, &cc[0], &cc[1], &cc[2]);
            cart_comp(ld, id, &cd[0], &cd[1], &cd[2]);
            double X[2 * LMAX + 1][2 * LMAX + 1][2 * LMAX + 1];
            for (int t = 0; t <= Lb; ++t)
                for (int u = 0; u <= Lb - t; ++u)
                    for (int v = 0; v <= Lb - t - u; ++v) {
                        double s = 0.0;
                        for (int st = 0; st <= cc[0] + cd[0]; ++st)
                            for (int su = 0; su <= cc[1] + cd[1]; ++su)
                                for (int sv = 0; sv <= cc[2] + cd[2]; ++sv)
                                    s += E3(ket, cc, cd, st, su, sv) * R[t + st][u + su][v + sv];
                        X[t][u][v] = s;
                    }
            for (int ia = 0; ia < na; ++ia)
                for (int ib = 0; ib < nb; ++ib) {
                    int ca[3], cb[3];
                    cart_comp(la, ia, &ca[0], &ca[1], &ca[2]);
                    cart_comp(lb, ib, &cb[0], &cb[1], &cb[2]);
                    double s = 0.0;
                    for (int t = 0; t <= ca[0] + cb[0]; ++t)
                        for (int u = 0; u <= ca[1] + cb[1]; ++u)
                            for (int v = 0; v <= ca[2] + cb[2]; ++v) {
                                double sgn = ((t + u + v) & 1) ? -1.0 : 1.0;       /* C-4 */
                                s += sgn * E3(bra, ca, cb, t, u, v) * X[t][u][v];
                            }
                    out[((ia * nb + ib) * nc + ic) * nd + id] += pref * s;
                }
        }
}

/*
 * Public: non-periodic primitive quartet over NORMALISED primitive Cartesian
 * Gaussians (eq 5-6), kernel as above.  Used by pins P1 (closed form) and P11
 * (finite differences).  out has na*nb*nc*nd entries, overwritten.
 */
void orc_prim_eri(int kernel, double omega,
                  int la, double a, const double *A, int lb, double b, const double *B,
                  int lc, double c, const double *C, int ld, double d, const double *D,
                  double *out)
{
    prim_pair bra, ket;
    make_prim_pair(&bra, la, lb, a, b, A, B);
    make_prim_pair(&ket, lc, ld, c, d, C, D);
    double Lv[3] = { ket.P[0] - bra.P[0], ket.P[1] - bra.P[1], ket.P[2] - bra.P[2] };
    int na = ncart(la), nb = ncart(lb), nc = ncart(lc), nd = ncart(ld);
    memset(out, 0, sizeof(double) * na * nb * nc * nd);
    prim_quartet_block(&bra, &ket, Lv, kernel, omega, out);
    for (int ia = 0; ia < na; ++ia)
        for (int ib = 0; ib < nb; ++ib)
            for (int ic = 0; ic < nc; ++ic)
                for (int id = 0; id < nd; ++id) {
                    int x, y, z;
                    double n = 1.0;
                    cart_comp(la, ia, &x, &y, &z); n *= prim_norm(a, x, y, z);
                    cart_comp(lb, ib, &x, &y, &z); n *= prim_norm(b, x, y, z);
                    cart_comp(lc, ic, &x, &y, &z); n *= prim_norm(c, x, y, z);
                    cart_comp(ld, id, &x, &y, &z); n *= prim_norm(d, x, y, z);
                    out[((ia * nb + ib) * nc + ic) * nd + id] *= n;
                }
}

/* ------------------------------------------------------------------ */
/* Lattice helpers                                                     */
/* ------------------------------------------------------------------ */
static double det3(const double *c)
{
    return c[0] * (c[4] * c[8] - c[5] * c[7]) - c[1] * (c[3] * c[8] - c[5] * c[6])
         + c[2] * (c[3] * c[7] - c[4] * c[6]);
}

/* reciprocal vectors b_i (rows), a_i . b_j = 2 pi delta_ij */
static void recip(const double *c, double *b)
{
    double d = det3(c);
    const double *a1 = c, *a2 = c + 3, *a3 = c + 6;
    double f = 2.0 * M_PI / d;
    b[0] = f * (a2[1] * a3[2] - a2[2] * a3[1]); b[1] = f * (a2[2] * a3[0] - a2[0] * a3[2]); b[2] = f * (a2[0] * a3[1] - a2[1] * a3[0]);
    b[3] = f * (a3[1] * a1[2] - a3[2] * a1[1]); b[4] = f * (a3[2] * a1[0] - a3[0] * a1[2]); b[5] = f * (a3[0] * a1[1] - a3[1] * a1[0]);
    b[6] = f * (a1[1] * a2[2] - a1[2] * a2[1]); b[7] = f * (a1[2] * a2[0] - a1[0] * a2[2]); b[8] = f * (a1[0] * a2[1] - a1[1] * a2[0]);
}

static double norm3(const double *v) { return sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]); }

/*
 * All translations T = n1 a1 + n2 a2 + n3 a3 with |T - c| < r (O2: plain triple loop with
 * bounds from the reciprocal vectors: |n_i - f_i| <= r |b_i| / 2 pi).  Returns count;
 * fills T (3*cap doubles) and n (3*cap ints, may be NULL) up to cap.
 */
static int translations_in_sphere(const double *cell, const double *bvec, const double c[3],
                                  double r, double **Tout, int **nout)
{
    double f[3], h[3];
    for (int i = 0; i < 3; ++i) {
        f[i] = (bvec[3 * i] * c[0] + bvec[3 * i + 1] * c[1] + bvec[3 * i + 2] * c[2]) / (2.0 * M_PI);
        h[i] = r * norm3(bvec + 3 * i) / (2.0 * M_PI);
    }
    int lo[3], hi[3];
    for (int i = 0; i < 3; ++i) { lo[i] = (int)floor(f[i] - h[i]); hi[i] = (int)ceil(f[i] + h[i]); }
    size_t cap = (size_t)(hi[0] - lo[0] + 1) * (hi[1] - lo[1] + 1) * (hi[2] - lo[2] + 1);
    double *T = malloc(sizeof(double) * 3 * (cap ? cap : 1));
    int *nn = malloc(sizeof(int) * 3 * (cap ? cap : 1));
    int cnt = 0;
    for (int n1 = lo[0]; n1 <= hi[0]; ++n1)
        for (int n2 = lo[1]; n2 <= hi[1]; ++n2)
            for (int n3 = lo[2]; n3 <= hi[2]; ++n3) {
                double t[3];
                for (int k = 0; k < 3; ++k) t[k] = n1 * cell[k] + n2 * cell[3 + k] + n3 * cell[6 + k];
                double d[3] = { t[0] - c[0], t[1] - c[1], t[2] - c[2] };
                if (d[0] * d[0] + d[1] * d[1] + d[2] * d[2] < r * r) {
                    T[3 * cnt] = t[0]; T[3 * cnt + 1] = t[1]; T[3 * cnt + 2] = t[2];
                    nn[3 * cnt] = n1; nn[3 * cnt + 1] = n2; nn[3 * cnt + 2] = n3;
                    ++cnt;
                }
            }
    *Tout = T;
    if (nout) *nout = nn; else free(nn);
    return cnt;
}

/* ------------------------------------------------------------------ */
/* Pair-image list (O3): all ORDERED shell pairs, all T2, all primitive */
/* pairs with |C_mu C_nu| e^{-mu_ab r^2} > delta_o.                     */
/* ------------------------------------------------------------------ */
typedef struct {
    int shA, shB;
    double ca, cb;           /* contraction coefficients (eq 4) */
    double bound;            /* max_comp |C_mu C_nu| * e^{-mu r^2} (eq 22 lhs) */
    prim_pair pp;
} pair_img;

typedef struct {
    int n;
    pair_img *v;
    int *by_first_off, *by_first;     /* CSR: pair-images with shA == s */
    int *by_second_off, *by_second;   /* CSR: pair-images with shB == s */
    int *ao_off;                      /* AO offset per shell, [nshell+1] */
    int nbf;
    double bvec[9], vol;
} pair_list;

static double max_norm(double a, int l)
{
    double m = 0;
    for (int k = 0; k < ncart(l); ++k) {
        int x, y, z; cart_comp(l, k, &x, &y, &z);
        double n = prim_norm(a, x, y, z);
        if (n > m) m = n;
    }
    return m;
}

static void build_pair_list(const orc_system *s, double delta_o, double rcut, pair_list *pl)
{
    int ns = s->nshell;
    recip(s->cell, pl->bvec);
    pl->vol = fabs(det3(s->cell));
    pl->ao_off = malloc(sizeof(int) * (ns + 1));
    pl->ao_off[0] = 0;
    for (int i = 0; i < ns; ++i) pl->ao_off[i + 1] = pl->ao_off[i] + ncart(s->sh_l[i]);
    pl->nbf = pl->ao_off[ns];
    size_t cap = 1024; pl->v = malloc(sizeof(pair_img) * cap); pl->n = 0;
    for (int A = 0; A < ns; ++A)
        for (int B = 0; B < ns; ++B) {
            const double *RA = s->xyz + 3 * s->sh_atom[A], *RB = s->xyz + 3 * s->sh_atom[B];
            int la = s->sh_l[A], lb = s->sh_l[B];
            for (int ia = 0; ia < s->sh_nprim[A]; ++ia)
                for (int ib = 0; ib < s->sh_nprim[B]; ++ib) {
                    double a = s->exps[s->sh_off[A] + ia], b = s->exps[s->sh_off[B] + ib];
                    double ca = s->coefs[s->sh_off[A] + ia], cb = s->coefs[s->sh_off[B] + ib];
                    double cc = fabs(ca * cb) * max_norm(a, la) * max_norm(b, lb);
                    double mu = a * b / (a + b);
                    if (cc <= delta_o) continue;
                    double r = sqrt(log(cc / delta_o) / mu);          /* eq 23 with delta_o */
                    if (rcut > 0 && r > rcut) r = rcut;                /* C-14 */
                    double c[3] = { RA[0] - RB[0], RA[1] - RB[1], RA[2] - RB[2] };
                    double *T; int nT = translations_in_sphere(s->cell, pl->bvec, c, r, &T, NULL);
                    for (int k = 0; k < nT; ++k) {
                        double Bt[3] = { RB[0] + T[3 * k], RB[1] + T[3 * k + 1], RB[2] + T[3 * k + 2] };
                        double d2 = 0; for (int x = 0; x < 3; ++x) d2 += (RA[x] - Bt[x]) * (RA[x] - Bt[x]);
                        double bound = cc * exp(-mu * d2);
                        if (bound <= delta_o) continue;
                        if ((size_t)pl->n == cap) { cap *= 2; pl->v = realloc(pl->v, sizeof(pair_img) * cap); }
                        pair_img *pi = &pl->v[pl->n++];
                        pi->shA = A; pi->shB = B; pi->ca = ca; pi->cb = cb; pi->bound = bound;
                        make_prim_pair(&pi->pp, la, lb, a, b, RA, Bt);
                    }
                    free(T);
                }
        }
    /* CSR indices */
    pl->by_first_off = calloc(ns + 1, sizeof(int)); pl->by_second_off = calloc(ns + 1, sizeof(int));
    for (int i = 0; i < pl->n; ++i) { pl->by_first_off[pl->v[i].shA + 1]++; pl->by_second_off[pl->v[i].shB + 1]++; }
    for (int i = 0; i < ns; ++i) { pl->by_first_off[i + 1] += pl->by_first_off[i]; pl->by_second_off[i + 1] += pl->by_second_off[i]; }
    pl->by_first = malloc(sizeof(int) * (pl->n ? pl->n : 1)); pl->by_second = malloc(sizeof(int) * (pl->n ? pl->n : 1));
    int *c1 = calloc(ns, sizeof(int)), *c2 = calloc(ns, sizeof(int));
    for (int i = 0; i < pl->n; ++i) {
        int A = pl->v[i].shA, B = pl->v[i].shB;
        pl->by_first[pl->by_first_off[A] + c1[A]++] = i;
        pl->by_second[pl->by_second_off[B] + c2[B]++] = i;
    }
    free(c1); free(c2);
}

static void free_pair_list(pair_list *pl)
{
    free(pl->v); free(pl->by_first_off); free(pl->by_first); free(pl->by_second_off);
    free(pl->by_second); free(pl->ao_off);
}

/* normalised, contracted coefficient of component k of a primitive (C_mu, L76) */
static void comp_coefs(double coef, double a, int l, double *out)
{
    for (int k = 0; k < ncart(l); ++k) {
        int x, y, z; cart_comp(l, k, &x, &y, &z);
        out[k] = coef * prim_norm(a, x, y, z);
    }
}

/* ------------------------------------------------------------------ */
/* Overlap matrix (eq 21)                                         */
/* ------------------------------------------------------------------ */
static void overlap_from_list(const orc_system *s, const pair_list *pl, double *S)
{
    int N = pl->nbf;
    memset(S, 0, sizeof(double) * N * N);
    for (int i = 0; i < pl->n; ++i) {
        const pair_img *pi = &pl->v[i];
        int la = pi->pp.la, lb = pi->pp.lb;
        double Ca[6], Cb[6];
        comp_coefs(pi->ca, pi->pp.a, la, Ca); comp_coefs(pi->cb, pi->pp.b, lb, Cb);
        double g = pow(M_PI / pi->pp.p, 1.5);
        for (int ka = 0; ka < ncart(la); ++ka)
            for (int kb = 0; kb < ncart(lb); ++kb) {
                int ca[3], cb[3];
                cart_comp(la, ka, &ca[0], &ca[1], &ca[2]); cart_comp(lb, kb, &cb[0], &cb[1], &cb[2]);
                S[(size_t)(pl->ao_off[pi->shA] + ka) * N + pl->ao_off[pi->shB] + kb] +=
                    Ca[ka] * Cb[kb] * E3(&pi->pp, ca, cb, 0, 0, 0) * g;
            }
    }
    (void)s;
}

int orc_nbf(const orc_system *s)
{
    int n = 0; for (int i = 0; i < s->nshell; ++i) n += ncart(s->sh_l[i]); return n;
}

int orc_overlap(const orc_system *s, double delta_o, double rcut, double *S)
{
    pair_list pl; build_pair_list(s, delta_o, rcut, &pl);
    overlap_from_list(s, &pl, S);
    int n = pl.n; free_pair_list(&pl); return n;
}

/* ------------------------------------------------------------------ */
/* rho_ab(G) of one pair-image for all component pairs:                */
/*  C_mu C_nu (pi/p)^{3/2} e^{-G^2/4p} e^{-iG.P} sum_t E_t (-iG)^t      */
/* (SURVEY 8(c) LR; derivative of the Gaussian's transform, eq 31-33). */
/* ------------------------------------------------------------------ */
static void pair_rho_G(const pair_img *pi, const double G[3], double *re, double *im /* na*nb */)
{
    const prim_pair *pp = &pi->pp;
    int la = pp->la, lb = pp->lb;
    double G2 = G[0] * G[0] + G[1] * G[1] + G[2] * G[2];
    double g = pow(M_PI / pp->p, 1.5) * exp(-G2 / (4.0 * pp->p));
    double ph = -(G[0] * pp->P[0] + G[1] * pp->P[1] + G[2] * pp->P[2]);
    double cr = cos(ph), ci = sin(ph);
    double Ca[6], Cb[6];
    comp_coefs(pi->ca, pp->a, la, Ca); comp_coefs(pi->cb, pp->b, lb, Cb);
    /* (-i)^n : n mod 4 -> (1,0),(0,-1),(-1,0),(0,1) */
    static const double mr[4] = { 1, 0, -1, 0 }, mi[4] = { 0, -1, 0, 1 };
    for (int ka = 0; ka < ncart(la); ++ka)
        for (int kb = 0; kb < ncart(lb); ++kb) {
            int ca[3], cb[3];
            cart_comp(la, ka, &ca[0], &ca[1], &ca[2]); cart_comp(lb, kb, &cb[0], &cb[1], &cb[2]);
            double sr = 0, si = 0;
            for (int t = 0; t <= ca[0] + cb[0]; ++t)
                for (int u = 0; u <= ca[1] + cb[1]; ++u)
                    for (int v = 0; v <= ca[2] + cb[2]; ++v) {
                        double e = E3(pp, ca, cb, t, u, v) * pow(G[0], t) * pow(G[1], u) * pow(G[2], v);
                        int n = (t + u + v) & 3;
                        sr += e * mr[n]; si += e * mi[n];
                    }
            double c = Ca[ka] * Cb[kb] * g;
            re[ka * ncart(lb) + kb] = c * (sr * cr - si * ci);
            im[ka * ncart(lb) + kb] = c * (sr * ci + si * cr);
        }
}

/* ------------------------------------------------------------------ */
/* J and K, parts returned separately.                                 */
/* blocks: nblk < 0 -> every (shell, shell) block; else the listed     */
/* (blk_mu[i], blk_nu[i]) shell blocks only (sampled mode). */
/* which: bit 0 = J, bit 1 = K.  parts: bit 0 SR, bit 1 LR, bit 2 SELF.*/
/* counts[0] = SR primitive quartets (incl. T1) evaluated for J,       */
/* counts[1] = same for K, counts[2] = pair-images, counts[3] = N_G.   */
/* ------------------------------------------------------------------ */
typedef struct {
    double delta_o;     /* pair / Ewald truncation of the oracle, default 1e-18 ("unscreened") */
    double r_cut;       /* >0: cap on |A-B-T2| and |Q-P+T1| (C-14) */
    double g_cut;       /* >0: |G| cutoff; 0: 2 w sqrt(ln(1/delta_o)) */
    int32_t which, parts;
    double g_min;       /* >0: only G with |G| >= g_min enter the LR sum (selection only: lets a test compare the */
                        /* outermost shell of G at full basis size without paying for the whole sphere)           */
} orc_opts;

static void sr_block(const orc_system *s, const pair_list *pl, const orc_opts *o, double omega,
                     const double *P, int M, int Nsh, int isK, double *out /* N*N */, long long *count)
{
    int N = pl->nbf;
    int lM = s->sh_l[M], lN = s->sh_l[Nsh];
    int nM = ncart(lM), nN = ncart(lN);
    /* bra candidates */
    int nb0 = pl->by_first_off[M], nb1 = pl->by_first_off[M + 1];
    long long cnt = 0;
    double acc_tot[36]; memset(acc_tot, 0, sizeof(acc_tot));
#pragma omp parallel reduction(+ : cnt)
    {
        double acc[36]; memset(acc, 0, sizeof(acc));
        double *blk = malloc(sizeof(double) * 1296);
#pragma omp for schedule(dynamic, 1)
        for (int ib = nb0; ib < nb1; ++ib) {
            const pair_img *bra = &pl->v[pl->by_first[ib]];
            if (!isK && bra->shB != Nsh) continue;
            int la = bra->pp.la, lb = bra->pp.lb, na = ncart(la), nb = ncart(lb);
            double Ca[6], Cb[6];
            comp_coefs(bra->ca, bra->pp.a, la, Ca); comp_coefs(bra->cb, bra->pp.b, lb, Cb);
            /* ket candidates: J: all pair-images; K: those whose second shell is Nsh */
            int k0 = isK ? pl->by_second_off[Nsh] : 0;
            int k1 = isK ? pl->by_second_off[Nsh + 1] : pl->n;
            for (int ik = k0; ik < k1; ++ik) {
                const pair_img *ket = isK ? &pl->v[pl->by_second[ik]] : &pl->v[ik];
                double p = bra->pp.p, q = ket->pp.p;
                double pref = 2.0 * pow(M_PI, 2.5) / (p * q * sqrt(p + q));
                double theta = omega * sqrt(p + q) / sqrt(p * q + omega * omega * (p + q));
                double C2e = bra->bound * ket->bound * pref * (1.0 - theta);        /* eq 67 */
                if (C2e <= o->delta_o) continue;
                double aw = 1.0 / (1.0 / p + 1.0 / q + 1.0 / (omega * omega));
                double r = sqrt(log(C2e / o->delta_o) / aw);                         /* eq 68 */
                if (o->r_cut > 0 && r > o->r_cut) r = o->r_cut;
                double c[3] = { bra->pp.P[0] - ket->pp.P[0], bra->pp.P[1] - ket->pp.P[1], bra->pp.P[2] - ket->pp.P[2] };
                double *T; int nT = translations_in_sphere(s->cell, pl->bvec, c, r, &T, NULL);
                if (nT == 0) { free(T); continue; }
                int lc = ket->pp.la, ld = ket->pp.lb, nc = ncart(lc), nd = ncart(ld);
                double Cc[6], Cd[6];
                comp_coefs(ket->ca, ket->pp.a, lc, Cc); comp_coefs(ket->cb, ket->pp.b, ld, Cd);
                memset(blk, 0, sizeof(double) * na * nb * nc * nd);
                for (int k = 0; k < nT; ++k) {
                    double Lv[3] = { ket->pp.P[0] - bra->pp.P[0] + T[3 * k], ket->pp.P[1] - bra->pp.P[1] + T[3 * k + 1],
                                     ket->pp.P[2] - bra->pp.P[2] + T[3 * k + 2] };
                    prim_quartet_block(&bra->pp, &ket->pp, Lv, 1, omega, blk);
                    ++cnt;
                }
                free(T);
                int ob = pl->ao_off[bra->shB];
                int oc = pl->ao_off[ket->shA], od = pl->ao_off[ket->shB];
                for (int a = 0; a < na; ++a)
                    for (int b = 0; b < nb; ++b)
                        for (int cidx = 0; cidx < nc; ++cidx)
                            for (int d = 0; d < nd; ++d) {
                                double I = Ca[a] * Cb[b] * Cc[cidx] * Cd[d] * blk[((a * nb + b) * nc + cidx) * nd + d];
                                if (!isK)       /* J_ab += P_cd (ab|cd), eq 73 */
                                    acc[a * nN + b] += P[(size_t)(oc + cidx) * N + od + d] * I;
                                else            /* K_ad += P_bc (ab|cd), eq 74 */
                                    acc[a * nN + d] += P[(size_t)(ob + b) * N + oc + cidx] * I;
                            }
            }
        }
#pragma omp critical
        for (int i = 0; i < nM * nN; ++i) acc_tot[i] += acc[i];
        free(blk);
    }
    int oM = pl->ao_off[M], oN = pl->ao_off[Nsh];
    for (int a = 0; a < nM; ++a)
        for (int b = 0; b < nN; ++b) out[(size_t)(oM + a) * N + oN + b] += acc_tot[a * nN + b];
    *count += cnt;
}

int orc_jk(const orc_system *s, double omega, const orc_opts *o, const double *P,
           int nblk, const int32_t *blk_mu, const int32_t *blk_nu,
           double *Jsr, double *Jlr, double *Jself, double *Ksr, double *Klr, double *Kself,
           double *Sout, long long *counts)
{
    pair_list pl; build_pair_list(s, o->delta_o, o->r_cut, &pl);
    int N = pl.nbf, ns = s->nshell;
    size_t NN = (size_t)N * N;
    counts[0] = counts[1] = 0; counts[2] = pl.n; counts[3] = 0;
    int doJ = o->which & 1, doK = (o->which >> 1) & 1;
    double *S = malloc(sizeof(double) * NN);
    overlap_from_list(s, &pl, S);
    if (Sout) memcpy(Sout, S, sizeof(double) * NN);

    /* block list */
    int nb = nblk; int32_t *bm, *bn;
    if (nblk < 0) {
        nb = ns * ns; bm = malloc(sizeof(int32_t) * nb); bn = malloc(sizeof(int32_t) * nb);
        for (int i = 0; i < ns; ++i) for (int j = 0; j < ns; ++j) { bm[i * ns + j] = i; bn[i * ns + j] = j; }
    } else {
        bm = malloc(sizeof(int32_t) * (nb ? nb : 1)); bn = malloc(sizeof(int32_t) * (nb ? nb : 1));
        memcpy(bm, blk_mu, sizeof(int32_t) * nb); memcpy(bn, blk_nu, sizeof(int32_t) * nb);
    }
    if (nblk >= 0) {                       /* a block listed twice is computed once */
        char *seen = calloc((size_t)ns * ns, 1);
        int m = 0;
        for (int ib = 0; ib < nb; ++ib) {
            size_t key = (size_t)bm[ib] * ns + bn[ib];
            if (seen[key]) continue;
            seen[key] = 1; bm[m] = bm[ib]; bn[m] = bn[ib]; ++m;
        }
        nb = m; free(seen);
    }
    if (doJ) { memset(Jsr, 0, 8 * NN); memset(Jlr, 0, 8 * NN); memset(Jself, 0, 8 * NN); }
    if (doK) { memset(Ksr, 0, 8 * NN); memset(Klr, 0, 8 * NN); memset(Kself, 0, 8 * NN); }

    /* ---- SR (O5) ---- */
    if (o->parts & 1)
        for (int ib = 0; ib < nb; ++ib) {
            if (doJ) sr_block(s, &pl, o, omega, P, bm[ib], bn[ib], 0, Jsr, &counts[0]);
            if (doK) sr_block(s, &pl, o, omega, P, bm[ib], bn[ib], 1, Ksr, &counts[1]);
        }

    /* ---- LR (O6): full G sphere, G != 0, per G build A(G) from the pair-images ---- */
    if (o->parts & 2) {
        double gcut = o->g_cut > 0 ? o->g_cut : 2.0 * omega * sqrt(log(1.0 / o->delta_o));
        double zero[3] = { 0, 0, 0 };
        /* reciprocal lattice: treat b_i as a "cell" whose reciprocal is a_i (2 pi absorbed) */
        double *G; int nG;
        {
            double acell[9]; for (int i = 0; i < 9; ++i) acell[i] = s->cell[i];
            nG = translations_in_sphere(pl.bvec, acell, zero, gcut, &G, NULL);
        }
        counts[3] = 0;
        for (int ig = 0; ig < nG; ++ig) {
            double G2 = G[3 * ig] * G[3 * ig] + G[3 * ig + 1] * G[3 * ig + 1] + G[3 * ig + 2] * G[3 * ig + 2];
            if (G2 >= 1e-20 && !(o->g_min > 0 && G2 < o->g_min * o->g_min)) counts[3]++;
        }
        int nthr = 1;
#ifdef _OPENMP
        nthr = omp_get_max_threads();
#endif
        double *Jt = doJ ? calloc(NN * nthr, 8) : NULL, *Kt = doK ? calloc(NN * nthr, 8) : NULL;
        /* distinct nu shells among K blocks */
        char *isNu = calloc(ns, 1);
        for (int ib = 0; ib < nb; ++ib) isNu[bn[ib]] = 1;
#pragma omp parallel
        {
            int tid = 0;
#ifdef _OPENMP
            tid = omp_get_thread_num();
#endif
            double *Are = malloc(8 * NN), *Aim = malloc(8 * NN);
            double *yre = malloc(8 * (size_t)N * 6), *yim = malloc(8 * (size_t)N * 6);
            int *nzi = malloc(sizeof(int) * N); double *nzr = malloc(8 * (size_t)N), *nzm = malloc(8 * (size_t)N);
            double *myJ = doJ ? Jt + NN * tid : NULL, *myK = doK ? Kt + NN * tid : NULL;
#pragma omp for schedule(dynamic, 1)
            for (int ig = 0; ig < nG; ++ig) {
                const double *Gv = G + 3 * ig;
                double G2 = Gv[0] * Gv[0] + Gv[1] * Gv[1] + Gv[2] * Gv[2];
                if (G2 < 1e-20) continue;                                      /* G = 0 omitted (L253) */
                if (o->g_min > 0 && G2 < o->g_min * o->g_min) continue;        /* window selection (tests)   */
                double w = 4.0 * M_PI / (pl.vol * G2) * exp(-G2 / (4.0 * omega * omega));
                memset(Are, 0, 8 * NN); memset(Aim, 0, 8 * NN);
                double re[36], im[36];
                for (int i = 0; i < pl.n; ++i) {
                    const pair_img *pi = &pl.v[i];
                    int na = ncart(pi->pp.la), nbb = ncart(pi->pp.lb);
                    pair_rho_G(pi, Gv, re, im);
                    int oa = pl.ao_off[pi->shA], ob = pl.ao_off[pi->shB];
                    for (int a = 0; a < na; ++a)
                        for (int b = 0; b < nbb; ++b) {
                            Are[(size_t)(oa + a) * N + ob + b] += re[a * nbb + b];
                            Aim[(size_t)(oa + a) * N + ob + b] += im[a * nbb + b];
                        }
                }
                if (doJ) {
                    double rr = 0, ri = 0;                                     /* rho(G) = sum P o A */
                    for (size_t k = 0; k < NN; ++k) { rr += P[k] * Are[k]; ri += P[k] * Aim[k]; }
                    for (int ib = 0; ib < nb; ++ib) {
                        int oM = pl.ao_off[bm[ib]], oN = pl.ao_off[bn[ib]];
                        int nM = ncart(s->sh_l[bm[ib]]), nN = ncart(s->sh_l[bn[ib]]);
                        for (int a = 0; a < nM; ++a)
                            for (int b = 0; b < nN; ++b) {
                                size_t k = (size_t)(oM + a) * N + oN + b;
                                myJ[k] += w * (Are[k] * rr + Aim[k] * ri);     /* Re(conj(A) rho) */
                            }
                    }
                }
                if (doK) {
                    /* K += w Re( conj(A) P A ) on the requested blocks, grouped by nu shell */
                    for (int nu = 0; nu < ns; ++nu) {
                        if (!isNu[nu]) continue;
                        int oN = pl.ao_off[nu], nN = ncart(s->sh_l[nu]);
                        /* y[l][d] = sum_sg P[l][sg] A[sg][nu_d]  (P is not assumed symmetric) */
                        for (int d = 0; d < nN; ++d) {
                            int nnz = 0;
                            for (int sg = 0; sg < N; ++sg) {
                                double ar = Are[(size_t)sg * N + oN + d], ai = Aim[(size_t)sg * N + oN + d];
                                if (ar == 0.0 && ai == 0.0) continue;
                                nzi[nnz] = sg; nzr[nnz] = ar; nzm[nnz] = ai; ++nnz;
                            }
                            for (int l = 0; l < N; ++l) {
                                const double *Prow = P + (size_t)l * N;
                                double sr = 0, si = 0;
                                for (int k = 0; k < nnz; ++k) { sr += Prow[nzi[k]] * nzr[k]; si += Prow[nzi[k]] * nzm[k]; }
                                yre[(size_t)l * nN + d] = sr; yim[(size_t)l * nN + d] = si;
                            }
                        }
                        for (int ib = 0; ib < nb; ++ib) {
                            if (bn[ib] != nu) continue;
                            int oM = pl.ao_off[bm[ib]], nM = ncart(s->sh_l[bm[ib]]);
                            for (int a = 0; a < nM; ++a)
                                for (int d = 0; d < nN; ++d) {
                                    double sum = 0;
                                    for (int l = 0; l < N; ++l)
                                        sum += Are[(size_t)(oM + a) * N + l] * yre[(size_t)l * nN + d]
                                             + Aim[(size_t)(oM + a) * N + l] * yim[(size_t)l * nN + d];
                                    myK[(size_t)(oM + a) * N + oN + d] += w * sum;
                                }
                        }
                    }
                }
            }
            free(Are); free(Aim); free(yre); free(yim); free(nzi); free(nzr); free(nzm);
        }
        for (int t = 0; t < nthr; ++t) {
            if (doJ) for (size_t k = 0; k < NN; ++k) Jlr[k] += Jt[NN * t + k];
            if (doK) for (size_t k = 0; k < NN; ++k) Klr[k] += Kt[NN * t + k];
        }
        free(Jt); free(Kt); free(isNu); free(G);
    }

    /* ---- SELF (O7): J -= pi/(Omega w^2) tr(PS) S ; K -= pi/(Omega w^2) S P S ---- */
    if (o->parts & 4) {
        double c0 = M_PI / (pl.vol * omega * omega);
        double trPS = 0; for (size_t k = 0; k < NN; ++k) trPS += P[k] * S[k];
        for (int ib = 0; ib < nb; ++ib) {
            int oM = pl.ao_off[bm[ib]], oN = pl.ao_off[bn[ib]];
            int nM = ncart(s->sh_l[bm[ib]]), nN = ncart(s->sh_l[bn[ib]]);
            for (int a = 0; a < nM; ++a)
                for (int b = 0; b < nN; ++b) {
                    size_t k = (size_t)(oM + a) * N + oN + b;
                    if (doJ) Jself[k] = -c0 * trPS * S[k];
                    if (doK) {
                        double sum = 0;
                        for (int l = 0; l < N; ++l) {
                            double sl = S[(size_t)(oM + a) * N + l];
                            if (sl == 0.0) continue;
                            const double *Prow = P + (size_t)l * N;
                            double t = 0;
                            for (int sg = 0; sg < N; ++sg) t += Prow[sg] * S[(size_t)sg * N + oN + b];
                            sum += sl * t;
                        }
                        Kself[k] = -c0 * sum;
                    }
                }
        }
    }
    free(S); free(bm); free(bn); free_pair_list(&pl);
    return 0;
}

/* ------------------------------------------------------------------ */
/* One-electron Ewald terms: kinetic matrix, nuclear     */
/* attraction matrix, nuclear repulsion energy.  Gamma point.            */
/* ------------------------------------------------------------------ */

/* E^{ij}_0 ... of one direction for i <= la, j <= lb (eq 17-20), any la, lb: the kinetic integral needs j up to l + 2 */
static void hermite_E_n(int la, int lb, double a, double b, double Ax, double Bx, int dj, int dt, double *E /* [la+1][dj][dt] */)
{
    double p = a + b, mu = a * b / p;
    double Px = (a * Ax + b * Bx) / p;
    double XPA = Px - Ax, XPB = Px - Bx;
#define EE(i, j, t) E[((i) * dj + (j)) * dt + (t)]
    for (int i = 0; i <= la; ++i) for (int j = 0; j < dj; ++j) for (int t = 0; t < dt; ++t) EE(i, j, t) = 0.0;
    EE(0, 0, 0) = exp(-mu * (Ax - Bx) * (Ax - Bx));                                  /* eq 19 */
    for (int i = 0; i < la; ++i)                                                     /* eq 17 */
        for (int t = 0; t <= i + 1; ++t) {
            double v = XPA * (t <= i ? EE(i, 0, t) : 0.0);
            if (t > 0) v += EE(i, 0, t - 1) / (2.0 * p);
            if (t + 1 <= i) v += (t + 1) * EE(i, 0, t + 1);
            EE(i + 1, 0, t) = v;
        }
    for (int i = 0; i <= la; ++i)                                                    /* eq 18 */
        for (int j = 0; j < lb; ++j)
            for (int t = 0; t <= i + j + 1; ++t) {
                double v = XPB * (t <= i + j ? EE(i, j, t) : 0.0);
                if (t > 0) v += EE(i, j, t - 1) / (2.0 * p);
                if (t + 1 <= i + j) v += (t + 1) * EE(i, j, t + 1);
                EE(i, j + 1, t) = v;
            }
#undef EE
}

/*
 * T (SI eq S1): T_mn = sum_{R,prims} C_m C_n (pi/p)^{3/2} t_local, with per direction
 *   k_tau = -j(j-1)/2 E^{i,j-2}_0 + (2j+1) b E^{i,j}_0 - 2 b^2 E^{i,j+2}_0     (-1/2 d^2/dx^2 acting on the second function)
 *   t_local = k_x E_0y E_0z + E_0x k_y E_0z + E_0x E_0y k_z.
 * Reading C-27: PAPER.md prints the x bracket in full; the y and z brackets are garbled (the -2b^2 E^{j+2} term is
 * detached and repeated).  The Laplacian treats the three directions alike, so the x bracket is used for each.
 *
 * V (eq 52), per point charge q_C at C, L = C - P + R_C (so that the sign (-1)^{|t|} of reading C-4 applies):
 *   SR   = q_C C_m C_n (2 pi/p) sum_{R_C} sum_t (-1)^{|t|} E_t [ R^0_t(p, L) - theta R^0_t(a_w, L) ],
 *          theta = w/sqrt(p + w^2), a_w = p w^2/(p + w^2)
 *   LR   = sum_{G != 0} 4 pi/(Omega G^2) e^{-G^2/4w^2} Re[ conj(rho_mn(G)) q_C e^{-iG.C} ]
 *   SELF = -pi/(Omega w^2) S_mn q_C
 * Sign convention of the paper: V_mnC is the Coulomb interaction of the pair density with a charge +q_C under the
 * zero-mean periodic kernel; the electron-nucleus attraction matrix is -V with q_C = Z_C.
 *
 * E_nuc (eq 91); enuc[0] = reciprocal part, [1] = real-space part, [2] = constant terms, [3] = total.
 */
int orc_one_electron(const orc_system *s, double omega, const orc_opts *o, const double *charge /* natom */,
                     double *T, double *Vsr, double *Vlr, double *Vself, double *enuc)
{
    pair_list pl; build_pair_list(s, o->delta_o, o->r_cut, &pl);
    int N = pl.nbf;
    size_t NN = (size_t)N * N;
    memset(T, 0, 8 * NN); memset(Vsr, 0, 8 * NN); memset(Vlr, 0, 8 * NN); memset(Vself, 0, 8 * NN);
    double *S = malloc(8 * NN); overlap_from_list(s, &pl, S);
    double qtot = 0.0; for (int c = 0; c < s->natom; ++c) qtot += charge[c];
    double w2 = omega * omega;
    /* ---- kinetic ---- */
    for (int ip = 0; ip < pl.n; ++ip) {
        const pair_img *pi = &pl.v[ip];
        const prim_pair *pp = &pi->pp;
        int la = pp->la, lb = pp->lb;
        enum { DJ = LMAX + 3, DT = 2 * LMAX + 3 };
        double E[3][(LMAX + 1) * DJ * DT];
        for (int k = 0; k < 3; ++k) hermite_E_n(la, lb + 2, pp->a, pp->b, pp->A[k], pp->B[k], DJ, DT, E[k]);
#define E0(k, i, j) ((j) < 0 ? 0.0 : E[k][((i) * DJ + (j)) * DT])
        double Ca[6], Cb[6];
        comp_coefs(pi->ca, pp->a, la, Ca); comp_coefs(pi->cb, pp->b, lb, Cb);
        double g = pow(M_PI / pp->p, 1.5), b = pp->b;
        for (int ka = 0; ka < ncart(la); ++ka)
            for (int kb = 0; kb < ncart(lb); ++kb) {
                int ca[3], cb[3];
                cart_comp(la, ka, &ca[0], &ca[1], &ca[2]); cart_comp(lb, kb, &cb[0], &cb[1], &cb[2]);
                double e0[3], kk[3];
                for (int k = 0; k < 3; ++k) {
                    int i = ca[k], j = cb[k];
                    e0[k] = E0(k, i, j);
                    kk[k] = -0.5 * j * (j - 1) * E0(k, i, j - 2) + (2 * j + 1) * b * E0(k, i, j) - 2.0 * b * b * E0(k, i, j + 2);
                }
                double t = kk[0] * e0[1] * e0[2] + e0[0] * kk[1] * e0[2] + e0[0] * e0[1] * kk[2];
                T[(size_t)(pl.ao_off[pi->shA] + ka) * N + pl.ao_off[pi->shB] + kb] += Ca[ka] * Cb[kb] * g * t;
            }
#undef E0
    }
    /* ---- V, short range ---- */
#pragma omp parallel for schedule(dynamic, 8)
    for (int ip = 0; ip < pl.n; ++ip) {
        const pair_img *pi = &pl.v[ip];
        const prim_pair *pp = &pi->pp;
        int la = pp->la, lb = pp->lb, Lb = la + lb;
        double p = pp->p;
        double theta = omega / sqrt(p + w2), aw = p * w2 / (p + w2);
        double Ca[6], Cb[6];
        comp_coefs(pi->ca, pp->a, la, Ca); comp_coefs(pi->cb, pp->b, lb, Cb);
        double acc[36]; for (int k = 0; k < 36; ++k) acc[k] = 0.0;
        for (int c = 0; c < s->natom; ++c) {
            if (charge[c] == 0.0) continue;
            double C1e = fabs(charge[c]) * pi->bound * 2.0 * M_PI / p;               /* eq 42 prefactor */
            double arg = C1e * (1.0 - theta) / o->delta_o;
            if (arg <= 1.0) continue;
            double r = sqrt((1.0 / p + 1.0 / w2) * log(arg));                        /* eq 43 */
            if (o->r_cut > 0 && r > o->r_cut) r = o->r_cut;
            const double *Cc = s->xyz + 3 * c;
            double ctr[3] = { pp->P[0] - Cc[0], pp->P[1] - Cc[1], pp->P[2] - Cc[2] };
            double *Tl; int nT = translations_in_sphere(s->cell, pl.bvec, ctr, r, &Tl, NULL);
            for (int k = 0; k < nT; ++k) {
                double Lv[3] = { Cc[0] + Tl[3 * k] - pp->P[0], Cc[1] + Tl[3 * k + 1] - pp->P[1], Cc[2] + Tl[3 * k + 2] - pp->P[2] };
                rtab R;
                for (int t = 0; t <= Lb; ++t) for (int u = 0; u <= Lb; ++u) for (int v = 0; v <= Lb; ++v) R[t][u][v] = 0.0;
                hermite_R_add(Lb, p, Lv, 1.0, R);
                hermite_R_add(Lb, aw, Lv, -theta, R);
                for (int ka = 0; ka < ncart(la); ++ka)
                    for (int kb = 0; kb < ncart(lb); ++kb) {
                        int ca[3], cb[3];
                        cart_comp(la, ka, &ca[0], &ca[1], &ca[2]); cart_comp(lb, kb, &cb[0], &cb[1], &cb[2]);
                        double sum = 0.0;
                        for (int t = 0; t <= ca[0] + cb[0]; ++t)
                            for (int u = 0; u <= ca[1] + cb[1]; ++u)
                                for (int v = 0; v <= ca[2] + cb[2]; ++v)
                                    sum += (((t + u + v) & 1) ? -1.0 : 1.0) * E3(pp, ca, cb, t, u, v) * R[t][u][v];
                        acc[ka * ncart(lb) + kb] += charge[c] * sum;
                    }
            }
            free(Tl);
        }
        for (int ka = 0; ka < ncart(la); ++ka)
            for (int kb = 0; kb < ncart(lb); ++kb) {
                double v = Ca[ka] * Cb[kb] * (2.0 * M_PI / p) * acc[ka * ncart(lb) + kb];
#pragma omp atomic
                Vsr[(size_t)(pl.ao_off[pi->shA] + ka) * N + pl.ao_off[pi->shB] + kb] += v;
            }
    }
    /* ---- V, long range; E_nuc reciprocal part ---- */
    double gcut = o->g_cut > 0 ? o->g_cut : 2.0 * omega * sqrt(log(1.0 / o->delta_o));
    double zero[3] = { 0, 0, 0 };
    double *G; int nG;
    {
        double acell[9]; for (int i = 0; i < 9; ++i) acell[i] = s->cell[i];
        nG = translations_in_sphere(pl.bvec, acell, zero, gcut, &G, NULL);
    }
    double e_lr = 0.0;
    for (int ig = 0; ig < nG; ++ig) {
        const double *Gv = G + 3 * ig;
        double G2 = Gv[0] * Gv[0] + Gv[1] * Gv[1] + Gv[2] * Gv[2];
        if (G2 < 1e-20) continue;
        double w = 4.0 * M_PI / (pl.vol * G2) * exp(-G2 / (4.0 * w2));
        double nr = 0.0, ni = 0.0;                                                    /* rho_nuc(G) = sum q_C e^{-iG.C} */
        for (int c = 0; c < s->natom; ++c) {
            double ph = -(Gv[0] * s->xyz[3 * c] + Gv[1] * s->xyz[3 * c + 1] + Gv[2] * s->xyz[3 * c + 2]);
            nr += charge[c] * cos(ph); ni += charge[c] * sin(ph);
        }
        e_lr += 0.5 * w * (nr * nr + ni * ni);          /* 1/2 sum_{A,B} q_A q_B cos(G.(A-B)), A = B included (eq 91) */
        double re[36], im[36];
        for (int i = 0; i < pl.n; ++i) {
            const pair_img *pi = &pl.v[i];
            int na = ncart(pi->pp.la), nb = ncart(pi->pp.lb);
            pair_rho_G(pi, Gv, re, im);
            for (int a = 0; a < na; ++a)
                for (int b = 0; b < nb; ++b)
                    Vlr[(size_t)(pl.ao_off[pi->shA] + a) * N + pl.ao_off[pi->shB] + b] += w * (re[a * nb + b] * nr + im[a * nb + b] * ni);
        }
    }
    free(G);
    /* ---- V, SELF ---- */
    for (size_t k = 0; k < NN; ++k) Vself[k] = -M_PI / (pl.vol * w2) * qtot * S[k];
    /* ---- E_nuc real-space part and constants (eq 91) ---- */
    double e_sr = 0.0, e_c = 0.0;
    {
        double rb = sqrt(log(1.0 / o->delta_o)) / omega;                               /* erfc(x) < e^{-x^2}: eq 92 */
        for (int a = 0; a < s->natom; ++a)
            for (int b = a; b < s->natom; ++b) {
                double d[3] = { s->xyz[3 * a] - s->xyz[3 * b], s->xyz[3 * a + 1] - s->xyz[3 * b + 1], s->xyz[3 * a + 2] - s->xyz[3 * b + 2] };
                double md[3] = { -d[0], -d[1], -d[2] };
                double *Tl; int nT = translations_in_sphere(s->cell, pl.bvec, md, rb, &Tl, NULL);
                double sum = 0.0;
                for (int k = 0; k < nT; ++k) {
                    double v[3] = { d[0] + Tl[3 * k], d[1] + Tl[3 * k + 1], d[2] + Tl[3 * k + 2] };
                    double r = norm3(v);
                    if (r < 1e-12) continue;                                           /* A = B, R = 0 */
                    sum += erfc(omega * r) / r;
                }
                free(Tl);
                e_sr += (a == b ? 0.5 : 1.0) * charge[a] * charge[b] * sum;
            }
        double q2 = 0.0; for (int a = 0; a < s->natom; ++a) q2 += charge[a] * charge[a];
        /* -4pi/(4 w^2 Omega) for every pair (A < B) and half of it for A = B: -pi/(Omega w^2) * qtot^2 / 2; -w/sqrt(pi) q_A^2 */
        e_c = -M_PI / (pl.vol * w2) * 0.5 * qtot * qtot - omega / sqrt(M_PI) * q2;
    }
    enuc[0] = e_lr; enuc[1] = e_sr; enuc[2] = e_c; enuc[3] = e_lr + e_sr + e_c;
    free(S);
    free_pair_list(&pl);
    return 0;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
