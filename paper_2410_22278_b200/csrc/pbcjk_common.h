// Internal data model of libpbc_jk (host setup <-> kernels).  Not part of the C ABI.
//
// Notation follows PAPER.md / SURVEY.md 8: primitive pair-image (a in shell A at its home position,
// b in shell B translated by R2): p = a+b, P = (aA + b(B+R2))/p (L131), coefficient
//   coef = c_a c_b N_a N_b exp(-ab/p |A-B-R2|^2) * sqrt(2) pi^{5/4} / p
// so that the eq-55 prefactor 2 pi^{5/2}/(p q sqrt(p+q)) of a quartet is coef_bra*coef_ket/sqrt(p+q).
// N_a is the eq-6 norm of the AXIS-ALIGNED component (x^l); the remaining per-component factor
// (sqrt(3) for d_xy, d_xz, d_yz) is folded into P on input and into J, K on output.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pbcjk {

constexpr int LMAX = 2;                 // s, p, d
constexpr int LTOT = 4 * LMAX;          // highest Hermite order of a quartet
constexpr int BOYS_NT = 8;              // Taylor terms (degree 7)
constexpr int BOYS_MCOL = 16;           // F_0..F_15 per table row = one 128-byte line
constexpr double BOYS_DX = 0.125;       // grid spacing
constexpr double BOYS_XMAX = 36.0;      // beyond: asymptotic form
constexpr int BOYS_ROWS = 289;          // 0, 1/8, ..., 36
constexpr double LN_PMAX_CAP = 13.8;    // ln(1e6): largest ln max|P'| the packed image range is validated for
constexpr float SCREEN_MARGIN = 2e-3f;  // slack (ln units) of the fp32 screen: it keeps a superset of the fp64 rule

__host__ __device__ constexpr int ncart(int l) { return (l + 1) * (l + 2) / 2; }
__host__ __device__ constexpr int nherm(int L) { return (L + 1) * (L + 2) * (L + 3) / 6; }
// flat index of Hermite (t,u,v): orders ascending; inside an order the Cartesian component order
// xx,xy,xz,yy,yz,zz.  hidx(t,u,v) - nherm(n-1) is the component index of a shell l = n.
__host__ __device__ constexpr int hidx(int t, int u, int v)
{
    int n = t + u + v;
    return n * (n + 1) * (n + 2) / 6 + (n - t) * (n - t + 1) / 2 + (n - t - u);
}

// ---- ordered primitive pair-images, sorted by (shell A, l of shell B, bound descending): K lists ----
struct PairListK {
    int n;
    const double *Px, *Py, *Pz, *p, *ip, *coef, *lb; // ip = 1/p, lb = ln(bound)
    const double *PAx, *PAy, *PAz, *PBx, *PBy, *PBz; // P - A, P - (B + R2)
    const int *aoB;                                  // AO offset of shell B
    const int *shB;                                  // shell index of B (row/column of the per-block max |P'|)
    const float4 *q4;                                // fp32 screen record: (P - A).xyz, lb  (relative to the home shell)
    const float *ipf;                                // fp32 1/p
    const float *rng;                                // ln|coef| + (l_A + l_B) ln(2p): fp32 range guard of the mixed mode
    const float *etabf;                              // fp32 copy of etab (mixed precision), same eoff
    const double *etab;                              // E^{AB}_t products of every entry (order: gen_sr_k.py)
    const long long *eoff;                           // [n] row start of entry i in etab
    const int *off;                                  // [nshell*3 + 1]: range of (A, lB)
    const double *ext;                               // [nshell*3]: max |P - A| in the range
    const double *ipmax;                             // [nshell*3]: max 1/p in the range
};

// ---- unordered primitive pair-images (shell A >= shell B), contiguous per shell pair ----
struct PairListU {
    int n, nsp;
    const double *Px, *Py, *Pz, *p, *ip, *coef, *lb;
    const double *PAx, *PAy, *PAz, *PBx, *PBy, *PBz;
    const double *bexp;                              // exponent b of the second (translated) primitive (kinetic integral)
    const int *sp;                                   // shell-pair index of each entry
    const int *sp_off;                               // [nsp + 1]
    const int *sp_shA, *sp_shB;                      // [nsp]
};

// ---- J kets: U entries regrouped by (atom of shell A, Hermite order Lk, bound descending) ----
struct KetListJ {
    int n, ngroup;                                   // ngroup = natom
    const double *Qx, *Qy, *Qz, *q, *iq, *coef, *lb;
    const int *uidx;                                 // index into U
    const int *off;                                  // [natom*5 + 1]
    const double *ext, *iqmax;                       // [natom*5]
    const double *gx, *gy, *gz;                      // [natom] group centre (atom position)
    const float4 *q4;                                // fp32 screen record: (Q - group centre).xyz, lb
    const float *iqf;                                // fp32 1/q
    const int *spA, *spB;                            // shells of the ket's pair (per-block max |P'| of the J screen)
    const int2 *goff;                                // [natom*5] (first ket, count) of the group
    const float4 *grec;                              // [natom*5] (ext, iqmax, lbmax, 0) of the group
    const float4 *g4;                                // [natom] atom position - g0
    double g0[3];                                    // reference point (cell centre); every atom lies within rc of it
    double rc;
    float lbmax[5], iqmaxall[5], extmax[5];          // per ket Hermite order: maxima over all groups
    int64_t dstride;                                 // D~[s*dstride + j]
};

struct Lattice {
    double a[9];        // rows a1,a2,a3
    double binv[9];     // f = binv * r  (fractional coordinates, rows = b_i / 2pi)
    double bnorm[3];    // |b_i| / 2pi   (half-width of the bounding box per unit radius, eq 99-103)
    double omega, omega2, iomega2;
    double volume;
};

struct ShellInfo {
    const int *l, *ao, *atom;       // [nshell]
    const double *cx, *cy, *cz;     // shell centre
    int nshell, nbf;
};

// counters (device, int64), one slot per kernel class:
//   J class index = LB*5 + LK (Hermite orders of bra and ket), K class index = ((la*3+lb)*3+lc)*3+ld
//   CNT_Q32_*: the part of CNT_Q_* evaluated in fp32 (mixed precision); CNT_FLAG: non-zero = max|P'| above LN_PMAX_CAP
constexpr int NCLS_J = 25, NCLS_K = 81;
enum { CNT_CAND_J = 0, CNT_Q_J = NCLS_J, CNT_CAND_K = 2 * NCLS_J, CNT_Q_K = 2 * NCLS_J + NCLS_K,
       CNT_Q32_J = 2 * NCLS_J + 2 * NCLS_K, CNT_Q32_K = 3 * NCLS_J + 2 * NCLS_K, CNT_FLAG = 3 * NCLS_J + 3 * NCLS_K,
       CNT_N = 3 * NCLS_J + 3 * NCLS_K + 1 };

}  // namespace pbcjk
