// Light kernels around the quartet kernels, and the reciprocal-space path.
//
//   rho_mn(G) = sum_{R2,prims} C_m C_n (pi/p)^{3/2} e^{-G^2/4p} e^{-iG.P} sum_t E^{mn}_t (-iG)^t
//   J^LR_mn   = sum_{G != 0} w(G) Re[conj(rho_mn(G)) rho(G)],  rho(G) = sum_ls P_ls rho_ls(G)   (eq 98 first term)
//   K^LR_mn   = sum_{G != 0} w(G) Re[sum_ls conj(rho_ml(G)) P_ls rho_sn(G)]
//             = sum_G w (Ar P Ar + Ai P Ai)      since rho_mn(G) = Ar + i Ai is symmetric in (m,n) at Gamma
//   SELF      = the G = 0 slot with weight -pi/(Omega w^2) and A = S                           (eq 35, eq 56 third term)
// Half sphere of G, +-G paired (factor 2 in w, L243).  A' = sqrt(w) A is stored so both GEMM
// operands carry the weight.  The K contraction is a dense FP64 GEMM over (G, lambda): it runs on
// the FP64 tensor cores (DMMA, mma.sync.m8n8k4.f64) -- tcgen05 has no f64 kind.
#include "pbcjk_lr.cuh"
#include "pbcjk_md.cuh"
#include <algorithm>
#include <cmath>
#include <mutex>

namespace pbcjk {

// ---------------------------------------------------------------- density prep (A4)
__global__ void scale_density_kernel(const double *__restrict__ P, double *__restrict__ Pp, float *__restrict__ Ppf, int N,
                                     int Np, const double *__restrict__ f, unsigned long long *maxbits)
{
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    double v = 0.0;
    if (idx < (size_t)N * N) {
        const int i = (int)(idx / N), j = (int)(idx % N);
        v = P[idx] * f[i] * f[j];
        Pp[(size_t)i * Np + j] = v;
        if (Ppf) Ppf[(size_t)i * Np + j] = (float)v;
        v = fabs(v);
    }
    // block maximum; one atomic per block (not on the quartet path)
    __shared__ double s[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double m = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) m = fmax(m, s[w]);
        atomicMax(maxbits, (unsigned long long)__double_as_longlong(m));
    }
}
__global__ void lnpmax_kernel(const unsigned long long *maxbits, double *lnPmax, unsigned long long *flag)
{
    double m = __longlong_as_double((long long)*maxbits);
    *lnPmax = log(fmax(m, 1e-300));
    // the lattice image range of the real-space scans was validated at create for max|P'| <= e^{LN_PMAX_CAP}
    if (*lnPmax > LN_PMAX_CAP) *flag = 1ull;
}
void launch_scale_density(const double *P, double *Pp, float *Ppf, int N, int Np, const double *fcomp,
                          unsigned long long *maxbits, double *lnPmax, unsigned long long *flag, cudaStream_t st)
{
    cudaMemsetAsync(maxbits, 0, sizeof(unsigned long long), st);
    const size_t tot = (size_t)N * N;
    scale_density_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(P, Pp, Ppf, N, Np, fcomp, maxbits);
    lnpmax_kernel<<<1, 1, 0, st>>>(maxbits, lnPmax, flag);
}

// ln(max |P'|) over every shell block (lambda, sigma) and its row maxima: the density-weighted screen
__global__ void density_blocks_kernel(const double *__restrict__ Pp, int Np, ShellInfo sh, float *__restrict__ lnPblk)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x, a = blockIdx.y;
    if (b >= sh.nshell) return;
    const int na = ncart(sh.l[a]), nb = ncart(sh.l[b]);
    const double *blk = Pp + (size_t)sh.ao[a] * Np + sh.ao[b];
    double m = 0.0;
    for (int i = 0; i < na; ++i)
        for (int j = 0; j < nb; ++j) m = fmax(m, fabs(blk[(size_t)i * Np + j]));
    // rounded up a little so that the fp32 value never undercuts the fp64 maximum
    lnPblk[(size_t)a * sh.nshell + b] = m > 0.0 ? (float)log(m) + 1e-5f : -200.f;
}
__global__ void density_rows_kernel(const float *__restrict__ lnPblk, int ns, float *__restrict__ lnProw)
{
    const int a = blockIdx.x;
    float m = -200.f;
    for (int b = threadIdx.x; b < ns; b += blockDim.x) m = fmaxf(m, lnPblk[(size_t)a * ns + b]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    __shared__ float s[8];
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) m = fmaxf(m, s[w]);
        lnProw[a] = m;
    }
}
__global__ void ket_density_kernel(const float *__restrict__ lnPblk, int ns, KetListJ KJ, float *__restrict__ kjP)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < KJ.n) kjP[j] = lnPblk[(size_t)KJ.spA[j] * ns + KJ.spB[j]];
}
void launch_density_blocks(const double *Pp, int Np, const ShellInfo &sh, const KetListJ &KJ, float *lnPblk, float *lnProw,
                           float *kjP, cudaStream_t st)
{
    dim3 grid((sh.nshell + 127) / 128, sh.nshell);
    density_blocks_kernel<<<grid, 128, 0, st>>>(Pp, Np, sh, lnPblk);
    density_rows_kernel<<<sh.nshell, 256, 0, st>>>(lnPblk, sh.nshell, lnProw);
    if (KJ.n > 0) ket_density_kernel<<<(KJ.n + 255) / 256, 256, 0, st>>>(lnPblk, sh.nshell, KJ, kjP);
}

__global__ void to_float_kernel(const double *__restrict__ src, float *__restrict__ dst, size_t n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = (float)src[i];
}
void launch_to_float(const double *src, float *dst, size_t n, cudaStream_t st)
{
    if (n == 0) return;
    to_float_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(src, dst, n);
}

// Hermite density of a ket primitive pair-image: D~_s = fac * sum_{cd} E^{cd}_s P'_cd   (eq 95)
// fac = 2 for shell(C) != shell(D): the pair (D, C - R3) is the same distribution translated.
__global__ void hermite_density_kernel(PairListU U, ShellInfo sh, KetListJ KJ, const double *__restrict__ Pp, int Np,
                                       double *__restrict__ Dt)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= KJ.n) return;
    const int u = KJ.uidx[j];
    const int sp = U.sp[u];
    const int A = U.sp_shA[sp], B = U.sp_shB[sp];
    const int la = sh.l[A], lb = sh.l[B];
    const double o2p = 0.5 * U.ip[u];
    E1Drt ex, ey, ez;
    ex.build(la, lb, U.PAx[u], U.PBx[u], o2p);
    ey.build(la, lb, U.PAy[u], U.PBy[u], o2p);
    ez.build(la, lb, U.PAz[u], U.PBz[u], o2p);
    double D[nherm(2 * LMAX)];
    const int L = la + lb, nh = nherm(L);
    for (int s = 0; s < nh; ++s) D[s] = 0.0;
    const int na = ncart(la), nb = ncart(lb);
    const double *Pb = Pp + (size_t)sh.ao[A] * Np + sh.ao[B];
    for (int a = 0; a < na; ++a)
        for (int b = 0; b < nb; ++b) {
            int ax, ay, az, bx, by, bz;
            cart_powers(la, a, ax, ay, az);
            cart_powers(lb, b, bx, by, bz);
            const double pv = Pb[(size_t)a * Np + b];
            for (int tx = 0; tx <= ax + bx; ++tx)
                for (int ty = 0; ty <= ay + by; ++ty)
                    for (int tz = 0; tz <= az + bz; ++tz)
                        D[hidx(tx, ty, tz)] += pv * ex.e[ax][bx][tx] * ey.e[ay][by][ty] * ez.e[az][bz][tz];
        }
    const double fac = (A != B) ? 2.0 : 1.0;
    for (int s = 0; s < nh; ++s) Dt[(size_t)s * KJ.dstride + j] = fac * D[s];
}
void launch_hermite_density(const PairListU &U, const ShellInfo &sh, const KetListJ &KJ, const double *Pp, int Np,
                            double *Dt, cudaStream_t st)
{
    if (KJ.n <= 0) return;
    hermite_density_kernel<<<(KJ.n + 127) / 128, 128, 0, st>>>(U, sh, KJ, Pp, Np, Dt);
}

// E^{AB}_t products of every ordered primitive pair-image (eq 16-20), row i at etab[eoff[i]]; order of a row:
// a in cart(lA), b in cart(lB), tx <= ax+bx, ty <= ay+by, tz <= az+bz (the order gen_sr_k.py assumes).  Runs once
// per geometry: the K quartet kernels read these rows instead of running the E recursion per quartet.
__global__ void etab_kernel(PairListK K, const int *__restrict__ lA, const int *__restrict__ lB, double *__restrict__ etab)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= K.n) return;
    const int la = lA[i], lb = lB[i];
    const double o2p = 0.5 * K.ip[i];
    E1Drt ex, ey, ez;
    ex.build(la, lb, K.PAx[i], K.PBx[i], o2p);
    ey.build(la, lb, K.PAy[i], K.PBy[i], o2p);
    ez.build(la, lb, K.PAz[i], K.PBz[i], o2p);
    double *row = etab + K.eoff[i];
    const int na = ncart(la), nb = ncart(lb);
    int n = 0;
    for (int a = 0; a < na; ++a)
        for (int b = 0; b < nb; ++b) {
            int ax, ay, az, bx, by, bz;
            cart_powers(la, a, ax, ay, az);
            cart_powers(lb, b, bx, by, bz);
            for (int tx = 0; tx <= ax + bx; ++tx)
                for (int ty = 0; ty <= ay + by; ++ty)
                    for (int tz = 0; tz <= az + bz; ++tz) row[n++] = ex.e[ax][bx][tx] * ey.e[ay][by][ty] * ez.e[az][bz][tz];
        }
}
void launch_etab(const PairListK &K, const int *lA, const int *lB, double *etab, cudaStream_t st)
{
    if (K.n <= 0) return;
    etab_kernel<<<(K.n + 127) / 128, 128, 0, st>>>(K, lA, lB, etab);
}

// J_ab = sum_{R2,prims} sum_t (-1)^{|t|} E^{ab}_t J_t  (eq 96-97); one warp per shell pair.
__global__ void j_backtransform_kernel(PairListU U, ShellInfo sh, const double *__restrict__ Jt, double *__restrict__ Jsr,
                                       int N)
{
    const int sp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (sp >= U.nsp) return;
    const int A = U.sp_shA[sp], B = U.sp_shB[sp];
    const int la = sh.l[A], lb = sh.l[B];
    const int na = ncart(la), nb = ncart(lb);
    double acc[36];
    for (int i = 0; i < 36; ++i) acc[i] = 0.0;
    for (int u = U.sp_off[sp] + lane; u < U.sp_off[sp + 1]; u += 32) {
        const double o2p = 0.5 * U.ip[u];
        E1Drt ex, ey, ez;
        ex.build(la, lb, U.PAx[u], U.PBx[u], o2p);
        ey.build(la, lb, U.PAy[u], U.PBy[u], o2p);
        ez.build(la, lb, U.PAz[u], U.PBz[u], o2p);
        for (int a = 0; a < na; ++a)
            for (int b = 0; b < nb; ++b) {
                int ax, ay, az, bx, by, bz;
                cart_powers(la, a, ax, ay, az);
                cart_powers(lb, b, bx, by, bz);
                double s = 0.0;
                for (int tx = 0; tx <= ax + bx; ++tx)
                    for (int ty = 0; ty <= ay + by; ++ty)
                        for (int tz = 0; tz <= az + bz; ++tz) {
                            double e = ex.e[ax][bx][tx] * ey.e[ay][by][ty] * ez.e[az][bz][tz];
                            if ((tx + ty + tz) & 1) e = -e;                       // reading C-4
                            s += e * Jt[(size_t)hidx(tx, ty, tz) * U.n + u];
                        }
                acc[a * nb + b] += s;
            }
    }
    for (int i = 0; i < na * nb; ++i) {
        double v = acc[i];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) {
            const int a = i / nb, b = i % nb;
            Jsr[(size_t)(sh.ao[A] + a) * N + sh.ao[B] + b] = v;
            if (A != B) Jsr[(size_t)(sh.ao[B] + b) * N + sh.ao[A] + a] = v;
        }
    }
}
void launch_j_backtransform(const PairListU &U, const ShellInfo &sh, const double *Jt, double *Jsr, int N,
                            cudaStream_t st)
{
    if (U.nsp <= 0) return;
    j_backtransform_kernel<<<(U.nsp + 3) / 4, 128, 0, st>>>(U, sh, Jt, Jsr, N);
}

// ---------------------------------------------------------------- rho_mn(G) generation (A7)
// Stack layout (slot fastest): A'[row*ld + col*S + slot], ld = Np*S, S = slots of the batch rounded up to 16
// (slot 2g = Re, 2g+1 = Im of G number g of the batch, weight sqrt(w) folded in; slots past the batch are 0).
// One block per shell pair of class (LA, LB), threads over the G of the batch: each thread writes its (Re, Im)
// pair as one 16-byte store, so a warp writes 512 contiguous bytes per matrix element.
// A CTA takes AGEN_PAIRS consecutive shell pairs of its class; with `rho_part` it also forms its share of
//   rho'[slot] = sum_mn P'_mn A'_mn[slot]      (eq 98 first term: the density's Fourier coefficients)
// from the values it has in registers -- one partial per (CTA, slot), summed in a fixed order by rho_final_kernel -- so
// the stored batch is not streamed a second time for it.
constexpr int AGEN_PAIRS = 8;
template <int LA, int LB>
__global__ void __launch_bounds__(64) agen_kernel(LRParams p, const int *__restrict__ sp_list, int nsp_cls, int g0, int nb, int S,
                                                  double w0, double *__restrict__ Astack, size_t ld, const double *__restrict__ Pp,
                                                  double *__restrict__ rho_part)
{
    constexpr int NA = ncart(LA), NB = ncart(LB);
    const int gl = blockIdx.y * blockDim.x + threadIdx.x;
    if (2 * gl >= S) return;
    double rr = 0.0, ri = 0.0;
    for (int ip = blockIdx.x * AGEN_PAIRS; ip < min((blockIdx.x + 1) * AGEN_PAIRS, nsp_cls); ++ip) {
    const int sp = sp_list[ip];
    const bool overlap = g0 < 0;
    const bool live = gl < nb;
    double Gx = 0, Gy = 0, Gz = 0, sw = live ? w0 : 0.0;
    if (!overlap && live) {
        Gx = p.Gx[g0 + gl]; Gy = p.Gy[g0 + gl]; Gz = p.Gz[g0 + gl]; sw = p.Gw[g0 + gl];
    }
    const double G2 = Gx * Gx + Gy * Gy + Gz * Gz;
    const PairListU &U = p.U;
    const int A = U.sp_shA[sp], B = U.sp_shB[sp];
    double accr[NA * NB], acci[NA * NB];
#pragma unroll
    for (int i = 0; i < NA * NB; ++i) { accr[i] = 0.0; acci[i] = 0.0; }
    if (live) {
        const double g[3] = {Gx, Gy, Gz};
        for (int u = U.sp_off[sp]; u < U.sp_off[sp + 1]; ++u) {
            const double pp = U.p[u], ip = U.ip[u];
            // coef holds sqrt2 pi^{5/4}/p; the transform needs (pi/p)^{3/2}
            const double cft = U.coef[u] * 0.94139626377671481 * rsqrt(pp) * exp(-0.25 * G2 * ip) * sw;
            double sn, cs;
            sincos(-(Gx * U.Px[u] + Gy * U.Py[u] + Gz * U.Pz[u]), &sn, &cs);
            const double phr = cft * cs, phi = cft * sn;
            const double o2p = 0.5 * ip;
            const double PA[3] = {U.PAx[u], U.PAy[u], U.PAz[u]}, PB[3] = {U.PBx[u], U.PBy[u], U.PBz[u]};
            // per direction: s[i][j] = sum_t E^{ij}_t (-iG)^t
            double sr[3][LA + 1][LB + 1], si[3][LA + 1][LB + 1];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                E1D<LA, LB> e;
                e.build(PA[d], PB[d], o2p);
                const double g1 = g[d], g2 = g1 * g1;
#pragma unroll
                for (int i = 0; i <= LA; ++i)
#pragma unroll
                    for (int j = 0; j <= LB; ++j) {
                        double r = e.e[i][j][0], im = 0.0;            // (-i)^t: 1, -i, -1, i
                        if (i + j >= 1) im = -e.e[i][j][1] * g1;
                        if (i + j >= 2) r = fma(-e.e[i][j][2], g2, r);
                        if (i + j >= 3) im = fma(e.e[i][j][3], g2 * g1, im);
                        if (i + j >= 4) r = fma(e.e[i][j][4], g2 * g2, r);
                        sr[d][i][j] = r; si[d][i][j] = im;
                    }
            }
#pragma unroll
            for (int a = 0; a < NA; ++a)
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    const int ax = cart_x(LA, a), ay = cart_y(LA, a), az = cart_z(LA, a);
                    const int bx = cart_x(LB, b), by = cart_y(LB, b), bz = cart_z(LB, b);
                    double r = sr[0][ax][bx], im = si[0][ax][bx];
                    const double r2 = r * sr[1][ay][by] - im * si[1][ay][by], i2 = r * si[1][ay][by] + im * sr[1][ay][by];
                    r = r2 * sr[2][az][bz] - i2 * si[2][az][bz];
                    im = r2 * si[2][az][bz] + i2 * sr[2][az][bz];
                    accr[a * NB + b] += r * phr - im * phi;
                    acci[a * NB + b] += r * phi + im * phr;
                }
        }
    }
    const int oa = p.sh.ao[A], ob = p.sh.ao[B];
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const double2 v = make_double2(accr[a * NB + b], overlap ? 0.0 : acci[a * NB + b]);
            *reinterpret_cast<double2 *>(Astack + (size_t)(oa + a) * ld + (size_t)(ob + b) * S + 2 * gl) = v;
            *reinterpret_cast<double2 *>(Astack + (size_t)(ob + b) * ld + (size_t)(oa + a) * S + 2 * gl) = v;
            if (rho_part) {
                const double pv = (A != B ? 2.0 : 1.0) * Pp[(size_t)(oa + a) * p.Np + ob + b];     // (m,n) and (n,m)
                rr = fma(pv, v.x, rr);
                ri = fma(pv, v.y, ri);
            }
        }
    }
    if (rho_part) *reinterpret_cast<double2 *>(rho_part + (size_t)blockIdx.x * S + 2 * gl) = make_double2(rr, ri);
}
static int agen_groups(const LRParams &p, int c) { return (p.n_sp_cls[c] + AGEN_PAIRS - 1) / AGEN_PAIRS; }
int agen_groups_total(const LRParams &p)
{
    int n = 0;
    for (int c = 0; c < 9; ++c) n += agen_groups(p, c);
    return n;
}
template <int LA, int LB>
static void launch_agen_class(const LRParams &p, int g0, int nb, int S, double w0, double *Astack, size_t ld, const double *Pp,
                              double *rho_part, cudaStream_t st)
{
    const int c = LA * 3 + LB, n = p.n_sp_cls[c];
    if (n <= 0) return;
    int goff = 0;
    for (int k = 0; k < c; ++k) goff += agen_groups(p, k);
    dim3 grid(agen_groups(p, c), (S / 2 + 63) / 64);
    agen_kernel<LA, LB><<<grid, 64, 0, st>>>(p, p.sp_cls[c], n, g0, nb, S, w0, Astack, ld, Pp,
                                              rho_part ? rho_part + (size_t)goff * S : nullptr);
}
int agen_launches(const LRParams &p)
{
    int n = 0;
    for (int c = 0; c < 9; ++c) n += p.n_sp_cls[c] > 0;
    return n;
}
static double *rho_partials(double *rho, int S);
// rho (optional): rho_scratch_doubles(S, groups) doubles -- S results (filled by launch_rho_final) then the per-CTA partials
void launch_agen(const LRParams &p, int g0, int nb, int S, double w0, double *Astack, const double *Pp, double *rho, cudaStream_t st)
{
    if (p.U.nsp <= 0 || nb <= 0) return;
    const size_t ld = (size_t)p.Np * S;
    double *part = rho ? rho_partials(rho, S) : nullptr;
#define AG(LA, LB) launch_agen_class<LA, LB>(p, g0, nb, S, w0, Astack, ld, Pp, part, st);
    AG(0, 0) AG(0, 1) AG(0, 2) AG(1, 0) AG(1, 1) AG(1, 2) AG(2, 0) AG(2, 1) AG(2, 2)
#undef AG
}

// rho'[slot] = sum over the agen CTAs' partials part[g][slot], in two fixed-order stages (deterministic): RHO_NB blocks each
// sum the partials g = b, b + RHO_NB, ... into part2[b][slot]; one block sums the RHO_NB rows.
constexpr int RHO_NB = 148;
__global__ void __launch_bounds__(128) rho_stage1_kernel(const double *__restrict__ part, int ngrp, int S, double *__restrict__ part2)
{
    const int slot = threadIdx.x;
    if (slot >= S) return;
    double t0 = 0.0, t1 = 0.0;
    int m = blockIdx.x;
    for (; m + RHO_NB < ngrp; m += 2 * RHO_NB) { t0 += part[(size_t)m * S + slot]; t1 += part[(size_t)(m + RHO_NB) * S + slot]; }
    if (m < ngrp) t0 += part[(size_t)m * S + slot];
    part2[(size_t)blockIdx.x * S + slot] = t0 + t1;
}
__global__ void __launch_bounds__(128) rho_stage2_kernel(const double *__restrict__ part2, int S, double *__restrict__ rho)
{
    const int slot = threadIdx.x;
    if (slot >= S) return;
    double r = 0.0;
    for (int b = 0; b < RHO_NB; ++b) r += part2[(size_t)b * S + slot];
    rho[slot] = r;
}
// layout of the scratch: S results | RHO_NB * S stage-1 sums | ngroups * S partials of the agen CTAs
int rho_scratch_doubles(int S, int ngroups) { return S * (1 + RHO_NB + ngroups); }
static double *rho_partials(double *rho, int S) { return rho + (size_t)S * (1 + RHO_NB); }
void launch_rho_final(const LRParams &p, int S, double *rho, cudaStream_t st)
{
    if (S <= 0) return;
    rho_stage1_kernel<<<RHO_NB, 128, 0, st>>>(rho_partials(rho, S), agen_groups_total(p), S, rho + S);
    rho_stage2_kernel<<<1, 128, 0, st>>>(rho + S, S, rho);
}

// Jacc[m][n] += sign * sum_slot A'[m][n][slot] rho'[slot]: one warp per matrix element, lanes over the slots.
// A'[m][n][.] and A'[n][m][.] hold the same bits (agen_kernel stores one value at both places), so only n <= m is read
// -- half of the batch -- and the sum goes to both elements.
__global__ void __launch_bounds__(256) jlr_accum_kernel(const double *__restrict__ Astack, size_t ld, int N, int S,
                                                        const double *__restrict__ rho, double sign, double *__restrict__ Jacc)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int m = blockIdx.y;
    double r[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) r[k] = lane + 32 * k < S ? rho[lane + 32 * k] : 0.0;
    for (int n = blockIdx.x * 8 + w; n <= m; n += gridDim.x * 8) {
        const double *a = Astack + (size_t)m * ld + (size_t)n * S;
        double acc = 0.0;
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (lane + 32 * k < S) acc = fma(a[lane + 32 * k], r[k], acc);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane == 0) {
            Jacc[(size_t)m * N + n] += sign * acc;
            if (n != m) Jacc[(size_t)n * N + m] += sign * acc;
        }
    }
}
void launch_jlr_accum(const double *Astack, int Np, int N, int S, const double *rho, double sign, double *Jacc, cudaStream_t st)
{
    if (S <= 0) return;
    dim3 grid(8, N);
    jlr_accum_kernel<<<grid, 256, 0, st>>>(Astack, (size_t)Np * S, N, S, rho, sign, Jacc);
}

// ---------------------------------------------------------------- FP64 tensor-core GEMM (A8, A9)
namespace {
constexpr int BM = 128, BN = 128, BK = 32;
constexpr int NSTAGE = 3;     // cp.async ring: tiles t+1, t+2 are in flight while tile t is multiplied, one barrier per tile
                              // (the kernel holds 166 registers x 256 threads: one CTA per SM, so nothing else hides the waits)
constexpr int SA = BK + 4;    // row stride of the A tile [m][k]: (lane/4)*20 + lane%4 hits every bank pair twice
constexpr int SB = BN + 8;    // row stride of the B tile [k][n]: (lane%4)*136 + lane/4 likewise

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}
}  // namespace

// C[z] = beta*C[z] + alpha * sum_{b in batches(z)} op(A_b) B_b
//   TA = false: A_b is row-major M x Kb (k contiguous);  TA = true: A_b is stored as Kb x M (m contiguous),
//   i.e. op(A) = A^T -- the Y^T Y form of the reciprocal-space K contraction.
//   dyn (device, may be null): dyn[0] = rank r of the factor P' = L L^T (or N in the fallback), dyn[1] = use B_alt.
//   use_dyn bit 0: only row tiles with bm*BM < r are computed; bit 1: Kb = roundup16(r); bit 2: B = B_alt if dyn[1];
//   bit 3: nbatch = r (the batches are the rows of the factor);
//   lower_only: tiles with bn > bm are skipped (symmetric result, completed in finalise).
//   TB = true: B_b is stored as Nc x Kb (k contiguous, ldb = row stride), i.e. C += op(A) B^T.
template <bool TA, bool TB>
__global__ void __launch_bounds__(256) dgemm_kernel(int Kb, int nbatch, double alpha, const double *__restrict__ A, size_t lda,
                                                    size_t strideA, const double *__restrict__ B, size_t ldb, size_t strideB,
                                                    double beta, double *__restrict__ C, size_t ldc, size_t strideC, int nsplit,
                                                    const int *__restrict__ dyn, int use_dyn, const double *__restrict__ B_alt,
                                                    int lower_only)
{
    extern __shared__ __align__(16) double smem[];
    constexpr int A_TILE = TA ? BK * SB : BM * SA;
    constexpr int B_TILE = TB ? BN * SA : BK * SB;
    double *As = smem;                       // [NSTAGE][A_TILE]
    double *Bs = smem + NSTAGE * A_TILE;     // [NSTAGE][B_TILE]
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int wm = w >> 2, wn = w & 3;
    const int bm = blockIdx.y, bn = blockIdx.x, z = blockIdx.z;
    if (lower_only && bn > bm) return;
    if (dyn) {
        const int r = dyn[0];
        if ((use_dyn & 1) && bm * BM >= r) return;
        if (use_dyn & 2) Kb = ((r + BK - 1) / BK) * BK;
        if ((use_dyn & 4) && dyn[1]) B = B_alt;
        if (use_dyn & 8) nbatch = r;
    }
    const int bat0 = (int)((long long)nbatch * z / nsplit), bat1 = (int)((long long)nbatch * (z + 1) / nsplit);
    const int kt_per = Kb / BK;
    const int ntile = (bat1 - bat0) * kt_per;
    C += (size_t)z * strideC;

    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    // Each thread copies 8 + 8 16-byte pieces per k-tile.  Their global addresses are one per-thread base pointer per operand
    // plus a multiple of a fixed stride, and the (batch, k) position of the next tile to fetch advances incrementally -- the
    // tiles are requested in order -- so that issuing a tile costs a few instructions per cp.async (the 64-bit index
    // arithmetic per piece, and a division per tile, took the DMMA warps of both schedulers off the pipe after every barrier).
    const double *gA, *gB;
    size_t stepA, stepB, kstepA, kstepB;
    int soffA, soffB;                                      // element offsets of this thread's first piece inside a stage
    if (TA) {
        gA = A + (size_t)bat0 * strideA + (size_t)(tid >> 6) * lda + bm * BM + (tid & 63) * 2;
        stepA = 4 * lda; kstepA = (size_t)BK * lda; soffA = (tid >> 6) * SB + (tid & 63) * 2;
    } else {
        gA = A + (size_t)bat0 * strideA + (size_t)(bm * BM + (tid >> 4)) * lda + (tid & 15) * 2;
        stepA = 16 * lda; kstepA = BK; soffA = (tid >> 4) * SA + (tid & 15) * 2;
    }
    if (TB) {
        gB = B + (size_t)bat0 * strideB + (size_t)(bn * BN + (tid >> 4)) * ldb + (tid & 15) * 2;
        stepB = 16 * ldb; kstepB = BK; soffB = (tid >> 4) * SA + (tid & 15) * 2;
    } else {
        gB = B + (size_t)bat0 * strideB + (size_t)(tid >> 6) * ldb + bn * BN + (tid & 63) * 2;
        stepB = 4 * ldb; kstepB = (size_t)BK * ldb; soffB = (tid >> 6) * SB + (tid & 63) * 2;
    }
    static_assert(BK == 32 && BM == 128 && BN == 128, "piece mapping of load_tile");
    int ld_kt = 0;                                          // k-tile of the next fetch inside its batch
    auto load_piece = [&](int buf, int i) {                 // piece i (0..7) of the A and of the B tile
        cp_async16(As + buf * A_TILE + soffA + i * (TA ? 4 * SB : 16 * SA), gA + i * stepA);
        cp_async16(Bs + buf * B_TILE + soffB + i * (TB ? 16 * SA : 4 * SB), gB + i * stepB);
    };
    auto load_advance = [&]() {
        asm volatile("cp.async.commit_group;\n" ::);
        if (++ld_kt == kt_per) {                            // next batch: back to k = 0
            ld_kt = 0;
            gA += strideA - (size_t)(kt_per - 1) * kstepA;
            gB += strideB - (size_t)(kt_per - 1) * kstepB;
        } else {
            gA += kstepA;
            gB += kstepB;
        }
    };

    // prologue: NSTAGE - 1 tiles in flight (empty commit groups keep the group count uniform)
#pragma unroll
    for (int t = 0; t < NSTAGE - 1; ++t) {
        if (t < ntile) {
#pragma unroll
            for (int i = 0; i < 8; ++i) load_piece(t, i);
            load_advance();
        }
        else asm volatile("cp.async.commit_group;\n" ::);
    }
    for (int t = 0; t < ntile; ++t) {
        const int buf = t % NSTAGE;
        asm volatile("cp.async.wait_group %0;\n" ::"n"(NSTAGE - 2));       // tile t has landed (for this thread)
        __syncthreads();                                                    // ... for all; and everyone is done with tile t-1
        // tile t + NSTAGE - 1 goes into the buffer of tile t-1: one A and one B piece per k-step, between the DMMAs
        const bool fetch = t + NSTAGE - 1 < ntile;
        const int fbuf = (t + NSTAGE - 1) % NSTAGE;
        const double *as = TA ? As + buf * A_TILE + (lane & 3) * SB + wm * 64 + (lane >> 2)
                              : As + buf * A_TILE + (wm * 64 + (lane >> 2)) * SA + (lane & 3);
        const double *bs = TB ? Bs + buf * B_TILE + (wn * 32 + (lane >> 2)) * SA + (lane & 3)
                              : Bs + buf * B_TILE + (lane & 3) * SB + wn * 32 + (lane >> 2);
#pragma unroll
        for (int kk = 0; kk < BK; kk += 4) {
            double a[8], b[4];
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = TA ? as[kk * SB + i * 8] : as[i * 8 * SA + kk];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = TB ? bs[j * 8 * SA + kk] : bs[kk * SB + j * 8];
            if (fetch) load_piece(fbuf, kk >> 2);
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
        if (fetch) load_advance();
        else asm volatile("cp.async.commit_group;\n" ::);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const size_t row = (size_t)bm * BM + wm * 64 + i * 8 + (lane >> 2);
            const size_t col = (size_t)bn * BN + wn * 32 + j * 8 + (lane & 3) * 2;
            double2 *dst = reinterpret_cast<double2 *>(C + row * ldc + col);
            double2 v = make_double2(alpha * acc[i][j][0], alpha * acc[i][j][1]);
            if (beta != 0.0) {
                const double2 o = *dst;
                v.x = fma(beta, o.x, v.x);
                v.y = fma(beta, o.y, v.y);
            }
            *dst = v;
        }
}

namespace {
constexpr int smemN = NSTAGE * (BM * SA + BK * SB) * (int)sizeof(double), smemT = NSTAGE * (2 * BK * SB) * (int)sizeof(double);
constexpr int smemNT = NSTAGE * (BM * SA + BN * SA) * (int)sizeof(double);
}  // namespace
// the opt-in is per device: pbc_jk_create calls this for the handle's device
void dgemm_set_attributes()
{
    cudaFuncSetAttribute(dgemm_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smemN);
    cudaFuncSetAttribute(dgemm_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smemT);
    cudaFuncSetAttribute(dgemm_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smemNT);
}
void launch_dgemm(const GemmArgs &g, cudaStream_t st)
{
    dim3 grid(g.Nc / BN, g.M / BM, g.nsplit);
    if (g.transA)
        dgemm_kernel<true, false><<<grid, 256, smemT, st>>>(g.Kb, g.nbatch, g.alpha, g.A, g.lda, g.strideA, g.B, g.ldb, g.strideB,
                                                            g.beta, g.C, g.ldc, g.strideC, g.nsplit, g.dyn, g.use_dyn, g.B_alt,
                                                            g.lower_only);
    else if (g.transB)
        dgemm_kernel<false, true><<<grid, 256, smemNT, st>>>(g.Kb, g.nbatch, g.alpha, g.A, g.lda, g.strideA, g.B, g.ldb, g.strideB,
                                                             g.beta, g.C, g.ldc, g.strideC, g.nsplit, g.dyn, g.use_dyn, g.B_alt,
                                                             g.lower_only);
    else
        dgemm_kernel<false, false><<<grid, 256, smemN, st>>>(g.Kb, g.nbatch, g.alpha, g.A, g.lda, g.strideA, g.B, g.ldb, g.strideB,
                                                             g.beta, g.C, g.ldc, g.strideC, g.nsplit, g.dyn, g.use_dyn, g.B_alt,
                                                             g.lower_only);
}

// ---------------------------------------------------------------- factor of P' for the K contraction (A8)
// K^LR = sum_G w Re[conj(A) P' A] costs 8 N^3 flop per G with a dense P'.  SCF densities are P = C C^T of rank
// n_occ << N, so P' = L L^T is factored once per build by a diagonally pivoted Cholesky decomposition (stop at
// residual diagonal <= 1e-13 max diag) and K^LR = sum_slots Y^T Y with Y = L^T A' (8 r N^2 flop per G).  A P' that is
// not positive semidefinite fails the residual test |P' - L L^T| and falls back, on the device, to L = P', r = N,
// K^LR = sum (P'A')^T A' -- same kernels, no host round trip.
//   dyn[0] = rank, dyn[1] = fallback flag, dyn[2] = done;  dscal[0] = max diag, dscal[1] = max |residual| (bits)
__global__ void chol_init_kernel(const double *__restrict__ Pp, int N, int Np, double *__restrict__ d0, int *dyn,
                                 double *dscal)
{
    __shared__ double s[32];
    double m = 0.0;
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        const double v = Pp[(size_t)i * Np + i];
        d0[i] = v;
        m = fmax(m, v);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) m = fmax(m, s[w]);
        dscal[0] = m;
        dscal[1] = 0.0;
        dyn[0] = 0; dyn[1] = 0; dyn[2] = 0;
    }
}

// All steps in ONE cooperative launch (the blocks are co-resident, so they may wait on one another): at step k every
// block finds the pivot (largest residual diagonal, lowest index on ties) on its own from the same d array, forms its
// rows of column k, and the grid meets at a barrier.  d_a / d_b alternate between steps so no block reads what another
// writes within a step; the stop decision is taken from data every block sees identically (no flag written and read
// in the same step).  bar: two ints (arrival count, generation), zeroed before the launch.
__device__ __forceinline__ void chol_grid_barrier(unsigned *bar, unsigned nblocks)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        volatile unsigned *gen = bar + 1;
        const unsigned g = *gen;
        __threadfence();
        if (atomicAdd(bar, 1u) == nblocks - 1) {
            *bar = 0;
            __threadfence();
            atomicAdd((unsigned *)bar + 1, 1u);
        } else {
            while (*gen == g) { }
        }
        __threadfence();
    }
    __syncthreads();
}

__global__ void __launch_bounds__(128) chol_all_kernel(const double *__restrict__ Pp, int N, int Np, double *__restrict__ LT,
                                                       double *__restrict__ dbuf, int *dyn, const double *__restrict__ dscal,
                                                       unsigned *bar)
{
    __shared__ double sv[4];
    __shared__ int si[4];
    const double dmax = dscal[0];
    int k = 0;
    for (; k < N; ++k) {
        const double *d_in = dbuf + (size_t)(k & 1) * Np;
        double *d_out = dbuf + (size_t)((k + 1) & 1) * Np;
        double best = -1.0;
        int bi = 0x7fffffff;
        for (int i = threadIdx.x; i < N; i += 128) {
            const double v = __ldcg(d_in + i);               // written by other blocks in the previous step: read through L2
            if (v > best) { best = v; bi = i; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
        }
        if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = best; si[threadIdx.x >> 5] = bi; }
        __syncthreads();
        best = sv[0]; bi = si[0];
#pragma unroll
        for (int w = 1; w < 4; ++w)
            if (sv[w] > best || (sv[w] == best && si[w] < bi)) { best = sv[w]; bi = si[w]; }
        __syncthreads();
        if (!(best > 1e-13 * dmax) || !(best > 0.0)) break;  // same decision in every block
        const double root = sqrt(best);
        for (int i = blockIdx.x * 128 + threadIdx.x; i < N; i += gridDim.x * 128) {
            double s0 = Pp[(size_t)bi * Np + i], s1 = 0.0, s2 = 0.0, s3 = 0.0;
            int j = 0;
            for (; j + 4 <= k; j += 4) {
                s0 = fma(-LT[(size_t)j * Np + i], __ldcg(LT + (size_t)j * Np + bi), s0);
                s1 = fma(-LT[(size_t)(j + 1) * Np + i], __ldcg(LT + (size_t)(j + 1) * Np + bi), s1);
                s2 = fma(-LT[(size_t)(j + 2) * Np + i], __ldcg(LT + (size_t)(j + 2) * Np + bi), s2);
                s3 = fma(-LT[(size_t)(j + 3) * Np + i], __ldcg(LT + (size_t)(j + 3) * Np + bi), s3);
            }
            for (; j < k; ++j) s0 = fma(-LT[(size_t)j * Np + i], __ldcg(LT + (size_t)j * Np + bi), s0);
            double v = ((s0 + s1) + (s2 + s3)) / root;
            if (i == bi) v = root;
            LT[(size_t)k * Np + i] = v;                      // row k, element i: only this thread ever writes or reads (own i)
            d_out[i] = (i == bi) ? 0.0 : __ldcg(d_in + i) - v * v;
        }
        chol_grid_barrier(bar, gridDim.x);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) { dyn[0] = k; dyn[2] = 1; }
}

// max |P' - L L^T| over the lower-triangular tiles (R holds L L^T there)
__global__ void chol_residual_kernel(const double *__restrict__ Pp, const double *__restrict__ R, int N, int Np, int ldR,
                                     unsigned long long *resbits)
{
    const int n = blockIdx.x * blockDim.x + threadIdx.x, m = blockIdx.y;
    double v = 0.0;
    if (n < N && (n / BN) <= (m / BM)) v = fabs(Pp[(size_t)m * Np + n] - R[(size_t)m * ldR + n]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0 && v > 0.0) atomicMax(resbits, (unsigned long long)__double_as_longlong(v));
}

// not positive semidefinite (or badly conditioned): L := P', r := N, stage-2 B operand := A'
__global__ void chol_fallback_kernel(const double *__restrict__ Pp, int N, int Np, double *__restrict__ LT, int *dyn,
                                     const double *__restrict__ dscal)
{
    const double res = __longlong_as_double((long long)((const unsigned long long *)dscal)[1]);
    if (res <= 1e-12 * fmax(dscal[0], 1e-300)) return;
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < (size_t)Np * Np) LT[idx] = Pp[idx];
    if (idx == 0) { dyn[0] = N; dyn[1] = 1; }
}

// Occupied-orbital entry point: the caller hands C (N x nocc, row-major) with P = C C^T.
//   P[m][n] = sum_i C[m][i] C[n][i]                                        (eq 72 L547 with the occupation folded into C)
//   LT[i][m] = f_m C[m][i], rank = nocc: the factor P' = L L^T of the K^LR contraction without a decomposition
__global__ void density_from_orbitals_kernel(const double *__restrict__ C, int N, int nocc, double *__restrict__ P)
{
    const int n = blockIdx.x * blockDim.x + threadIdx.x, m = blockIdx.y;
    if (n >= N) return;
    const double *cm = C + (size_t)m * nocc, *cn = C + (size_t)n * nocc;
    double a0 = 0.0, a1 = 0.0;
    int i = 0;
    for (; i + 2 <= nocc; i += 2) { a0 = fma(cm[i], cn[i], a0); a1 = fma(cm[i + 1], cn[i + 1], a1); }
    if (i < nocc) a0 = fma(cm[i], cn[i], a0);
    P[(size_t)m * N + n] = a0 + a1;
}
__global__ void factor_from_orbitals_kernel(const double *__restrict__ C, int N, int nocc, int Np, const double *__restrict__ f,
                                            double *__restrict__ LT, int *dyn)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
    if (m < N) LT[(size_t)i * Np + m] = f[m] * C[(size_t)m * nocc + i];
    if (m == 0 && i == 0) { dyn[0] = nocc; dyn[1] = 0; dyn[2] = 1; }
}
void launch_density_from_orbitals(const double *C, int N, int nocc, double *P, cudaStream_t st)
{
    dim3 grid((N + 127) / 128, N);
    density_from_orbitals_kernel<<<grid, 128, 0, st>>>(C, N, nocc, P);
}
void launch_factor_from_orbitals(const double *C, int N, int nocc, int Np, int Npt, const double *fcomp, double *LT, int *dyn,
                                 cudaStream_t st)
{
    cudaMemsetAsync(LT, 0, (size_t)Npt * Np * sizeof(double), st);
    dim3 grid((N + 127) / 128, nocc);
    factor_from_orbitals_kernel<<<grid, 128, 0, st>>>(C, N, nocc, Np, fcomp, LT, dyn);
}

void launch_factor_density(const double *Pp, int N, int Np, int Npt, double *LT, double *dbuf, int *dyn, double *dscal,
                           double *scratch, cudaStream_t st)
{
    cudaMemsetAsync(LT, 0, (size_t)Npt * Np * sizeof(double), st);
    chol_init_kernel<<<1, 1024, 0, st>>>(Pp, N, Np, dbuf, dyn, dscal);
    // one cooperative launch for all steps (at most one block per 128 rows, capped by what is co-resident)
    {
        int dev = 0, nsm = 1, per_sm = 1;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, chol_all_kernel, 128, 0);
        int nblk = std::min((N + 127) / 128, nsm * std::max(per_sm, 1));
        unsigned *bar = reinterpret_cast<unsigned *>(dyn + 4);
        cudaMemsetAsync(bar, 0, 2 * sizeof(unsigned), st);
        void *args[] = {(void *)&Pp, (void *)&N, (void *)&Np, (void *)&LT, (void *)&dbuf, (void *)&dyn, (void *)&dscal, (void *)&bar};
        cudaLaunchCooperativeKernel((const void *)chol_all_kernel, dim3(nblk), dim3(128), args, 0, st);
    }
    // residual: scratch = L L^T on the lower-triangular tiles
    GemmArgs g;
    // (128 x 128 tiles over Npt; the part of a tile past Np multiplies whatever follows in LT into rows / columns of the
    //  scratch that nothing reads)
    g.M = Npt; g.Nc = Npt; g.Kb = Np; g.nbatch = 1; g.alpha = 1.0; g.A = LT; g.lda = Np; g.strideA = 0; g.B = LT; g.ldb = Np;
    g.strideB = 0; g.beta = 0.0; g.C = scratch; g.ldc = Npt; g.strideC = 0; g.nsplit = 1; g.transA = true; g.dyn = dyn;
    g.use_dyn = 2; g.lower_only = 1;
    launch_dgemm(g, st);
    dim3 grid((N + 127) / 128, N);
    chol_residual_kernel<<<grid, 128, 0, st>>>(Pp, scratch, N, Np, Npt, (unsigned long long *)(dscal + 1));
    const size_t tot = (size_t)Np * Np;
    chol_fallback_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(Pp, N, Np, LT, dyn, dscal);
}
int factor_density_launches(int) { return 1 + 1 + 3; }

// ---------------------------------------------------------------- finalise (A10)
__global__ void finalize_j_kernel(const double *__restrict__ Jsr, const double *__restrict__ Jlr, int N,
                                  const double *__restrict__ f, double *__restrict__ J)
{
    const int n = blockIdx.x * blockDim.x + threadIdx.x, m = blockIdx.y;
    if (n >= N) return;
    double v = 0.0;
    if (Jsr) v += 0.5 * (Jsr[(size_t)m * N + n] + Jsr[(size_t)n * N + m]);
    if (Jlr) v += 0.5 * (Jlr[(size_t)m * N + n] + Jlr[(size_t)n * N + m]);
    J[(size_t)m * N + n] = f[m] * f[n] * v;
}
void launch_finalize_j(const double *Jsr, const double *Jlr, int N, const double *fcomp, double *J, cudaStream_t st)
{
    dim3 grid((N + 127) / 128, N);
    finalize_j_kernel<<<grid, 128, 0, st>>>(Jsr, Jlr, N, fcomp, J);
}

// K_sr holds the blocks (mu, nu) with l_mu > l_nu, or l_mu == l_nu and mu >= nu; the rest by K = K^T.
__global__ void finalize_k_kernel(const double *__restrict__ Ksr, ShellInfo sh, const double *__restrict__ Klr, int nsplit,
                                  size_t strideK, int Np, int N, const double *__restrict__ f,
                                  const int *__restrict__ shell_of_ao, double *__restrict__ K)
{
    const int n = blockIdx.x * blockDim.x + threadIdx.x, m = blockIdx.y;
    if (n >= N) return;
    double v = 0.0;
    if (Ksr) {
        const int sm = shell_of_ao[m], sn = shell_of_ao[n];
        const int lm = sh.l[sm], ln = sh.l[sn];
        if (sm == sn) v = 0.5 * (Ksr[(size_t)m * N + n] + Ksr[(size_t)n * N + m]);
        else if (lm > ln || (lm == ln && sm > sn)) v = Ksr[(size_t)m * N + n];
        else v = Ksr[(size_t)n * N + m];
    }
    if (Klr) {
        // only the tiles with (row tile >= column tile) were computed (K^LR is symmetric)
        const int tm = m / 128, tn = n / 128;
        double t = 0.0;
        for (int z = 0; z < nsplit; ++z) {
            const double lo = Klr[z * strideK + (size_t)m * Np + n], up = Klr[z * strideK + (size_t)n * Np + m];
            t += tm > tn ? lo : (tm < tn ? up : 0.5 * (lo + up));
        }
        v += t;
    }
    K[(size_t)m * N + n] = f[m] * f[n] * v;
}
void launch_finalize_k(const double *Ksr, const ShellInfo &sh, const double *Klr, int nsplit, size_t strideK, int Np,
                       int N, const double *fcomp, const int *shell_of_ao, double *K, cudaStream_t st)
{
    dim3 grid((N + 127) / 128, N);
    finalize_k_kernel<<<grid, 128, 0, st>>>(Ksr, sh, Klr, nsplit, strideK, Np, N, fcomp, shell_of_ao, K);
}

__global__ void extract_overlap_kernel(const double *__restrict__ Astack, size_t ld, int S, int N, const double *__restrict__ f,
                                       double *__restrict__ Sm)
{
    const int n = blockIdx.x * blockDim.x + threadIdx.x, m = blockIdx.y;
    if (n >= N) return;
    Sm[(size_t)m * N + n] = f[m] * f[n] * Astack[(size_t)m * ld + (size_t)n * S];
}
void launch_extract_overlap(const double *Astack, int Np, int S, int N, const double *fcomp, double *Sm, cudaStream_t st)
{
    dim3 grid((N + 127) / 128, N);
    extract_overlap_kernel<<<grid, 128, 0, st>>>(Astack, (size_t)Np * S, S, N, fcomp, Sm);
}

// ---------------------------------------------------------------- allocation-free overlap (pbc_jk_overlap_noalloc)
// The crystalline overlap S = rho_mn(G = 0) (eq 21) is formed by agen_kernel in a scratch stack A'[m][n][slot] and read out
// by extract_overlap_kernel.  This variant keeps that scratch (2 slots per element) in a file-scope device array, so the
// call allocates nothing.  Every GPU that loads the library holds the array (NOALLOC_MAX_NP^2 * 2 doubles = 4 MiB) until
// the process exits; all calls share it (calls that overlap on the GPU race) and it keeps the last call's contents, so
// every call clears the part it reads (elements of shell pairs without a primitive pair-image are never written by agen).
constexpr int NOALLOC_SLOTS = 2;                          // (Re, Im) of the one "G vector" of the overlap mode
static __device__ __align__(256) double g_noalloc_scratch[(size_t)NOALLOC_MAX_NP * NOALLOC_MAX_NP * NOALLOC_SLOTS];

// Set-up, once per device, with that device current: in host code `g_noalloc_scratch` is a host-side stand-in, not a device
// address -- the address the kernels need comes from cudaGetSymbolAddress.
cudaError_t noalloc_scratch_address(int device, double **ptr)
{
    static std::mutex mtx;
    static double *cache[64] = {};
    *ptr = nullptr;
    if (device < 0 || device >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mtx);
    if (!cache[device]) {
        void *a = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&a, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        cache[device] = static_cast<double *>(a);
    }
    *ptr = cache[device];
    return cudaSuccess;
}

// scratch: the device address from noalloc_scratch_address; S_out: N x N, device.  Enqueues a clear, the agen kernels and the
// read-out on `st`; no allocation, no synchronisation.
cudaError_t launch_overlap_noalloc(const LRParams &p, double *scratch, int N, double *S_out, cudaStream_t st)
{
    if (p.Np > NOALLOC_MAX_NP) return cudaErrorInvalidValue;
    const cudaError_t e = cudaMemsetAsync(scratch, 0, (size_t)p.Np * p.Np * NOALLOC_SLOTS * sizeof(double), st);
    if (e != cudaSuccess) return e;
    launch_agen(p, -1, 1, NOALLOC_SLOTS, 1.0, scratch, nullptr, nullptr, st);
    launch_extract_overlap(scratch, p.Np, NOALLOC_SLOTS, N, p.fcomp, S_out, st);
    return cudaGetLastError();
}

}  // namespace pbcjk
