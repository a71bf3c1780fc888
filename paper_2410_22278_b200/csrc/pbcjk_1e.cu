// One-electron Ewald terms at the Gamma point: kinetic matrix (PAPER SI eq S1), the
// interaction V of every pair density with point charges (eq 52) and, on the host, the Ewald energy of the point
// charges (eq 91).  They reuse the machinery of the J path: the unordered primitive pair-image list U, the
// rho_mn(G) stack of the reciprocal-space passes (V^LR is J^LR with rho(G) replaced by the structure factor of the
// charges) and the Hermite back-transform of the J-engine (a point charge is a ket of Hermite order 0 with q -> inf).
//
// Sign convention (the paper's): V_mn = sum_C q_C (mn | delta_C) under the zero-mean periodic Coulomb kernel; the
// electron-nucleus attraction matrix is -V with q_C = Z_C.
#include "pbcjk_1e.cuh"
#include "pbcjk_sr.cuh"

namespace pbcjk {

// ---------------------------------------------------------------- kinetic (SI eq S1)
// One direction of E^{ij}_0 for i <= LMAX, j <= LMAX + 2 (eq 17-18 with E^{00}_0 = 1): -1/2 d^2/dx^2 of the second
// function needs j - 2, j, j + 2.
struct E1Dkin {
    double e[LMAX + 1][LMAX + 3][2 * LMAX + 3];
    __device__ void build(int la, int lb, double PA, double PB, double o2p)
    {
        for (int i = 0; i <= LMAX; ++i)
            for (int j = 0; j < LMAX + 3; ++j)
                for (int t = 0; t < 2 * LMAX + 3; ++t) e[i][j][t] = 0.0;
        e[0][0][0] = 1.0;
        for (int i = 0; i < la; ++i)
            for (int t = 0; t <= i + 1; ++t) {
                double v = 0.0;
                if (t <= i) v = PA * e[i][0][t];
                if (t > 0) v += o2p * e[i][0][t - 1];
                if (t + 1 <= i) v += (t + 1) * e[i][0][t + 1];
                e[i + 1][0][t] = v;
            }
        for (int i = 0; i <= la; ++i)
            for (int j = 0; j < lb; ++j)
                for (int t = 0; t <= i + j + 1; ++t) {
                    double v = 0.0;
                    if (t <= i + j) v = PB * e[i][j][t];
                    if (t > 0) v += o2p * e[i][j][t - 1];
                    if (t + 1 <= i + j) v += (t + 1) * e[i][j][t + 1];
                    e[i][j + 1][t] = v;
                }
    }
};

// T_ab = sum_{R2,prims} C_a C_b (pi/p)^{3/2} [k_x E_y E_z + E_x k_y E_z + E_x E_y k_z],
//   k = -j(j-1)/2 E^{i,j-2}_0 + (2j+1) b E^{i,j}_0 - 2 b^2 E^{i,j+2}_0     (reading C-27: the same bracket per direction)
// one warp per shell pair of U (A >= B), mirrored; component factors f folded in on output.
__global__ void kinetic_kernel(PairListU U, ShellInfo sh, const double *__restrict__ f, double *__restrict__ T, int N)
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
        const double p = U.p[u], o2p = 0.5 * U.ip[u], b = U.bexp[u];
        // coef holds sqrt2 pi^{5/4}/p; the overlap-type integrals need (pi/p)^{3/2}
        const double c = U.coef[u] * 0.94139626377671481 * rsqrt(p);
        E1Dkin e[3];
        e[0].build(la, lb + 2, U.PAx[u], U.PBx[u], o2p);
        e[1].build(la, lb + 2, U.PAy[u], U.PBy[u], o2p);
        e[2].build(la, lb + 2, U.PAz[u], U.PBz[u], o2p);
        for (int ka = 0; ka < na; ++ka)
            for (int kb = 0; kb < nb; ++kb) {
                int ia[3], jb[3];
                cart_powers(la, ka, ia[0], ia[1], ia[2]);
                cart_powers(lb, kb, jb[0], jb[1], jb[2]);
                double e0[3], kk[3];
                for (int d = 0; d < 3; ++d) {
                    const int i = ia[d], j = jb[d];
                    e0[d] = e[d].e[i][j][0];
                    double k = (2 * j + 1) * b * e0[d] - 2.0 * b * b * e[d].e[i][j + 2][0];
                    if (j >= 2) k -= 0.5 * j * (j - 1) * e[d].e[i][j - 2][0];
                    kk[d] = k;
                }
                acc[ka * nb + kb] += c * (kk[0] * e0[1] * e0[2] + e0[0] * kk[1] * e0[2] + e0[0] * e0[1] * kk[2]);
            }
    }
    for (int i = 0; i < na * nb; ++i) {
        double v = acc[i];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) {
            const int a = i / nb, b = i % nb;
            const int m = sh.ao[A] + a, n = sh.ao[B] + b;
            v *= f[m] * f[n];
            T[(size_t)m * N + n] = v;
            if (A != B) T[(size_t)n * N + m] = v;
        }
    }
}
void launch_kinetic(const PairListU &U, const ShellInfo &sh, const double *fcomp, double *T, int N, cudaStream_t st)
{
    cudaMemsetAsync(T, 0, (size_t)N * N * sizeof(double), st);
    if (U.nsp <= 0) return;
    kinetic_kernel<<<(U.nsp + 3) / 4, 128, 0, st>>>(U, sh, fcomp, T, N);
}

// ---------------------------------------------------------------- V, short range (eq 52 second term)
// One warp per U entry (bra of Hermite order LB); lanes over (charge, lattice image) pairs; for a pair inside the reach
//   Vt[t] += q_C c_ab sqrt2 pi^{-1/4} [ R^0_t(p, L) - theta R^0_t(a_w, L) ],  L = C + R_C - P,
//   theta = w/sqrt(p + w^2), a_w = p w^2/(p + w^2)          (U.coef * sqrt2 pi^{-1/4} = C_a C_b e^{-mu R^2} 2 pi/p)
// The (-1)^{|t|} E^{ab}_t contraction is the J-engine's back-transform (eq 96-97).  Reach (eq 42-43): a pair is
// evaluated iff bound_ab |q_C| e^{-a_w |L|^2} exceeds delta (the bound of the pair list is an upper bound of the
// eq-42 prefactor up to a constant of order one, so delta is taken two decades below the pair threshold).
template <int LB>
__global__ void __launch_bounds__(128) sr_v_kernel(PairListU U, Lattice lat, BoysTab boys, const int *__restrict__ bra_idx, int nbra,
                                                   const double *__restrict__ cxyz, const double *__restrict__ q, int natom,
                                                   double qabs_max, double ln_delta, double g0x, double g0y, double g0z, double rc,
                                                   double *__restrict__ Vt)
{
    constexpr int NT = nherm(LB);
    const int lane = threadIdx.x & 31;
    const int ib = blockIdx.x * 4 + (threadIdx.x >> 5);
    if (ib >= nbra) return;
    const int u = bra_idx[ib];
    const double Px = U.Px[u], Py = U.Py[u], Pz = U.Pz[u], p = U.p[u];
    const double coef = U.coef[u] * 1.0622519320271968;           // sqrt2 pi^{-1/4}
    const double th = lat.omega * rsqrt(p + lat.omega2);
    const double aw = p * th * th;
    const double budget = U.lb[u] + log(fmax(qabs_max, 1e-300)) - ln_delta;   // ln(bound |q|max / delta)
    double acc[NT];
#pragma unroll
    for (int t = 0; t < NT; ++t) acc[t] = 0.0;
    if (budget > 0.0) {
        const double reach = sqrt(budget / aw);
        ImageBox box;
        box.set(lat, Px - g0x, Py - g0y, Pz - g0z, reach + rc);    // images T with |g0 + T - P| within reach + rc
        const long long nitem = (long long)box.n * natom;
        for (long long e = lane; e < nitem; e += 32) {
            const int c = (int)(e % natom), im = (int)(e / natom);
            const double qc = q[c];
            if (qc == 0.0) continue;
            int n0, n1, n2;
            box.decode(im, n0, n1, n2);
            const double X = cxyz[3 * c] + (n0 * lat.a[0] + n1 * lat.a[3] + n2 * lat.a[6]) - Px;
            const double Y = cxyz[3 * c + 1] + (n0 * lat.a[1] + n1 * lat.a[4] + n2 * lat.a[7]) - Py;
            const double Z = cxyz[3 * c + 2] + (n0 * lat.a[2] + n1 * lat.a[5] + n2 * lat.a[8]) - Pz;
            const double r2 = X * X + Y * Y + Z * Z;
            if (aw * r2 >= budget) continue;
            double Rm[LB + 1];
            boys_merged<LB, double>(boys, r2, p, aw, th, qc * coef, Rm);
            double R[NT];
            hermite_R<LB>(R, Rm, X, Y, Z);
#pragma unroll
            for (int t = 0; t < NT; ++t) acc[t] += R[t];
        }
    }
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        double v = acc[t];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) Vt[(size_t)t * U.n + u] = v;
    }
}
void launch_sr_v(const PairListU &U, const Lattice &lat, const BoysTab &boys, const int *const jbra[5], const int njbra[5],
                 const double *cxyz, const double *q, int natom, double qabs_max, double ln_delta, const double g0[3], double rc,
                 double *Vt, cudaStream_t st)
{
#define SRV(LB)                                                                                                            \
    if (njbra[LB] > 0)                                                                                                     \
        sr_v_kernel<LB><<<(njbra[LB] + 3) / 4, 128, 0, st>>>(U, lat, boys, jbra[LB], njbra[LB], cxyz, q, natom, qabs_max,   \
                                                             ln_delta, g0[0], g0[1], g0[2], rc, Vt);
    SRV(0) SRV(1) SRV(2) SRV(3) SRV(4)
#undef SRV
}

// ---------------------------------------------------------------- V, long range (eq 52 first term)
// rho'[2g] + i rho'[2g+1] = sqrt(w_g) sum_C q_C e^{-iG.C} for the G of one batch (slots past the batch: 0);
// g0 < 0: the G = 0 slot (SELF), rho'[0] = w0 * sum_C q_C.
__global__ void rho_nuc_kernel(const double *__restrict__ Gx, const double *__restrict__ Gy, const double *__restrict__ Gz,
                               const double *__restrict__ Gw, int g0, int nb, int S, double w0, const double *__restrict__ cxyz,
                               const double *__restrict__ q, int natom, double *__restrict__ rho)
{
    const int gl = blockIdx.x * blockDim.x + threadIdx.x;
    if (2 * gl >= S) return;
    double re = 0.0, im = 0.0;
    if (gl < nb) {
        if (g0 < 0) {
            for (int c = 0; c < natom; ++c) re += q[c];
            re *= w0;
        } else {
            const double gx = Gx[g0 + gl], gy = Gy[g0 + gl], gz = Gz[g0 + gl], sw = Gw[g0 + gl];
            for (int c = 0; c < natom; ++c) {
                double sn, cs;
                sincos(-(gx * cxyz[3 * c] + gy * cxyz[3 * c + 1] + gz * cxyz[3 * c + 2]), &sn, &cs);
                re += q[c] * cs;
                im += q[c] * sn;
            }
            re *= sw; im *= sw;
        }
    }
    rho[2 * gl] = re;
    rho[2 * gl + 1] = im;
}
void launch_rho_nuc(const LRParams &p, int g0, int nb, int S, double w0, const double *cxyz, const double *q, int natom, double *rho,
                    cudaStream_t st)
{
    rho_nuc_kernel<<<(S / 2 + 63) / 64, 64, 0, st>>>(p.Gx, p.Gy, p.Gz, p.Gw, g0, nb, S, w0, cxyz, q, natom, rho);
}

}  // namespace pbcjk
