// Real-space K kernels (eq 74 L558 with eq 56/69): class (LA LB | LC LD), bra = (mu: LA, lambda: LB),
// ket = (nu: LD, sigma: LC).  One CTA owns the output block (mu, nu); warps take the bra primitive
// pair-images of mu round-robin; lanes the ket primitive pair-images of nu and the lattice image R1.
//   K[mu_a, nu_d] += sum P'[lambda_b, sigma_c] (mu_a lambda_b | sigma_c nu_d)
//
// Phase 1 (scan) is the same screen as the J-engine's scan_group (eq 67, bounding box eq 99-103),
// written as a resumable iterator so that the quartet evaluator -- straight-line code generated per
// class by gen_sr_k.py -- is expanded at exactly one call site.  The Hermite integrals of classes with
// L > 4 live in shared memory (one column per thread); the E products of both pairs come from the
// tables built at create (PairListK::etab), so no E recursion runs per quartet.
#pragma once
#include "pbcjk_sr.cuh"

namespace pbcjk {

template <int LA, int LB, int LC, int LD> struct KEval;      // specialisations: build/gen/k_eval_*.cuh

__host__ __device__ constexpr int k_nthreads(int L) { return L >= 7 ? 64 : 128; }

template <int LA, int LB, int LC, int LD>
constexpr size_t k_smem_bytes()
{
    constexpr int L = LA + LB + LC + LD, NT = k_nthreads(L), NW = NT / 32;
    size_t d = (L > 4 ? (size_t)nherm(L) * NT : 0) + (size_t)NW * bra_terms<LA, LB>() + (size_t)NW * ncart(LA) * ncart(LD);
    return d * sizeof(double) + (size_t)NW * QCAP * sizeof(int2);
}

template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(k_nthreads(LA + LB + LC + LD))
sr_k_kernel(SRParams p, const int2 *__restrict__ blocks, int nblocks)
{
    constexpr int L = LA + LB + LC + LD;
    constexpr int NT = k_nthreads(L), NW = NT / 32;
    constexpr int NA = ncart(LA), ND = ncart(LD);
    constexpr int NTERM = bra_terms<LA, LB>();
    constexpr bool RSMEM = L > 4;
    using Ev = KEval<LA, LB, LC, LD>;
    static_assert(Ev::NBRA == NTERM, "generator and kernel disagree on the bra table");
    extern __shared__ __align__(16) double smem[];
    double *Rs = smem + threadIdx.x;                                  // [nherm(L)][NT] when RSMEM
    double *sE = smem + (RSMEM ? nherm(L) * NT : 0);                  // [NW][NTERM]
    double *s_red = sE + NW * NTERM;                                  // [NW][NA*ND]
    int2 *queue = reinterpret_cast<int2 *>(s_red + NW * NA * ND);     // [NW][QCAP]
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    sE += w * NTERM;
    queue += w * QCAP;
    const int2 blk = blocks[blockIdx.x];
    const int mu = blk.x, nu = blk.y;
    const int b0 = __ldg(p.K.off + mu * 3 + LB), b1 = __ldg(p.K.off + mu * 3 + LB + 1);
    const int k0 = __ldg(p.K.off + nu * 3 + LC), k1 = __ldg(p.K.off + nu * 3 + LC + 1);
    if (b1 <= b0 || k1 <= k0) return;
    const Lattice &lat = p.lat;
    const double *__restrict__ tab = p.boys;
    const int N = p.sh.nbf;
    const double gx = __ldg(p.sh.cx + nu), gy = __ldg(p.sh.cy + nu), gz = __ldg(p.sh.cz + nu);
    const double kext = __ldg(p.K.ext + nu * 3 + LC), kiqmax = __ldg(p.K.ipmax + nu * 3 + LC);
    const double lbmax_ket = __ldg(p.K.lb + k0);
    const double thr0 = *p.lnPmax - p.ln_tau;
    const double *__restrict__ kQx = p.K.Px, *__restrict__ kQy = p.K.Py, *__restrict__ kQz = p.K.Pz;
    const double *__restrict__ kiq = p.K.ip, *__restrict__ klb = p.K.lb;
    const unsigned ltmask = (1u << lane) - 1u;

    double Kacc[NA * ND];
#pragma unroll
    for (int i = 0; i < NA * ND; ++i) Kacc[i] = 0.0;
    unsigned ncand = 0;
    unsigned long long nquart = 0;

    for (int i = b0 + w; i < b1; i += NW) {
        const double thr = __ldg(p.K.lb + i) + thr0;
        const double budget = thr + lbmax_ket;
        if (budget <= 0.0) break;                           // bras sorted: the rest is weaker
        const double Pix = __ldg(p.K.Px + i), Piy = __ldg(p.K.Py + i), Piz = __ldg(p.K.Pz + i);
        const double pi_ = __ldg(p.K.p + i), coefi = __ldg(p.K.coef + i);
        const double ipi = __ldg(p.K.ip + i);
        const double *__restrict__ Pb = p.Pp + (size_t)__ldg(p.K.aoB + i) * p.ldP;
        // bra table E^{mu lambda}_T -> shared memory (warp-uniform operand of the evaluator)
        {
            const double *__restrict__ src = p.K.etab + __ldg(p.K.eoff + i);
            __syncwarp();
            for (int n = lane; n < NTERM; n += 32) sE[n] = __ldg(src + n);
            __syncwarp();
        }
        // bounding box of the lattice images within reach of the ket group (eq 99-103)
        const double isum_max = ipi + kiqmax + lat.iomega2;
        const double rho = sqrt(budget * isum_max) + kext;
        const double cx = Pix - gx, cy = Piy - gy, cz = Piz - gz;
        const double f0 = lat.binv[0] * cx + lat.binv[1] * cy + lat.binv[2] * cz;
        const double f1 = lat.binv[3] * cx + lat.binv[4] * cy + lat.binv[5] * cz;
        const double f2 = lat.binv[6] * cx + lat.binv[7] * cy + lat.binv[8] * cz;
        const int lo0 = (int)ceil(f0 - rho * lat.bnorm[0]), hi0 = (int)floor(f0 + rho * lat.bnorm[0]);
        const int lo1 = (int)ceil(f1 - rho * lat.bnorm[1]), hi1 = (int)floor(f1 + rho * lat.bnorm[1]);
        const int lo2 = (int)ceil(f2 - rho * lat.bnorm[2]), hi2 = (int)floor(f2 + rho * lat.bnorm[2]);
        const int d1 = hi1 - lo1 + 1, d2 = hi2 - lo2 + 1;
        const int nimg = (hi0 >= lo0 && d1 > 0 && d2 > 0) ? (hi0 - lo0 + 1) * d1 * d2 : 0;
        const double inv_isum_max = 1.0 / isum_max, rho2 = rho * rho;
        const int d12 = d1 * d2;
        int base = 0, j0 = k0, qn = 0, timg = 0, timg_l = 0;
        unsigned imask = 0;                                 // images of the current batch still to visit
        bool have = false;
        double need = 0.0, need_l = 0.0, ox = 0.0, oy = 0.0, oz = 0.0;

        for (;;) {
            // ---- phase 1: screen (ket, image) candidates until 32 survivors are queued ----
            while (qn < 32) {
                if (!have) {
                    if (imask == 0) {
                        if (base >= nimg) break;
                        // 32 images of the box at a time, one per lane: sphere filter and the bound each
                        // image needs from a ket (eq 67 with the closest approach of the ket group)
                        const int im = base + lane;
                        base += 32;
                        bool ok = false;
                        if (im < nimg) {
                            const int n0 = lo0 + im / d12, r = im % d12;
                            const int n1 = lo1 + r / d2, n2 = lo2 + r % d2;
                            const double Tx = n0 * lat.a[0] + n1 * lat.a[3] + n2 * lat.a[6];
                            const double Ty = n0 * lat.a[1] + n1 * lat.a[4] + n2 * lat.a[7];
                            const double Tz = n0 * lat.a[2] + n1 * lat.a[5] + n2 * lat.a[8];
                            const double ex = Tx - cx, ey = Ty - cy, ez = Tz - cz;
                            const double dist2 = ex * ex + ey * ey + ez * ez;
                            ok = dist2 <= rho2;
                            double dlb = sqrt(dist2) - kext;    // lower bound of |Q + T - P|
                            dlb = dlb > 0.0 ? dlb : 0.0;
                            need_l = dlb * dlb * inv_isum_max - thr;   // a ket survives only if lb_ket > need
                            timg_l = pack_img(n0, n1, n2);
                        }
                        imask = __ballot_sync(0xffffffffu, ok);
                        continue;
                    }
                    const int src = __ffs(imask) - 1;
                    imask &= imask - 1;
                    need = __shfl_sync(0xffffffffu, need_l, src);
                    timg = __shfl_sync(0xffffffffu, timg_l, src);
                    double Tx, Ty, Tz;
                    unpack_img(timg, lat, Tx, Ty, Tz);
                    ox = Tx - Pix; oy = Ty - Piy; oz = Tz - Piz;
                    j0 = k0;
                    have = true;
                }
                if (j0 >= k1 || __ldg(klb + j0) <= need) { have = false; continue; }   // sorted by lb
                const int j = j0 + lane;
                bool pass = false;
                if (j < k1) {
                    const double dx = __ldg(kQx + j) + ox, dy = __ldg(kQy + j) + oy, dz = __ldg(kQz + j) + oz;
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    const double isum = ipi + __ldg(kiq + j) + lat.iomega2;
                    pass = (thr + __ldg(klb + j)) * isum > r2 && r2 <= p.rcut2;
                    ++ncand;
                }
                const unsigned m = __ballot_sync(0xffffffffu, pass);
                if (pass) queue[qn + __popc(m & ltmask)] = make_int2(j, timg);
                qn += __popc(m);
                j0 += 32;
                __syncwarp();
            }
            if (qn == 0) break;
            // ---- phase 2: one primitive quartet-image per lane ----
            const int take = qn < 32 ? qn : 32;
            qn -= take;
            if (lane < take) {
                const int2 e = queue[qn + lane];
                const int j = e.x;
                double Tx, Ty, Tz;
                unpack_img(e.y, lat, Tx, Ty, Tz);
                const double X = __ldg(kQx + j) + Tx - Pix, Y = __ldg(kQy + j) + Ty - Piy, Z = __ldg(kQz + j) + Tz - Piz;
                const double q = __ldg(p.K.p + j);
                const double r2 = X * X + Y * Y + Z * Z;
                const double s = rsqrt(pi_ + q);
                const double alpha = pi_ * q * s * s;
                const double th = lat.omega * rsqrt(alpha + lat.omega2);
                const double alpha_w = alpha * th * th;
                const double pref = coefi * __ldg(p.K.coef + j) * s;
                double Rm[L + 1];
                boys_merged<L>(tab, r2, alpha, alpha_w, th, pref, Rm);
                Ev::template run<NT>(sE, p.K.etab + __ldg(p.K.eoff + j), Pb + __ldg(p.K.aoB + j), p.ldP, Rm, X, Y, Z, Rs, Kacc);
            }
            nquart += take;
            __syncwarp();
        }
    }
    // warp shuffle reduction, then shared-memory reduction across the CTA's warps
#pragma unroll
    for (int i = 0; i < NA * ND; ++i) {
        double v = Kacc[i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) s_red[w * NA * ND + i] = v;
    }
    __syncthreads();
    if (threadIdx.x < NA * ND) {
        double v = 0.0;
#pragma unroll
        for (int ww = 0; ww < NW; ++ww) v += s_red[ww * NA * ND + threadIdx.x];
        const int a = threadIdx.x / ND, d = threadIdx.x % ND;
        double *dst = p.Ksr + (size_t)(__ldg(p.sh.ao + mu) + a) * N + __ldg(p.sh.ao + nu) + d;
        *dst += v;                                          // this CTA is the only owner of the block
    }
    unsigned long long c = ncand;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) {
        constexpr int cls = ((LA * 3 + LB) * 3 + LC) * 3 + LD;
        atomicAdd(p.counters + CNT_CAND_K + cls, c);
        atomicAdd(p.counters + CNT_Q_K + cls, nquart);
    }
}

template <int LA, int LB, int LC, int LD>
void launch_sr_k_class(const SRParams &p, const int2 *blocks, int nblocks, cudaStream_t st)
{
    constexpr size_t smem = k_smem_bytes<LA, LB, LC, LD>();
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(sr_k_kernel<LA, LB, LC, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        attr_set = true;
    }
    sr_k_kernel<LA, LB, LC, LD><<<nblocks, k_nthreads(LA + LB + LC + LD), smem, st>>>(p, blocks, nblocks);
}

}  // namespace pbcjk
