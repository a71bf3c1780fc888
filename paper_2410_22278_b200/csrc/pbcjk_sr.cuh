// Real-space (erfc(w r)/r) quartet kernels: J-engine (eq 95-98) and K (eq 74 L558 with
// eq 56/69).  One kernel family per angular-momentum class, generated from templates.
//
// Mapping (differs from PAPER 3.2 L753, which gives one THREAD a bra pair and lets it loop over
// its own lattice sphere -> warp divergence, L882):
//   * one WARP owns one bra primitive pair-image; its data are warp-uniform.
//   * phase 1 (cheap, divergent): lanes stream over the ket primitive pair-images of a group
//     (sorted by bound, so the loop ends early) for every lattice image R1 in the bounding box of
//     eq 99-103, test the eq-67 bound per (ket, R1) and push survivors into a per-warp
//     shared-memory queue (ballot + popc compaction).
//   * phase 2 (expensive, convergent): whenever 32 survivors are queued, every lane evaluates one
//     primitive quartet-image: merged Boys values, Hermite R recursion, contraction.
//   * accumulators stay in registers; warp-shuffle + shared-memory reductions; every output
//     element has exactly one owner, so there are no global atomics on the data path.
#pragma once
#include "pbcjk_md.cuh"

namespace pbcjk {

struct SRParams {
    PairListK K;
    PairListU U;
    KetListJ KJ;
    Lattice lat;
    ShellInfo sh;
    const double *boys;
    const double *Pp;        // P with component factors folded in, row stride ldP
    int ldP;
    const double *Dt;        // Hermite densities of the J kets, Dt[s*dstride + j]   (eq 95)
    double *Jt;              // Hermite J of the U entries, Jt[t*U.n + u]            (eq 98, raw)
    double *Ksr;             // N x N, accumulated block by block
    const double *lnPmax;    // device scalar ln(max |P'|)
    double ln_tau;           // ln(d_schwarz)
    double rcut2;            // r_cut^2 (C-14) or +inf
    unsigned long long *counters;
};

constexpr int QCAP = 64;

__device__ __forceinline__ int pack_img(int n0, int n1, int n2)
{
    return ((n0 + 512) << 20) | ((n1 + 512) << 10) | (n2 + 512);
}
__device__ __forceinline__ void unpack_img(int t, const Lattice &lat, double &Tx, double &Ty, double &Tz)
{
    double n0 = (double)((t >> 20) - 512), n1 = (double)(((t >> 10) & 1023) - 512), n2 = (double)((t & 1023) - 512);
    Tx = fma(n0, lat.a[0], fma(n1, lat.a[3], n2 * lat.a[6]));
    Ty = fma(n0, lat.a[1], fma(n1, lat.a[4], n2 * lat.a[7]));
    Tz = fma(n0, lat.a[2], fma(n1, lat.a[5], n2 * lat.a[8]));
}

// Phase 1 for one ket group [k0,k1) (sorted by lb descending) against the warp's bra, over all
// lattice images within `rho` of the group centre (eq 99-103: bounding box, then sphere filter).
// thr = lb_bra + ln(Pmax) - ln(tau); a (ket, image) survives iff
//   thr + lb_ket - r^2/(1/p + 1/q + 1/w^2) > 0       (eq 67 with C_2e split per pair)
template <class Eval>
__device__ __forceinline__ void scan_group(const Lattice &lat, double Pix, double Piy, double Piz,
                                           double ipi, double thr, double gx, double gy, double gz,
                                           double ext, double iqmax, int k0, int k1,
                                           const double *__restrict__ kQx, const double *__restrict__ kQy,
                                           const double *__restrict__ kQz, const double *__restrict__ kiq,
                                           const double *__restrict__ klb, double rcut2, int2 *queue,
                                           int &qn, int lane, unsigned &ncand, unsigned &nq, Eval &&eval)
{
    if (k1 <= k0) return;
    const double lbmax = __ldg(klb + k0);
    const double budget = thr + lbmax;
    if (budget <= 0.0) return;
    const double isum_max = ipi + iqmax + lat.iomega2;
    double rr = sqrt(budget * isum_max);
    const double rho = rr + ext;
    const double cx = Pix - gx, cy = Piy - gy, cz = Piz - gz;   // offset of the sphere centre
    const double f0 = lat.binv[0] * cx + lat.binv[1] * cy + lat.binv[2] * cz;
    const double f1 = lat.binv[3] * cx + lat.binv[4] * cy + lat.binv[5] * cz;
    const double f2 = lat.binv[6] * cx + lat.binv[7] * cy + lat.binv[8] * cz;
    const int lo0 = (int)ceil(f0 - rho * lat.bnorm[0]), hi0 = (int)floor(f0 + rho * lat.bnorm[0]);
    const int lo1 = (int)ceil(f1 - rho * lat.bnorm[1]), hi1 = (int)floor(f1 + rho * lat.bnorm[1]);
    const int lo2 = (int)ceil(f2 - rho * lat.bnorm[2]), hi2 = (int)floor(f2 + rho * lat.bnorm[2]);
    const unsigned ltmask = (1u << lane) - 1u;
    const int d1 = hi1 - lo1 + 1, d2 = hi2 - lo2 + 1, d12 = d1 * d2;
    const int nimg = (hi0 >= lo0 && d1 > 0 && d2 > 0) ? (hi0 - lo0 + 1) * d12 : 0;
    const double inv_isum_max = 1.0 / isum_max, rho2 = rho * rho;
    for (int base = 0; base < nimg; base += 32) {
        // 32 images of the box at a time, one per lane: sphere filter and the bound a ket needs there
        const int im = base + lane;
        bool ok = false;
        double need_l = 0.0;
        int timg_l = 0;
        if (im < nimg) {
            const int n0 = lo0 + im / d12, r = im % d12;
            const int n1 = lo1 + r / d2, n2 = lo2 + r % d2;
            const double Tx = n0 * lat.a[0] + n1 * lat.a[3] + n2 * lat.a[6];
            const double Ty = n0 * lat.a[1] + n1 * lat.a[4] + n2 * lat.a[7];
            const double Tz = n0 * lat.a[2] + n1 * lat.a[5] + n2 * lat.a[8];
            const double ex = Tx - cx, ey = Ty - cy, ez = Tz - cz;
            const double dist2 = ex * ex + ey * ey + ez * ez;
            ok = dist2 <= rho2;
            double dlb = sqrt(dist2) - ext;                     // lower bound of |Q + T - P|
            dlb = dlb > 0.0 ? dlb : 0.0;
            need_l = dlb * dlb * inv_isum_max - thr;            // ket survives only if lb_ket > need
            timg_l = pack_img(n0, n1, n2);
        }
        unsigned imask = __ballot_sync(0xffffffffu, ok);
        while (imask) {
            const int src = __ffs(imask) - 1;
            imask &= imask - 1;
            const double need = __shfl_sync(0xffffffffu, need_l, src);
            const int timg = __shfl_sync(0xffffffffu, timg_l, src);
            double Tx, Ty, Tz;
            unpack_img(timg, lat, Tx, Ty, Tz);
            const double ox = Tx - Pix, oy = Ty - Piy, oz = Tz - Piz;
            for (int j0 = k0; j0 < k1; j0 += 32) {
                if (__ldg(klb + j0) <= need) break;             // sorted: nothing further survives
                const int j = j0 + lane;
                bool pass = false;
                if (j < k1) {
                    const double dx = __ldg(kQx + j) + ox, dy = __ldg(kQy + j) + oy, dz = __ldg(kQz + j) + oz;
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    const double isum = ipi + __ldg(kiq + j) + lat.iomega2;
                    pass = (thr + __ldg(klb + j)) * isum > r2 && r2 <= rcut2;
                    ++ncand;
                }
                const unsigned m = __ballot_sync(0xffffffffu, pass);
                if (pass) queue[qn + __popc(m & ltmask)] = make_int2(j, timg);
                qn += __popc(m);
                __syncwarp();
                if (qn >= 32) {
                    qn -= 32;
                    const int2 e = queue[qn + lane];
                    __syncwarp();
                    eval(e.x, e.y);
                    ++nq;
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// J-engine: bra Hermite order LB (= la+lb), ket Hermite order LK.  One warp per bra U entry.
//   Jt[t] += sum_kets pref * sum_s R_{t+s}(Q - P + R1) D~_s        (eq 98 second term, reading C-4;
//   the (-1)^{|t|} and E^{ab}_t are applied by the back-transform kernel, eq 97)
// ------------------------------------------------------------------------------------------
template <int LB, int LK>
__global__ void __launch_bounds__(128) sr_j_kernel(SRParams p, const int *__restrict__ bra_idx, int nbra)
{
    constexpr int L = LB + LK;
    constexpr int NT = nherm(LB), NS = nherm(LK);
    __shared__ int2 s_queue[4][QCAP];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int ib = blockIdx.x * 4 + w;
    if (ib >= nbra) return;
    const int u = __ldg(bra_idx + ib);
    const double Pix = p.U.Px[u], Piy = p.U.Py[u], Piz = p.U.Pz[u];
    const double pi_ = p.U.p[u], coefi = p.U.coef[u];
    const double ipi = p.U.ip[u];
    const double thr = p.U.lb[u] + *p.lnPmax - p.ln_tau;
    double Jt[NT];
#pragma unroll
    for (int t = 0; t < NT; ++t) Jt[t] = 0.0;
    int qn = 0;
    unsigned ncand = 0, nq = 0;
    int2 *queue = s_queue[w];
    const Lattice &lat = p.lat;
    const double *__restrict__ tab = p.boys;

    auto eval = [&](int j, int timg) {
        double Tx, Ty, Tz;
        unpack_img(timg, lat, Tx, Ty, Tz);
        const double X = __ldg(p.KJ.Qx + j) + Tx - Pix, Y = __ldg(p.KJ.Qy + j) + Ty - Piy,
                     Z = __ldg(p.KJ.Qz + j) + Tz - Piz;
        const double q = __ldg(p.KJ.q + j);
        const double r2 = X * X + Y * Y + Z * Z;
        const double s = rsqrt(pi_ + q);
        const double alpha = pi_ * q * s * s;
        const double th = lat.omega * rsqrt(alpha + lat.omega2);
        const double alpha_w = alpha * th * th;
        const double pref = coefi * __ldg(p.KJ.coef + j) * s;
        double Rm[L + 1];
        boys_merged<L>(tab, r2, alpha, alpha_w, th, pref, Rm);
        double R[nherm(L)];
        hermite_R<L>(R, Rm, X, Y, Z);
        double D[NS];
#pragma unroll
        for (int sI = 0; sI < NS; ++sI) D[sI] = __ldg(p.Dt + (size_t)sI * p.KJ.dstride + j);
#pragma unroll
        for (int tx = 0; tx <= LB; ++tx)
#pragma unroll
            for (int ty = 0; ty <= LB - tx; ++ty)
#pragma unroll
                for (int tz = 0; tz <= LB - tx - ty; ++tz) {
                    double acc = Jt[hidx(tx, ty, tz)];
#pragma unroll
                    for (int sx = 0; sx <= LK; ++sx)
#pragma unroll
                        for (int sy = 0; sy <= LK - sx; ++sy)
#pragma unroll
                            for (int sz = 0; sz <= LK - sx - sy; ++sz)
                                acc = fma(R[hidx(tx + sx, ty + sy, tz + sz)], D[hidx(sx, sy, sz)], acc);
                    Jt[hidx(tx, ty, tz)] = acc;
                }
    };

    for (int g = 0; g < p.KJ.ngroup; ++g) {
        const int gi = g * 5 + LK;
        const int k0 = __ldg(p.KJ.off + gi), k1 = __ldg(p.KJ.off + gi + 1);
        if (k1 <= k0) continue;
        scan_group(lat, Pix, Piy, Piz, ipi, thr, __ldg(p.KJ.gx + g), __ldg(p.KJ.gy + g), __ldg(p.KJ.gz + g),
                   __ldg(p.KJ.ext + gi), __ldg(p.KJ.iqmax + gi), k0, k1, p.KJ.Qx, p.KJ.Qy, p.KJ.Qz, p.KJ.iq,
                   p.KJ.lb, p.rcut2, queue, qn, lane, ncand, nq, eval);
    }
    if (qn > 0) {                                   // flush: partial warp
        if (lane < qn) {
            const int2 e = queue[lane];
            eval(e.x, e.y);
        }
    }
    // warp reduction (fixed order => deterministic)
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        double v = Jt[t];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        Jt[t] = v;
    }
    if (lane == 0) {
#pragma unroll
        for (int t = 0; t < NT; ++t) p.Jt[(size_t)t * p.U.n + u] += Jt[t];
    }
    // statistics (once per warp, not on the data path)
    unsigned long long c = ncand, e32 = (unsigned long long)nq * 32ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) {
        atomicAdd(p.counters + CNT_CAND_J + LB * 5 + LK, c);
        atomicAdd(p.counters + CNT_Q_J + LB * 5 + LK, e32 + (unsigned long long)qn);
    }
}

// number of non-zero separable E^{ab}_t over all component pairs of a shell pair (rows of PairListK::etab);
// the K kernels themselves are in pbcjk_srk.cuh
template <int LA, int LB>
__host__ __device__ constexpr int bra_terms()
{
    int n = 0;
    for (int a = 0; a < ncart(LA); ++a)
        for (int b = 0; b < ncart(LB); ++b)
            n += (cart_x(LA, a) + cart_x(LB, b) + 1) * (cart_y(LA, a) + cart_y(LB, b) + 1) *
                 (cart_z(LA, a) + cart_z(LB, b) + 1);
    return n;
}

// launchers (defined in the instantiation units)
void launch_sr_j(int LB, int LK, const SRParams &p, const int *bra_idx, int nbra, cudaStream_t st);
void launch_sr_k(int la, int lb, int lc, int ld, const SRParams &p, const int2 *blocks, int nblocks, cudaStream_t st);

}  // namespace pbcjk
