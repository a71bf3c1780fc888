// Real-space K kernels (eq 74 L558 with eq 56/69): class (LA LB | LC LD), bra = (mu: LA, lambda: LB),
// ket = (nu: LD, sigma: LC).  One CTA owns the output block (mu, nu); warps take the bra primitive
// pair-images of mu round-robin; lanes the ket primitive pair-images of nu and the lattice image R1.
//   K[mu_a, nu_d] += sum P'[lambda_b, sigma_c] (mu_a lambda_b | sigma_c nu_d)
//
// Phase 1 (scan) is the same screen as the J-engine's scan_group (eq 67, bounding box eq 99-103),
// written as a resumable iterator so that the quartet evaluator -- straight-line code generated per
// class by gen_sr_k.py -- is expanded at exactly one call site.  Survivors wait in a per-warp ring that
// spans several bras (each keeps its E row and centre in a shared-memory slot), so the evaluator runs
// with 32 active lanes except for the last call of a warp.  The Hermite integrals of classes with
// L > 4 live in shared memory (one column per thread); the E products of both pairs come from the
// tables built at create (PairListK::etab), so no E recursion runs per quartet.
#pragma once
#include "pbcjk_sr.cuh"

namespace pbcjk {

template <int LA, int LB, int LC, int LD> struct KEval;      // specialisations: build/gen/k_eval_*.cuh

// CTA size: 128 threads in every class.  The warps of a CTA enter the evaluator in lockstep at L >= 5 (see LOCKSTEP
// below), so four warps share the instruction fetches; the R column of a thread takes 8*nherm(L) bytes of shared
// memory (1320 B at L = 8: one CTA per SM).  Measured on water64 / si64: 64-thread CTAs at L >= 7 are 3 % slower,
// 256-thread CTAs at L = 5 are 4-6 % slower, lockstep at L = 3, 4 is 10 % slower.
__host__ __device__ constexpr int k_nthreads(int) { return 128; }

// bra slots per warp: a queued quartet refers to its bra by slot, so the queue carries survivors across bras
// and the evaluator runs with (nearly) all 32 lanes; the slot stride is odd so that lanes reading the E tables
// of different slots hit different banks.
__host__ __device__ constexpr int k_nslot(int nterm, int) { return nterm > 150 ? 4 : 8; }
__host__ __device__ constexpr int k_slot_stride(int nterm) { return (nterm + 6) | 1; }   // E row + 6 scalars, odd
constexpr int KQ = 64;                                       // ring capacity per warp (power of two)

template <int LA, int LB, int LC, int LD>
constexpr size_t k_smem_bytes()
{
    constexpr int L = LA + LB + LC + LD, NT = k_nthreads(L), NW = NT / 32;
    constexpr int NTERM = bra_terms<LA, LB>();
    size_t d = (L > 4 ? (size_t)nherm(L) * NT : 0) + (size_t)NW * k_nslot(NTERM, L) * k_slot_stride(NTERM) +
               (size_t)NW * ncart(LA) * ncart(LD);
    return d * sizeof(double) + (size_t)NW * KQ * (sizeof(int2) + sizeof(int));
}

// light classes: at most 128 registers (L <= 3: 4 CTAs, 16 warps per SM) or 168 (L = 4: 3 CTAs); the few spilled
// doubles (<= 300 B per thread) cost less than the lost occupancy
__host__ __device__ constexpr int k_minblocks(int L) { return L <= 3 ? 4 : (L == 4 ? 3 : 1); }

template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(k_nthreads(LA + LB + LC + LD), k_minblocks(LA + LB + LC + LD))
sr_k_kernel(SRParams p, const int2 *__restrict__ blocks, int nblocks)
{
    constexpr int L = LA + LB + LC + LD;
    constexpr int NT = k_nthreads(L), NW = NT / 32;
    constexpr int NA = ncart(LA), ND = ncart(LD);
    constexpr int NTERM = bra_terms<LA, LB>();
    constexpr int NSLOT = k_nslot(NTERM, L), SSTR = k_slot_stride(NTERM);
    constexpr bool RSMEM = L > 4;
    constexpr bool LOCKSTEP = L >= 5;
    using Ev = KEval<LA, LB, LC, LD>;
    static_assert(Ev::NBRA == NTERM, "generator and kernel disagree on the bra table");
    extern __shared__ __align__(16) double smem[];
    double *Rs = smem + threadIdx.x;                                  // [nherm(L)][NT] when RSMEM
    double *sB = smem + (RSMEM ? nherm(L) * NT : 0);                  // [NW][NSLOT][SSTR]: E row, Px,Py,Pz,p,coef,aoB
    double *s_red = sB + NW * NSLOT * SSTR;                           // [NW][NA*ND]
    int2 *queue = reinterpret_cast<int2 *>(s_red + NW * NA * ND);     // [NW][KQ] (ket, packed image)
    int *qbra = reinterpret_cast<int *>(queue + NW * KQ);             // [NW][KQ] running number of the bra
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    sB += w * NSLOT * SSTR;
    queue += w * KQ;
    qbra += w * KQ;
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

    // scan state of the warp (all warp-uniform except need_l, timg_l)
    int i = b0 + w;                       // next / current bra primitive pair-image
    int bcnt = 0;                         // bras started so far; the current one is number bcnt - 1
    bool bra_active = false, have = false;
    int head = 0, qn = 0;                 // ring of survivors
    int base = 0, nimg = 0, j0 = k0, timg = 0, timg_l = 0;
    int lo0 = 0, lo1 = 0, lo2 = 0, d2 = 1, d12 = 1;
    unsigned imask = 0;
    double thr = 0.0, ipi = 0.0, Pix = 0.0, Piy = 0.0, Piz = 0.0, cx = 0.0, cy = 0.0, cz = 0.0;
    double inv_isum_max = 0.0, rho2 = 0.0, need = 0.0, need_l = 0.0, ox = 0.0, oy = 0.0, oz = 0.0;

    for (;;) {
        // ---- phase 1: screen (bra, ket, image) candidates until 32 survivors are queued ----
        while (qn < 32) {
            if (!bra_active) {
                if (i >= b1) break;                                   // no bra left
                thr = __ldg(p.K.lb + i) + thr0;
                const double budget = thr + lbmax_ket;
                if (budget <= 0.0) { i = b1; break; }                 // bras sorted: the rest is weaker
                // the slot this bra takes must not be referenced by a queued survivor any more
                if (qn > 0 && bcnt - qbra[head] >= NSLOT) break;      // evaluate what is queued first
                double *slot = sB + (bcnt % NSLOT) * SSTR;
                Pix = __ldg(p.K.Px + i); Piy = __ldg(p.K.Py + i); Piz = __ldg(p.K.Pz + i);
                ipi = __ldg(p.K.ip + i);
                {
                    const double *__restrict__ src = p.K.etab + __ldg(p.K.eoff + i);
                    __syncwarp();
                    for (int n = lane; n < NTERM; n += 32) slot[n] = __ldg(src + n);
                    if (lane == 0) {
                        slot[NTERM] = Pix; slot[NTERM + 1] = Piy; slot[NTERM + 2] = Piz;
                        slot[NTERM + 3] = __ldg(p.K.p + i); slot[NTERM + 4] = __ldg(p.K.coef + i);
                        slot[NTERM + 5] = (double)__ldg(p.K.aoB + i);
                    }
                    __syncwarp();
                }
                // bounding box of the lattice images within reach of the ket group (eq 99-103)
                const double isum_max = ipi + kiqmax + lat.iomega2;
                const double rho = sqrt(budget * isum_max) + kext;
                cx = Pix - gx; cy = Piy - gy; cz = Piz - gz;
                const double f0 = lat.binv[0] * cx + lat.binv[1] * cy + lat.binv[2] * cz;
                const double f1 = lat.binv[3] * cx + lat.binv[4] * cy + lat.binv[5] * cz;
                const double f2 = lat.binv[6] * cx + lat.binv[7] * cy + lat.binv[8] * cz;
                lo0 = (int)ceil(f0 - rho * lat.bnorm[0]);
                lo1 = (int)ceil(f1 - rho * lat.bnorm[1]);
                lo2 = (int)ceil(f2 - rho * lat.bnorm[2]);
                const int hi0 = (int)floor(f0 + rho * lat.bnorm[0]), hi1 = (int)floor(f1 + rho * lat.bnorm[1]);
                const int hi2 = (int)floor(f2 + rho * lat.bnorm[2]);
                const int d1 = hi1 - lo1 + 1;
                d2 = hi2 - lo2 + 1;
                d12 = d1 * d2;
                nimg = (hi0 >= lo0 && d1 > 0 && d2 > 0) ? (hi0 - lo0 + 1) * d12 : 0;
                inv_isum_max = 1.0 / isum_max;
                rho2 = rho * rho;
                base = 0; imask = 0; have = false;
                bra_active = true;
                ++bcnt;
            }
            if (!have) {
                if (imask == 0) {
                    if (base >= nimg) { bra_active = false; i += NW; continue; }     // this bra is done
                    // 32 images of the box at a time, one per lane: sphere filter and the bound each image
                    // needs from a ket (eq 67 at the closest approach of the ket group)
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
                        double dlb = sqrt(dist2) - kext;        // lower bound of |Q + T - P|
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
            if (pass) {
                const int pos = (head + qn + __popc(m & ltmask)) & (KQ - 1);
                queue[pos] = make_int2(j, timg);
                qbra[pos] = bcnt - 1;
            }
            qn += __popc(m);
            j0 += 32;
            __syncwarp();
        }
        if (LOCKSTEP) {
            // the evaluators of the high classes are 10-60 thousand instructions of straight-line code, far more than
            // the instruction caches hold (ncu: 45 % of the stall samples of (dp|dp) were "no instruction"); the warps
            // of a CTA therefore enter the evaluator together and share the fetched lines.  Every warp passes this
            // barrier once per round until no warp has anything queued.
            if (!__syncthreads_or(qn > 0)) break;
            if (qn == 0) continue;
        } else if (qn == 0) break;                                    // nothing queued and no bra left
        // ---- phase 2: one primitive quartet-image per lane, oldest survivors first ----
        const int take = qn < 32 ? qn : 32;
        if (lane < take) {
            const int pos = (head + lane) & (KQ - 1);
            const int2 e = queue[pos];
            const double *__restrict__ slot = sB + (qbra[pos] % NSLOT) * SSTR;
            const int j = e.x;
            double Tx, Ty, Tz;
            unpack_img(e.y, lat, Tx, Ty, Tz);
            const double X = __ldg(kQx + j) + Tx - slot[NTERM], Y = __ldg(kQy + j) + Ty - slot[NTERM + 1],
                         Z = __ldg(kQz + j) + Tz - slot[NTERM + 2];
            const double pb = slot[NTERM + 3], q = __ldg(p.K.p + j);
            const double r2 = X * X + Y * Y + Z * Z;
            const double s = rsqrt(pb + q);
            const double alpha = pb * q * s * s;
            const double th = lat.omega * rsqrt(alpha + lat.omega2);
            const double alpha_w = alpha * th * th;
            const double pref = slot[NTERM + 4] * __ldg(p.K.coef + j) * s;
            const double *__restrict__ Pb = p.Pp + (size_t)(int)slot[NTERM + 5] * p.ldP + __ldg(p.K.aoB + j);
            double Rm[L + 1];
            boys_merged<L>(tab, r2, alpha, alpha_w, th, pref, Rm);
            Ev::template run<NT>(slot, p.K.etab + __ldg(p.K.eoff + j), Pb, p.ldP, Rm, X, Y, Z, Rs, Kacc);
        }
        head = (head + take) & (KQ - 1);
        qn -= take;
        nquart += take;
        __syncwarp();
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
