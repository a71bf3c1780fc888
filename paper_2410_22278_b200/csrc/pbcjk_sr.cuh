// Real-space (erfc(w r)/r) quartet kernels: J-engine (eq 95-98) and K (eq 74 L558 with
// eq 56/69).  One kernel family per angular-momentum class, generated from templates.
//
// Mapping (differs from PAPER 3.2 L753, which gives one THREAD a bra pair and lets it loop over
// its own lattice sphere -> warp divergence, L882).  Both families run a two-level screen in front
// of a convergent evaluator:
//   * level A (lane-parallel, fp32): an ITEM is a (ket group, lattice image) pair for the J-engine
//     (the warp owns one bra) or a (bra, lattice image) pair for K (the CTA owns one ket group).  32
//     items are screened at a time, one per lane: distance of the bra centre to the translated group
//     centre, the bound `need` a ket of that group must exceed there (eq 67 at the closest approach),
//     and -- the kets of a group being sorted by bound -- the NUMBER of kets that exceed it, by binary
//     search.  Items with a zero count cost nothing further.
//   * level B: for every live item (ballot + shuffle broadcast) the lanes test its kets, 32 at a time, with the eq-67 screen in fp32 on 16-byte screen records (positions relative to the group
//     centre), then with the per-shell-block max |P| (L819); survivors go to a per-warp ring in shared
//     memory (ballot + popc compaction).
//   * evaluation (expensive, convergent, fp64): whenever 32 survivors are queued every lane evaluates
//     one primitive quartet-image: merged Boys values, Hermite R recursion, contraction.
//   * accumulators stay in registers; warp-shuffle + shared-memory reductions; every output element
//     has exactly one owner, so there are no global atomics on the data path.
// The fp32 screen keeps a superset of the fp64 rule (slack SCREEN_MARGIN in the logarithm of the bound).
#pragma once
#include "pbcjk_md.cuh"
#include <type_traits>

namespace pbcjk {

struct SRParams {
    PairListK K;
    PairListU U;
    KetListJ KJ;
    Lattice lat;
    ShellInfo sh;
    BoysTab boys;
    const double *Pp;        // P with component factors folded in, row stride ldP
    const float *Ppf;        // fp32 copy of P' (mixed precision), same stride
    int ldP;
    const double *Dt;        // Hermite densities of the J kets, Dt[s*dstride + j]   (eq 95)
    double *Jt;              // Hermite J of the U entries, Jt[t*U.n + u]            (eq 98, raw)
    double *Ksr;             // N x N, accumulated block by block
    const double *lnPmax;    // device scalar ln(max |P'|)
    const float *lnPblk;     // [nshell*nshell] ln(max |P'|) over each shell block (L819)
    const float *lnProw;     // [nshell] row maxima of lnPblk
    const float *kjP;        // [KJ.n] lnPblk of each J ket's own shell pair
    double ln_tau;           // ln(d_schwarz)
    double rcut2;            // r_cut^2 (C-14) or +inf
    float ln_switch;         // mixed precision: ln(mixed_switch); quartets whose ln(bound_bra bound_ket max|P block|)
                             // is below it are evaluated in fp32 (PAPER 3.5 L819)
    int shard_rank, shard_n; // multi-GPU: this rank takes blocks / bras with index % shard_n == shard_rank
    unsigned long long *counters;
};

#ifndef J_UNR
#define J_UNR 6                 // candidate passes per screening step
#endif
constexpr int J_KET_BITS = 26;  // ring entries pack (ket, image): at most 2^26 J kets (checked at create), NIMG_J = 64 images per chunk
constexpr int QCAP = 256;       // survivor ring per warp (power of two): up to 31 queued + 32 * J_UNR new survivors per screening step
static_assert(31 + 32 * J_UNR <= QCAP, "ring too small");
constexpr int NIMG_J = 64;      // lattice images per warp-level list chunk (J-engine)

__device__ __forceinline__ void lattice_T(const Lattice &lat, int n0, int n1, int n2, double &Tx, double &Ty, double &Tz)
{
    Tx = n0 * lat.a[0] + n1 * lat.a[3] + n2 * lat.a[6];
    Ty = n0 * lat.a[1] + n1 * lat.a[4] + n2 * lat.a[7];
    Tz = n0 * lat.a[2] + n1 * lat.a[5] + n2 * lat.a[8];
}

// Bounding box (eq 99-103) of the lattice points within `rad` of the point c.
struct ImageBox {
    int lo0, lo1, lo2, d2, d12, n;
    __device__ __forceinline__ void set(const Lattice &lat, double cx, double cy, double cz, double rad)
    {
        const double f0 = lat.binv[0] * cx + lat.binv[1] * cy + lat.binv[2] * cz;
        const double f1 = lat.binv[3] * cx + lat.binv[4] * cy + lat.binv[5] * cz;
        const double f2 = lat.binv[6] * cx + lat.binv[7] * cy + lat.binv[8] * cz;
        lo0 = (int)ceil(f0 - rad * lat.bnorm[0]);
        lo1 = (int)ceil(f1 - rad * lat.bnorm[1]);
        lo2 = (int)ceil(f2 - rad * lat.bnorm[2]);
        const int hi0 = (int)floor(f0 + rad * lat.bnorm[0]), hi1 = (int)floor(f1 + rad * lat.bnorm[1]);
        const int hi2 = (int)floor(f2 + rad * lat.bnorm[2]);
        const int d1 = hi1 - lo1 + 1;
        d2 = hi2 - lo2 + 1;
        d12 = d1 * d2;
        n = (hi0 >= lo0 && d1 > 0 && d2 > 0) ? (hi0 - lo0 + 1) * d12 : 0;
    }
    __device__ __forceinline__ void decode(int im, int &n0, int &n1, int &n2) const
    {
        n0 = lo0 + im / d12;
        const int r = im % d12;
        n1 = lo1 + r / d2;
        n2 = lo2 + r % d2;
    }
};

// number of leading entries of a list sorted by descending bound (q4[].w) that exceed `need` (per lane).
// Four-way search: the three pivots of a step are independent loads, so the chain of dependent loads is half as long as that
// of a binary search (level A of the screens waits on this chain in nearly every batch of 32 items).
__device__ __forceinline__ int count_above_sorted(const float4 *__restrict__ q4, int n, float need)
{
    int lo = 0, hi = n;                                      // invariant: entries < lo exceed need, entries >= hi do not
    while (hi - lo > 3) {
        const int q = (hi - lo) >> 2;
        const int m1 = lo + q, m2 = lo + 2 * q, m3 = lo + 3 * q;
        const float v1 = __ldg(&q4[m1].w), v2 = __ldg(&q4[m2].w), v3 = __ldg(&q4[m3].w);
        if (v2 > need) {
            if (v3 > need) lo = m3 + 1;
            else { lo = m2 + 1; hi = m3; }
        } else {
            if (v1 > need) { lo = m1 + 1; hi = m2; }
            else hi = m1;
        }
    }
    while (lo < hi && __ldg(&q4[lo].w) > need) ++lo;         // at most three entries left
    return lo;
}

// ------------------------------------------------------------------------------------------
// J-engine: bra Hermite order LB (= la+lb), ket Hermite order LK.  One warp per bra U entry.
//   Jt[t] += sum_kets pref * sum_s R_{t+s}(Q - P + R1) D~_s        (eq 98 second term, reading C-4;
//   the (-1)^{|t|} and E^{ab}_t are applied by the back-transform kernel, eq 97)
// Ket groups: (atom of the ket's home shell, LK), sorted by bound; an item is (atom, lattice image).
// ------------------------------------------------------------------------------------------
template <int LB, int LK>
__global__ void __launch_bounds__(128) sr_j_kernel(SRParams p, const int *__restrict__ bra_idx, int nbra)
{
    constexpr int L = LB + LK;
    constexpr int NT = nherm(LB), NS = nherm(LK);
    __shared__ unsigned s_queue[4][QCAP];                       // ket index | image index << J_KET_BITS
    __shared__ double s_T[4][3][NIMG_J];
    __shared__ float s_C[4][3][NIMG_J];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int ib = blockIdx.x * 4 + w;
    if (p.shard_n > 1) ib = ib * p.shard_n + p.shard_rank;
    if (ib >= nbra) return;
    const KetListJ &KJ = p.KJ;
    const Lattice &lat = p.lat;
    const int u = __ldg(bra_idx + ib);
    const double Pix = p.U.Px[u], Piy = p.U.Py[u], Piz = p.U.Pz[u];
    const double pi_ = p.U.p[u], coefi = p.U.coef[u];
    const float ipi = (float)p.U.ip[u];
    const float M = SCREEN_MARGIN;
    const float ln_tau = (float)p.ln_tau;
    const float lbi = (float)p.U.lb[u];
    const float thr = lbi + (float)*p.lnPmax - ln_tau;          // level A: global max |P'|
    const float thrx = lbi - ln_tau;                              // level B refinement: + per-ket block max
    const float iw2 = (float)lat.iomega2;
    const float rcut2f = p.rcut2 < 1e30 ? (float)p.rcut2 * 1.00001f : 3.0e38f;
    double Jt[NT];
#pragma unroll
    for (int t = 0; t < NT; ++t) Jt[t] = 0.0;
    unsigned *queue = s_queue[w];
    double *sT = &s_T[w][0][0];
    float *sC = &s_C[w][0][0];
    const unsigned ltmask = (1u << lane) - 1u;
    unsigned ncand = 0;
    unsigned long long nquart = 0;
    int head = 0, qn = 0;

    // images of the whole ket set within reach of this bra: sphere around P - g0 (g0 = cell centre; every atom
    // lies within KJ.rc of it), radius = reach of the strongest ket of order LK + its extent + rc
    const float budget_all = thr + KJ.lbmax[LK] + M;
    ImageBox box;
    box.n = 0;
    double Rall = 0.0;
    const double c0x = Pix - KJ.g0[0], c0y = Piy - KJ.g0[1], c0z = Piz - KJ.g0[2];
    if (budget_all > 0.f) {
        Rall = sqrt((double)budget_all * (double)(ipi + KJ.iqmaxall[LK] + iw2)) + KJ.extmax[LK] + KJ.rc + 1e-3;
        box.set(lat, c0x, c0y, c0z, Rall);
    }
    const int natom = KJ.ngroup;
    for (int ibox = 0; ibox < box.n;) {
        // ---- image list chunk of this warp ----
        int nimg = 0;
        __syncwarp();
        while (ibox < box.n && nimg <= NIMG_J - 32) {
            const int im = ibox + lane;
            bool ok = false;
            double Tx = 0, Ty = 0, Tz = 0;
            if (im < box.n) {
                int n0, n1, n2;
                box.decode(im, n0, n1, n2);
                lattice_T(lat, n0, n1, n2, Tx, Ty, Tz);
                const double ex = c0x - Tx, ey = c0y - Ty, ez = c0z - Tz;
                ok = ex * ex + ey * ey + ez * ez <= Rall * Rall;
            }
            const unsigned m = __ballot_sync(0xffffffffu, ok);
            if (ok) {
                const int pos = nimg + __popc(m & ltmask);
                sT[pos] = Tx; sT[NIMG_J + pos] = Ty; sT[2 * NIMG_J + pos] = Tz;
                sC[pos] = (float)(c0x - Tx); sC[NIMG_J + pos] = (float)(c0y - Ty); sC[2 * NIMG_J + pos] = (float)(c0z - Tz);
            }
            nimg += __popc(m);
            ibox += 32;
        }
        __syncwarp();
        const int nitems = natom * nimg;
        const float inv_nimg = 1.f / (float)max(nimg, 1);
        int ebase = 0;
        unsigned imask = 0;
        bool have = false, items_done = false;
        // per-lane item, current item
        int it_cnt = 0, it_k0 = 0, it_t = 0;
        float it_Dx = 0.f, it_Dy = 0.f, it_Dz = 0.f;
        int c_cnt = 0, c_k0 = 0, c_t = 0, jpos = 0;
        float c_Dx = 0.f, c_Dy = 0.f, c_Dz = 0.f;
        for (;;) {
            while (qn < 32) {
                if (!have) {
                    if (imask == 0) {
                        if (ebase >= nitems) { items_done = true; break; }
                        const int e = ebase + lane;
                        ebase += 32;
                        it_cnt = 0;
                        if (e < nitems) {
                            int a = (int)((float)e * inv_nimg), t = e - a * nimg;       // e / nimg without the integer division
                            if (t < 0) { --a; t += nimg; } else if (t >= nimg) { ++a; t -= nimg; }
                            const int gi = a * 5 + LK;
                            const int2 go = __ldg(KJ.goff + gi);                   // (first ket, count)
                            if (go.y > 0) {
                                const float4 gr = __ldg(KJ.grec + gi);             // (ext, iqmax, lbmax, -)
                                const float4 ga = __ldg(KJ.g4 + a);                // atom position - g0
                                const float Dx = sC[t] - ga.x, Dy = sC[NIMG_J + t] - ga.y, Dz = sC[2 * NIMG_J + t] - ga.z;
                                const float dist = sqrtf(Dx * Dx + Dy * Dy + Dz * Dz);
                                const float dlb = fmaxf(dist * (1.f - 4e-6f) - gr.x - 1e-4f, 0.f);
                                const float need = __fdividef(dlb * dlb, ipi + gr.y + iw2) - thr - 2.f * M;
                                if (need < gr.z) {                                 // the strongest ket could survive
                                    it_cnt = count_above_sorted(KJ.q4 + go.x, go.y, need);   // kets sorted by bound
                                    it_k0 = go.x; it_t = t; it_Dx = Dx; it_Dy = Dy; it_Dz = Dz;
                                }
                            }
                        }
                        imask = __ballot_sync(0xffffffffu, it_cnt > 0);
                        continue;
                    }
                    const int src = __ffs(imask) - 1;
                    imask &= imask - 1;
                    c_cnt = __shfl_sync(0xffffffffu, it_cnt, src);
                    c_k0 = __shfl_sync(0xffffffffu, it_k0, src);
                    c_t = __shfl_sync(0xffffffffu, it_t, src);
                    c_Dx = __shfl_sync(0xffffffffu, it_Dx, src);
                    c_Dy = __shfl_sync(0xffffffffu, it_Dy, src);
                    c_Dz = __shfl_sync(0xffffffffu, it_Dz, src);
                    jpos = 0;
                    have = true;
                }
                if (jpos >= c_cnt) { have = false; continue; }
                // Several passes of 32 candidates per step -- 2, or J_UNR when the item still holds more than 64 --: all
                // records are requested before any is tested (a pass is a chain of dependent loads and a ballot: the scan is
                // bound by that latency, not by issue slots; si64 J 625 -> 492 ms, water64 120 -> 116 ms)
                auto passes = [&](auto UC) {
                    constexpr int U = decltype(UC)::value;
                    const int jbase = jpos + lane;
                    const int npass = min(U, (c_cnt - jpos + 31) >> 5);        // warp-uniform
                    jpos += 32 * U;
                    float4 k4[U];
                    float iq[U], kp[U];
#pragma unroll
                    for (int u2 = 0; u2 < U; ++u2) {
                        const int jj = jbase + 32 * u2;
                        k4[u2] = make_float4(0.f, 0.f, 0.f, 0.f); iq[u2] = 0.f; kp[u2] = 0.f;
                        if (jj < c_cnt) { k4[u2] = __ldg(KJ.q4 + c_k0 + jj); iq[u2] = __ldg(KJ.iqf + c_k0 + jj); kp[u2] = __ldg(p.kjP + c_k0 + jj); }
                    }
#pragma unroll
                    for (int u2 = 0; u2 < U; ++u2) {
                        if (u2 < npass) {
                            const int jj = jbase + 32 * u2;
                            bool pass = false;
                            if (jj < c_cnt) {
                                const float ex = k4[u2].x - c_Dx, ey = k4[u2].y - c_Dy, ez = k4[u2].z - c_Dz;   // Q + T - P
                                const float r2 = ex * ex + ey * ey + ez * ez;
                                const float isum = ipi + iq[u2] + iw2;
                                pass = (thrx + k4[u2].w + kp[u2] + M) * isum > r2 && r2 <= rcut2f;   // per-block max |P'| (L819)
                                ++ncand;
                            }
                            const unsigned m = __ballot_sync(0xffffffffu, pass);
                            if (pass) queue[(head + qn + __popc(m & ltmask)) & (QCAP - 1)] = (unsigned)(c_k0 + jj) | ((unsigned)c_t << J_KET_BITS);
                            qn += __popc(m);
                        }
                    }
                };
                if (c_cnt - jpos <= 32 && imask != 0) {
                    // the last pass of this item runs together with the first pass of the next live item of the batch (an
                    // item holds 12 candidates on average on water64: one item per step is one latency chain per item)
                    const int src = __ffs(imask) - 1;
                    imask &= imask - 1;
                    const int d_cnt = __shfl_sync(0xffffffffu, it_cnt, src), d_k0 = __shfl_sync(0xffffffffu, it_k0, src),
                              d_t = __shfl_sync(0xffffffffu, it_t, src);
                    const float d_Dx = __shfl_sync(0xffffffffu, it_Dx, src), d_Dy = __shfl_sync(0xffffffffu, it_Dy, src),
                                d_Dz = __shfl_sync(0xffffffffu, it_Dz, src);
                    const int jj0 = jpos + lane, jj1 = lane;
                    const bool va = jj0 < c_cnt, vb = jj1 < d_cnt;
                    float4 ka = make_float4(0.f, 0.f, 0.f, 0.f), kb = ka;
                    float iqa = 0.f, iqb = 0.f, kpa = 0.f, kpb = 0.f;
                    if (va) { ka = __ldg(KJ.q4 + c_k0 + jj0); iqa = __ldg(KJ.iqf + c_k0 + jj0); kpa = __ldg(p.kjP + c_k0 + jj0); }
                    if (vb) { kb = __ldg(KJ.q4 + d_k0 + jj1); iqb = __ldg(KJ.iqf + d_k0 + jj1); kpb = __ldg(p.kjP + d_k0 + jj1); }
                    bool pa = false, pb = false;
                    if (va) {
                        const float ex = ka.x - c_Dx, ey = ka.y - c_Dy, ez = ka.z - c_Dz;
                        const float r2 = ex * ex + ey * ey + ez * ez;
                        pa = (thrx + ka.w + kpa + M) * (ipi + iqa + iw2) > r2 && r2 <= rcut2f;
                        ++ncand;
                    }
                    if (vb) {
                        const float ex = kb.x - d_Dx, ey = kb.y - d_Dy, ez = kb.z - d_Dz;
                        const float r2 = ex * ex + ey * ey + ez * ez;
                        pb = (thrx + kb.w + kpb + M) * (ipi + iqb + iw2) > r2 && r2 <= rcut2f;
                        ++ncand;
                    }
                    const unsigned ma = __ballot_sync(0xffffffffu, pa);
                    if (pa) queue[(head + qn + __popc(ma & ltmask)) & (QCAP - 1)] = (unsigned)(c_k0 + jj0) | ((unsigned)c_t << J_KET_BITS);
                    qn += __popc(ma);
                    const unsigned mb = __ballot_sync(0xffffffffu, pb);
                    if (pb) queue[(head + qn + __popc(mb & ltmask)) & (QCAP - 1)] = (unsigned)(d_k0 + jj1) | ((unsigned)d_t << J_KET_BITS);
                    qn += __popc(mb);
                    c_cnt = d_cnt; c_k0 = d_k0; c_t = d_t; c_Dx = d_Dx; c_Dy = d_Dy; c_Dz = d_Dz;
                    jpos = 32;
                } else if (c_cnt - jpos > 64) passes(std::integral_constant<int, J_UNR>());
                else passes(std::integral_constant<int, 2>());
                __syncwarp();
            }
            if (!(qn >= 32 || (items_done && qn > 0))) break;
            // ---- evaluation: one primitive quartet-image per lane ----
            const int take = qn < 32 ? qn : 32;
            if (lane < take) {
                const unsigned e = queue[(head + lane) & (QCAP - 1)];
                const int j = (int)(e & ((1u << J_KET_BITS) - 1u)), t = (int)(e >> J_KET_BITS);
                const double X = __ldg(KJ.Qx + j) + sT[t] - Pix, Y = __ldg(KJ.Qy + j) + sT[NIMG_J + t] - Piy,
                             Z = __ldg(KJ.Qz + j) + sT[2 * NIMG_J + t] - Piz;
                const double q = __ldg(KJ.q + j);
                const double r2 = X * X + Y * Y + Z * Z;
                const double s = rsqrt(pi_ + q);
                const double alpha = pi_ * q * s * s;
                const double th = lat.omega * rsqrt(alpha + lat.omega2);
                const double alpha_w = alpha * th * th;
                const double pref = r2 <= p.rcut2 ? coefi * __ldg(KJ.coef + j) * s : 0.0;
                double Rm[L + 1];
                boys_merged<L, double>(p.boys, r2, alpha, alpha_w, th, pref, Rm);
                double R[nherm(L)];
                hermite_R<L>(R, Rm, X, Y, Z);
                double D[NS];
#pragma unroll
                for (int sI = 0; sI < NS; ++sI) D[sI] = __ldg(p.Dt + (size_t)sI * KJ.dstride + j);
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
            }
            head = (head + take) & (QCAP - 1);
            qn -= take;
            nquart += take;
            __syncwarp();
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
    unsigned long long c = ncand;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) {
        atomicAdd(p.counters + CNT_CAND_J + LB * 5 + LK, c);
        atomicAdd(p.counters + CNT_Q_J + LB * 5 + LK, nquart);
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

// launchers (defined in the instantiation units); `mixed` selects the fp64+fp32 K kernels
void launch_sr_j(int LB, int LK, const SRParams &p, const int *bra_idx, int nbra, cudaStream_t st);
void launch_sr_k(int la, int lb, int lc, int ld, bool mixed, const SRParams &p, const int2 *blocks, int nblocks, cudaStream_t st);
// opt in to the dynamic shared memory of every K class on the current device (once per handle)
void sr_k_set_attributes();

}  // namespace pbcjk
