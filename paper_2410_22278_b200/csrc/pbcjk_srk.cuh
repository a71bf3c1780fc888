// Real-space K kernels (eq 74 L558 with eq 56/69): class (LA LB | LC LD), bra = (mu: LA, lambda: LB),
// ket = (nu: LD, sigma: LC).  One CTA owns the output block (mu, nu):
//   K[mu_a, nu_d] += sum P'[lambda_b, sigma_c] (mu_a lambda_b | sigma_c nu_d)
//
// Screen (see pbcjk_sr.cuh): the CTA lists the lattice images R1 that can couple the bra group (mu, all lambda of
// class LB) with the ket group (nu, all sigma of class LC) once (eq 99-103: bounding box, then sphere filter); an
// ITEM is a (bra primitive pair-image, image) pair; the warps take the items 32 at a time, one per lane (level A:
// distance to the ket group, the bound a ket needs there, number of kets above it by binary search in the list sorted
// by bound), then test the kets of every live item in fp32 (level B: eq 67 with the row maximum of |P'|, then with
// the maximum over the shell block (lambda, sigma), L819).  Survivors wait in a per-warp ring as (bra, ket, image);
// whenever 32 are queued each lane evaluates one primitive quartet-image with the straight-line evaluator generated
// per class by gen_sr_k.py.  The Hermite integrals of classes with L > 4 live in shared memory (one column per
// thread); the E products of both pairs come from the tables built at create (PairListK::etab), so no E recursion
// runs per quartet.
//
// MIXED (PAPER 3.5 L817-821): a second ring takes the survivors whose ln(bound_bra bound_ket max|P block|) is below
// ln(mixed_switch); they run the same evaluator instantiated for float (fp32 tables, fp32 density), accumulated
// into the fp64 block sums.  The bound used for the switch leaves out the exp(-alpha_w r^2) factor of eq 67 on
// purpose: the erfc-attenuated integral is a difference of two Boys terms, and fp32 rounding acts on the terms, not
// on their difference.
#pragma once
#include "pbcjk_sr.cuh"

namespace pbcjk {

template <int LA, int LB, int LC, int LD> struct KEval;      // specialisations: build/gen/k_eval_*.cuh

__device__ __forceinline__ double ldg_volatile(const double *p)
{
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ float ldg_volatile(const float *p)
{
    float v;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}

// CTA size: 128 threads in every class.  The warps of a CTA enter the evaluator in lockstep at L >= 5 (see LOCKSTEP
// below), so four warps share the instruction fetches; the R column of a thread takes 8*nherm(L) bytes of shared
// memory (1320 B at L = 8: one CTA per SM).
// (256-thread CTAs at L = 5, 6 -- 8 warps per lockstep round -- measured 86 / 48 ms against 70 / 47 ms with 128)
__host__ __device__ constexpr int k_nthreads(int) { return 128; }
#define K_MIXED_LMAX 4                                        // highest class order with a mixed-precision kernel
#ifndef K_LOCK_LMIN
#define K_LOCK_LMIN 5                                         // lowest class order evaluated in lockstep rounds (fp64 kernels; at 4: 70 -> 84 ms)
#endif
constexpr int KQ = 64;                                       // ring capacity per warp (power of two), classes with L <= 4
// Classes with L >= 5 evaluate in lockstep rounds in which the FOUR rings of the CTA are drained as one queue (see the
// kernel): a warp may then collect up to 64 survivors before a round, so its ring holds up to 95 (128 / ring 256 measured:
// water64 K 366.6 -> 363.3 ms but si64 K 1868 -> 1977 ms; 32: 392 and 1956 ms)
__host__ __device__ constexpr bool k_lockstep(int L, bool mixed) { return L >= K_LOCK_LMIN && !mixed; }
__host__ __device__ constexpr int k_ring(int L, bool mixed) { return k_lockstep(L, mixed) ? 128 : KQ; }
__host__ __device__ constexpr int k_qstop(int L, bool mixed) { return k_lockstep(L, mixed) ? 64 : 32; }
#ifndef K_PAIR
#define K_PAIR 1                                              // level B: pair an item's last pass with the next item's first
#endif
constexpr int NIMG_K = 128;                                  // lattice images per CTA-level list chunk


template <int LA, int LB, int LC, int LD, bool MIXED>
constexpr size_t k_smem_bytes()
{
    constexpr int L = LA + LB + LC + LD, NT = k_nthreads(L), NW = NT / 32;
    size_t d = (L > 4 ? (size_t)nherm(L) * NT : 0) + (size_t)NW * ncart(LA) * ncart(LD) + 3 * NIMG_K;
    return d * sizeof(double) + 3 * NIMG_K * sizeof(float) + (size_t)NW * k_ring(L, MIXED) * sizeof(int2) * (MIXED ? 2 : 1);
}

// light classes: at most 128 registers (L <= 3: 4 CTAs, 16 warps per SM) or 168 (L = 4: 3 CTAs); the few spilled
// doubles cost less than the lost occupancy
__host__ __device__ constexpr int k_minblocks(int L) { return L <= 3 ? 4 : (L == 4 ? 3 : 1); }

// CTA-wide: number of leading entries (sorted by descending q4[].w) above `bound`
__device__ __forceinline__ int count_above_cta(const float4 *__restrict__ q4, int n, float bound)
{
    int tot = 0;
    for (int base = 0; base < n; base += blockDim.x) {
        const int idx = base + threadIdx.x;
        const int c = __syncthreads_count(idx < n && __ldg(&q4[idx].w) > bound);
        tot += c;
        if (c < (int)blockDim.x) break;
    }
    return tot;
}

template <int LA, int LB, int LC, int LD, bool MIXED>
__global__ void __launch_bounds__(k_nthreads(LA + LB + LC + LD), k_minblocks(LA + LB + LC + LD))
sr_k_kernel(SRParams p, const int2 *__restrict__ blocks, int nblocks)
{
    constexpr int L = LA + LB + LC + LD;
    constexpr int NT = k_nthreads(L), NW = NT / 32;
    constexpr int NA = ncart(LA), ND = ncart(LD);
    constexpr bool RSMEM = L > 4;
    constexpr bool LOCKSTEP = k_lockstep(L, MIXED);
    constexpr int KQ = k_ring(L, MIXED), QSTOP = k_qstop(L, MIXED);                 // shadows the namespace constant
    static_assert(!(LOCKSTEP && MIXED), "the mixed mode exists for L <= 4 only");
    using Ev = KEval<LA, LB, LC, LD>;
    static_assert(Ev::NBRA == bra_terms<LA, LB>(), "generator and kernel disagree on the bra table");
    extern __shared__ __align__(16) double smem[];
    // R columns when RSMEM: [warp][nherm(L)][32], one column per thread inside the warp's own slice -- the float columns of
    // a warp's fp32 pass (MIXED) reuse that slice, so warps evaluating in different precisions never touch each other
    double *Rs = smem + (size_t)(threadIdx.x >> 5) * nherm(L) * 32 + (threadIdx.x & 31);
    double *s_red = smem + (RSMEM ? nherm(L) * NT : 0);               // [NW][NA*ND]
    double *sT = s_red + NW * NA * ND;                                // [3][NIMG_K] lattice vectors of the image list
    float *sC = reinterpret_cast<float *>(sT + 3 * NIMG_K);           // [3][NIMG_K] centre(mu) - centre(nu) - T
    int2 *queue = reinterpret_cast<int2 *>(sC + 3 * NIMG_K);          // [NW][KQ] (bra | ket << 16, image)
    int2 *queue32 = queue + NW * KQ;                                  // [NW][KQ] fp32 ring (MIXED)
    __shared__ int s_ctl[2];
    __shared__ int s_cnt[8], s_head[8], s_done[8];                    // LOCKSTEP: the rings of the four warps, published per round
    int2 *const qall = queue;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    queue += w * KQ;
    queue32 += w * KQ;
    const PairListK &K = p.K;
    const int bidx = p.shard_n > 1 ? blockIdx.x * p.shard_n + p.shard_rank : blockIdx.x;
    if (bidx >= nblocks) return;
    const int2 blk = blocks[bidx];
    const int mu = blk.x, nu = blk.y;
    const int b0 = __ldg(K.off + mu * 3 + LB), b1 = __ldg(K.off + mu * 3 + LB + 1);
    const int k0 = __ldg(K.off + nu * 3 + LC), k1 = __ldg(K.off + nu * 3 + LC + 1);
    if (b1 <= b0 || k1 <= k0) return;
    const Lattice &lat = p.lat;
    const int N = p.sh.nbf, ns = p.sh.nshell;
    const float M = SCREEN_MARGIN;
    const float ln_tau = (float)p.ln_tau;
    const float lnPmax = (float)*p.lnPmax;
    const float iw2 = (float)lat.iomega2;
    const float rcut2f = p.rcut2 < 1e30 ? (float)p.rcut2 * 1.00001f : 3.0e38f;
    const float lbmax_bra = __ldg(&K.q4[b0].w), lbmax_ket = __ldg(&K.q4[k0].w);
    const float budget_blk = lbmax_bra + lbmax_ket + lnPmax - ln_tau + M;
    if (budget_blk <= 0.f) return;
    // entries that can survive at all (lists sorted by bound)
    const int nb_eff = count_above_cta(K.q4 + b0, b1 - b0, -(lbmax_ket + lnPmax - ln_tau + M));
    const int nk_eff = count_above_cta(K.q4 + k0, k1 - k0, -(lbmax_bra + lnPmax - ln_tau + M));
    const float kext = (float)__ldg(K.ext + nu * 3 + LC), kiqmax = (float)__ldg(K.ipmax + nu * 3 + LC);
    const float4 *__restrict__ kq4 = K.q4 + k0;
    const float *__restrict__ kipf = K.ipf + k0;
    const int *__restrict__ kshB = K.shB + k0;
    const unsigned ltmask = (1u << lane) - 1u;

    // lattice images within reach of the two groups: sphere around centre(mu) - centre(nu)
    const double cx = __ldg(p.sh.cx + mu) - __ldg(p.sh.cx + nu), cy = __ldg(p.sh.cy + mu) - __ldg(p.sh.cy + nu),
                 cz = __ldg(p.sh.cz + mu) - __ldg(p.sh.cz + nu);
    const double Rblk = sqrt((double)budget_blk * ((double)__ldg(K.ipmax + mu * 3 + LB) + kiqmax + iw2)) + kext +
                        __ldg(K.ext + mu * 3 + LB) + 1e-3;
    ImageBox box;
    box.set(lat, cx, cy, cz, Rblk);

    double Kacc[NA * ND];
#pragma unroll
    for (int i = 0; i < NA * ND; ++i) Kacc[i] = 0.0;
    unsigned ncand = 0;
    unsigned long long nquart = 0, nquart32 = 0;
    int head = 0, qn = 0, head32 = 0, qn32 = 0;

    for (int ibox = 0; ibox < box.n;) {
        // ---- CTA-level image list chunk, filled by warp 0 in box order (deterministic) ----
        __syncthreads();
        if (w == 0) {
            int n = 0, ib = ibox;
            while (ib < box.n && n <= NIMG_K - 32) {
                const int im = ib + lane;
                bool ok = false;
                double Tx = 0, Ty = 0, Tz = 0;
                if (im < box.n) {
                    int n0, n1, n2;
                    box.decode(im, n0, n1, n2);
                    lattice_T(lat, n0, n1, n2, Tx, Ty, Tz);
                    const double ex = cx - Tx, ey = cy - Ty, ez = cz - Tz;
                    ok = ex * ex + ey * ey + ez * ez <= Rblk * Rblk;
                }
                const unsigned m = __ballot_sync(0xffffffffu, ok);
                if (ok) {
                    const int pos = n + __popc(m & ltmask);
                    sT[pos] = Tx; sT[NIMG_K + pos] = Ty; sT[2 * NIMG_K + pos] = Tz;
                    sC[pos] = (float)(cx - Tx); sC[NIMG_K + pos] = (float)(cy - Ty); sC[2 * NIMG_K + pos] = (float)(cz - Tz);
                }
                n += __popc(m);
                ib += 32;
            }
            if (lane == 0) { s_ctl[0] = n; s_ctl[1] = ib; }
        }
        __syncthreads();
        const int nimg = s_ctl[0];
        ibox = s_ctl[1];
        const int nitems = nb_eff * nimg;
        const float inv_nimg = 1.f / (float)max(nimg, 1);
        int ebase = w * 32;
        unsigned imask = 0;
        bool have = false, items_done = false;
        // per-lane item (level A result) and the item being scanned (warp-uniform)
        int it_cnt = 0, it_ibt = 0, c_ibt = 0, c_cnt = 0, jpos = 0;  // it_ibt: bra | image << 16
        float it_Dx = 0.f, it_Dy = 0.f, it_Dz = 0.f, it_thr = 0.f, it_ipi = 0.f;
        float c_Dx = 0.f, c_Dy = 0.f, c_Dz = 0.f, c_thr = 0.f, c_ipi = 0.f;
        for (;;) {
            // ---- screen until 32 survivors are queued (in either ring) or the items run out ----
            while (qn < QSTOP && (!MIXED || qn32 < 32)) {
                if (!have) {
                    if (imask == 0) {
                        if (ebase >= nitems) { items_done = true; break; }
                        const int e = ebase + lane;
                        ebase += 32 * NW;
                        it_cnt = 0;
                        if (e < nitems) {
                            int ib = (int)((float)e * inv_nimg), t = e - ib * nimg;   // e / nimg without the integer division
                            if (t < 0) { --ib; t += nimg; } else if (t >= nimg) { ++ib; t -= nimg; }
                            const int i = b0 + ib;
                            const float4 b4 = __ldg(K.q4 + i);                     // (P - mu).xyz, lb
                            const float ipi = __ldg(K.ipf + i);
                            const float thr = b4.w + __ldg(p.lnProw + __ldg(K.shB + i)) - ln_tau;
                            const float Dx = b4.x + sC[t], Dy = b4.y + sC[NIMG_K + t], Dz = b4.z + sC[2 * NIMG_K + t];
                            const float dist = sqrtf(Dx * Dx + Dy * Dy + Dz * Dz);   // |P - (nu + T)|
                            const float dlb = fmaxf(dist * (1.f - 4e-6f) - kext - 1e-4f, 0.f);
                            const float need = __fdividef(dlb * dlb, ipi + kiqmax + iw2) - thr - 2.f * M;
                            if (need < lbmax_ket) {                                // the strongest ket could survive
                                it_cnt = count_above_sorted(kq4, nk_eff, need);    // kets sorted by bound
                                it_ibt = ib | (t << 16); it_Dx = Dx; it_Dy = Dy; it_Dz = Dz;
                                it_thr = thr; it_ipi = ipi;
                            }
                        }
                        imask = __ballot_sync(0xffffffffu, it_cnt > 0);
                        continue;
                    }
                    const int src = __ffs(imask) - 1;
                    imask &= imask - 1;
                    c_ibt = __shfl_sync(0xffffffffu, it_ibt, src);
                    c_Dx = __shfl_sync(0xffffffffu, it_Dx, src);
                    c_Dy = __shfl_sync(0xffffffffu, it_Dy, src);
                    c_Dz = __shfl_sync(0xffffffffu, it_Dz, src);
                    c_thr = __shfl_sync(0xffffffffu, it_thr, src);
                    c_ipi = __shfl_sync(0xffffffffu, it_ipi, src);
                    c_cnt = __shfl_sync(0xffffffffu, it_cnt, src);
                    jpos = 0;
                    have = true;
                }
                if (jpos >= c_cnt) { have = false; continue; }
                // test of one candidate per lane (screen record k4, 1/q already loaded) and compaction of the survivors
                auto test_push = [&](int jj, bool valid, const float4 &k4, float iq, int ibt, float Dx, float Dy, float Dz, float thr, float ipi) {
                    bool pass = false, lo32 = false;
                    if (valid) {
                        const float ex = k4.x - Dx, ey = k4.y - Dy, ez = k4.z - Dz;   // Q + T - P
                        const float r2 = ex * ex + ey * ey + ez * ez;
                        const float isum = ipi + iq + iw2;
                        pass = (thr + k4.w + M) * isum > r2 && r2 <= rcut2f;
                        ++ncand;
                        if (pass) {                                               // max |P'| over the shell block (L819)
                            const int i = b0 + (ibt & 0xffff);
                            const float lbsum = __ldg(&K.q4[i].w) + k4.w +
                                                __ldg(p.lnPblk + (size_t)__ldg(K.shB + i) * ns + __ldg(kshB + jj));
                            pass = (lbsum - ln_tau + M) * isum > r2;
                            if constexpr (MIXED)
                                lo32 = pass && lbsum < p.ln_switch && __ldg(K.rng + i) + __ldg(K.rng + k0 + jj) < 60.f;
                        }
                    }
                    if constexpr (MIXED) {
                        const unsigned m32 = __ballot_sync(0xffffffffu, lo32), m64 = __ballot_sync(0xffffffffu, pass && !lo32);
                        if (lo32) queue32[(head32 + qn32 + __popc(m32 & ltmask)) & (KQ - 1)] = make_int2((ibt & 0xffff) | (jj << 16), ibt >> 16);
                        else if (pass) queue[(head + qn + __popc(m64 & ltmask)) & (KQ - 1)] = make_int2((ibt & 0xffff) | (jj << 16), ibt >> 16);
                        qn32 += __popc(m32);
                        qn += __popc(m64);
                    } else {
                        const unsigned m = __ballot_sync(0xffffffffu, pass);
                        if (pass) queue[(head + qn + __popc(m & ltmask)) & (KQ - 1)] = make_int2((ibt & 0xffff) | (jj << 16), ibt >> 16);
                        qn += __popc(m);
                    }
                };
                const int jj = jpos + lane;
                const bool va = jj < c_cnt;
                float4 ka = make_float4(0.f, 0.f, 0.f, 0.f);
                float iqa = 0.f;
                if (va) { ka = __ldg(kq4 + jj); iqa = __ldg(kipf + jj); }          // (Q - nu).xyz, lb; 1/q
                if (K_PAIR && !MIXED && c_cnt - jpos <= 32 && imask != 0 && qn + (c_cnt - jpos) + 32 <= KQ) {   // (the ring takes both passes)
                    // the last pass of this item runs together with the first pass of the next live item of the batch (both
                    // records are requested before either is tested: a pass is a chain of dependent loads and a ballot); water64 K
                    // 365 -> 359 ms, water343 3038 -> 3004 ms; the mixed-precision kernels (two rings) lose 1 % with it
                    const int src = __ffs(imask) - 1;
                    imask &= imask - 1;
                    const int d_ibt = __shfl_sync(0xffffffffu, it_ibt, src), d_cnt = __shfl_sync(0xffffffffu, it_cnt, src);
                    const float d_Dx = __shfl_sync(0xffffffffu, it_Dx, src), d_Dy = __shfl_sync(0xffffffffu, it_Dy, src),
                                d_Dz = __shfl_sync(0xffffffffu, it_Dz, src), d_thr = __shfl_sync(0xffffffffu, it_thr, src),
                                d_ipi = __shfl_sync(0xffffffffu, it_ipi, src);
                    const bool vb = lane < d_cnt;
                    float4 kb = make_float4(0.f, 0.f, 0.f, 0.f);
                    float iqb = 0.f;
                    if (vb) { kb = __ldg(kq4 + lane); iqb = __ldg(kipf + lane); }
                    test_push(jj, va, ka, iqa, c_ibt, c_Dx, c_Dy, c_Dz, c_thr, c_ipi);
                    test_push(lane, vb, kb, iqb, d_ibt, d_Dx, d_Dy, d_Dz, d_thr, d_ipi);
                    c_ibt = d_ibt; c_cnt = d_cnt; c_Dx = d_Dx; c_Dy = d_Dy; c_Dz = d_Dz; c_thr = d_thr; c_ipi = d_ipi;
                    jpos = 32;
                } else {
                    jpos += 32;
                    test_push(jj, va, ka, iqa, c_ibt, c_Dx, c_Dy, c_Dz, c_thr, c_ipi);
                }
                __syncwarp();
            }
            // a partly filled ring is evaluated only when this chunk's items are exhausted (its image indices
            // refer to the current list)
            bool act = false, w32 = false;
            int i = b0, j = k0, t = 0, consumed = 0;
            if constexpr (LOCKSTEP) {
                // The evaluators of the high classes are 10-60 thousand instructions of straight-line code, far more than
                // the instruction caches hold: the warps of a CTA enter the evaluator together and share the fetched lines.
                // A class of this kind holds only a few passes of quartets per warp, unevenly spread, so the four rings are
                // drained as ONE queue (ring of warp 0 first, then 1, ...): thread g of the CTA takes entry g of that queue,
                // whichever warp screened it -- every round runs with up to 128 busy lanes until all rings are empty.  (ncu
                // on (dd|dp) before this: 39 % of the stall samples at the round barrier, 18 active lanes per instruction.)
                if (lane == 0) { s_cnt[w] = qn; s_head[w] = head; s_done[w] = items_done ? 1 : 0; }
                __syncthreads();
                int cnt[NW], tot = 0, before = 0;
                bool alldone = true;
#pragma unroll
                for (int x = 0; x < NW; ++x) {
                    cnt[x] = s_cnt[x];
                    if (x < w) before += cnt[x];
                    tot += cnt[x];
                    alldone = alldone && s_done[x] != 0;
                }
                const int take = tot < NT ? tot : NT;
                const int g = threadIdx.x;
                act = g < take;
                if (act) {
                    int sw = 0, base = 0;
#pragma unroll
                    for (int x = 0; x < NW - 1; ++x)
                        if (sw == x && g >= base + cnt[x]) { base += cnt[x]; ++sw; }
                    const int2 e = qall[sw * KQ + ((s_head[sw] + (g - base)) & (KQ - 1))];
                    i = b0 + (e.x & 0xffff); j = k0 + (int)((unsigned)e.x >> 16); t = e.y;
                }
                consumed = take - before;                              // entries of this warp's ring taken by the round
                consumed = consumed < 0 ? 0 : (consumed > qn ? qn : consumed);
                __syncthreads();                                       // counters and entries are read: the owners may push again
                if (tot == 0) {
                    if (alldone) break;
                    continue;
                }
            } else {
                const bool w64 = qn >= 32 || (items_done && qn > 0);
                w32 = MIXED && (qn32 >= 32 || (items_done && qn32 > 0));
                if (!w64 && !w32) break;
                if (w64) {
                    consumed = qn < 32 ? qn : 32;
                    act = lane < consumed;
                    if (act) {
                        const int2 e = queue[(head + lane) & (KQ - 1)];
                        i = b0 + (e.x & 0xffff); j = k0 + (int)((unsigned)e.x >> 16); t = e.y;
                    }
                }
            }
            // ---- evaluation: one primitive quartet-image per lane, oldest survivors first ----
            if (act) {
                const double *__restrict__ bE = K.etab + __ldg(K.eoff + i);
                const double X = __ldg(K.Px + j) + sT[t] - __ldg(K.Px + i), Y = __ldg(K.Py + j) + sT[NIMG_K + t] - __ldg(K.Py + i),
                             Z = __ldg(K.Pz + j) + sT[2 * NIMG_K + t] - __ldg(K.Pz + i);
                const double pb = __ldg(K.p + i), q = __ldg(K.p + j);
                const double r2 = X * X + Y * Y + Z * Z;
                const double s = rsqrt(pb + q);
                const double alpha = pb * q * s * s;
                const double th = lat.omega * rsqrt(alpha + lat.omega2);
                const double alpha_w = alpha * th * th;
                const double pref = r2 <= p.rcut2 ? __ldg(K.coef + i) * __ldg(K.coef + j) * s : 0.0;
                const double *__restrict__ Pb = p.Pp + (size_t)__ldg(K.aoB + i) * p.ldP + __ldg(K.aoB + j);
                double Rm[L + 1];
                boys_merged<L, double>(p.boys, r2, alpha, alpha_w, th, pref, Rm);
                Ev::template run<32, double>(bE, K.etab + __ldg(K.eoff + j), Pb, p.ldP, Rm, X, Y, Z, Rs, Kacc);
            }
            head = (head + consumed) & (KQ - 1);
            qn -= consumed;
            nquart += consumed;
            __syncwarp();
            if constexpr (MIXED) if (w32) {
                const int take = qn32 < 32 ? qn32 : 32;
                int i = b0, j = k0, t = 0;
                if (lane < take) {
                    const int2 e = queue32[(head32 + lane) & (KQ - 1)];
                    i = b0 + (e.x & 0xffff); j = k0 + (int)((unsigned)e.x >> 16); t = e.y;
                }
                const long long eo = __ldg(K.eoff + i);
                const float *__restrict__ bE = K.etabf + eo;
                if (lane < take) {
                    const double Xd = __ldg(K.Px + j) + sT[t] - __ldg(K.Px + i), Yd = __ldg(K.Py + j) + sT[NIMG_K + t] - __ldg(K.Py + i),
                                 Zd = __ldg(K.Pz + j) + sT[2 * NIMG_K + t] - __ldg(K.Pz + i);
                    const float X = (float)Xd, Y = (float)Yd, Z = (float)Zd;
                    const float pb = (float)__ldg(K.p + i), q = (float)__ldg(K.p + j);
                    const float r2 = X * X + Y * Y + Z * Z;
                    const float s = rsqrtf(pb + q);
                    const float alpha = pb * q * s * s;
                    const float th = (float)lat.omega * rsqrtf(alpha + (float)lat.omega2);
                    const float alpha_w = alpha * th * th;
                    const float pref = Xd * Xd + Yd * Yd + Zd * Zd <= p.rcut2 ? (float)(__ldg(K.coef + i) * __ldg(K.coef + j)) * s : 0.f;
                    const float *__restrict__ Pb = p.Ppf + (size_t)__ldg(K.aoB + i) * p.ldP + __ldg(K.aoB + j);
                    float Rm[L + 1];
                    boys_merged<L, float>(p.boys, r2, alpha, alpha_w, th, pref, Rm);
                    float K32[NA * ND];
#pragma unroll
                    for (int c = 0; c < NA * ND; ++c) K32[c] = 0.f;
                    Ev::template run<32, float>(bE, K.etabf + __ldg(K.eoff + j), Pb, p.ldP, Rm, X, Y, Z,
                                                          reinterpret_cast<float *>(smem + (size_t)w * nherm(L) * 32) + lane, K32);
#pragma unroll
                    for (int c = 0; c < NA * ND; ++c) Kacc[c] += (double)K32[c];      // fp64 accumulation (reading C-22)
                }
                head32 = (head32 + take) & (KQ - 1);
                qn32 -= take;
                nquart32 += take;
                __syncwarp();
            }
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
        atomicAdd(p.counters + CNT_Q_K + cls, nquart + nquart32);
        if constexpr (MIXED) atomicAdd(p.counters + CNT_Q32_K + cls, nquart32);
    }
}

template <int LA, int LB, int LC, int LD, bool MIXED>
void launch_sr_k_class(const SRParams &p, const int2 *blocks, int nblocks, cudaStream_t st)
{
    constexpr size_t smem = k_smem_bytes<LA, LB, LC, LD, MIXED>();
    const int grid = p.shard_n > 1 ? (nblocks + p.shard_n - 1) / p.shard_n : nblocks;
    if (grid <= 0) return;
    sr_k_kernel<LA, LB, LC, LD, MIXED><<<grid, k_nthreads(LA + LB + LC + LD), smem, st>>>(p, blocks, nblocks);
}

// the attribute is per device: pbc_jk_create calls this for the handle's device
template <int LA, int LB, int LC, int LD, bool MIXED>
void set_sr_k_attr()
{
    cudaFuncSetAttribute(sr_k_kernel<LA, LB, LC, LD, MIXED>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)k_smem_bytes<LA, LB, LC, LD, MIXED>());
}

}  // namespace pbcjk
