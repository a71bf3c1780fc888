// C ABI of libpbc_jk (include/pbc_jk.h): host-side setup and the build
// orchestration (A4-A10).  All arithmetic of the path runs in the CUDA kernels of this directory.
#include "../../include/pbc_jk.h"
#include "pbcjk_common.h"
#include "pbcjk_1e.cuh"
#include "pbcjk_lr.cuh"
#include "pbcjk_sr.cuh"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <new>
#include <string>
#include <vector>

using namespace pbcjk;

namespace {

thread_local std::string g_create_error;

struct DevPool {
    std::vector<void *> ptrs;
    template <class T>
    cudaError_t alloc(T **p, size_t n)
    {
        *p = nullptr;
        cudaError_t e = cudaMalloc((void **)p, std::max<size_t>(n, 1) * sizeof(T));
        if (e == cudaSuccess) ptrs.push_back(*p);
        return e;
    }
    template <class T>
    cudaError_t upload(const T **p, const std::vector<T> &v)
    {
        T *d = nullptr;
        cudaError_t e = alloc(&d, v.size());
        if (e != cudaSuccess) return e;
        if (!v.empty()) e = cudaMemcpy(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
        *p = d;
        return e;
    }
    void free_all()
    {
        for (void *p : ptrs) cudaFree(p);
        ptrs.clear();
    }
};

struct HostPair {
    int shA, shB;
    double p, ip, P[3], PA[3], PB[3], coef, lb, b;
};

}  // namespace

struct pbc_jk {
    std::string err;
    DevPool pool;
    int N = 0, Np = 0, Npt = 0, nshell = 0, natom = 0, nG = 0;   // Np: N padded to 64 (strides, GEMM k and n); Npt: to the 128-row GEMM tiles
    int device = 0, nsm = 148;           // the CUDA device the handle lives on (current device at create)
    int parts = 7;
    pbc_cutoffs cut{};
    Lattice lat{};
    ShellInfo sh{};
    PairListK K{};
    PairListU U{};
    KetListJ KJ{};
    LRParams lr{};
    BoysTab boys{};
    const double *fcomp = nullptr;
    const int *shell_of_ao = nullptr;
    // J bra index lists per Hermite order, K block lists per (la, ld)
    const int *jbra[5] = {};
    int njbra[5] = {};
    const int2 *kblk[3][3] = {};
    int nkblk[3][3] = {};
    // workspaces
    double *Pp = nullptr, *lnPmax = nullptr, *Dt = nullptr, *Jt = nullptr, *Jsr = nullptr, *Jlr = nullptr;
    float *Ppf = nullptr, *lnPblk = nullptr, *lnProw = nullptr, *kjP = nullptr;   // fp32 P' (mixed), per-block ln max|P'|
    bool mixed = false;                  // precision = 1: fp32 K quartets below the switch (PAPER 3.5)
    double mixed_switch = 1e-5;
    int shard_rank = 0, shard_n = 1;     // multi-GPU share of every build (pbc_jk_set_shard)
    double *Ksr = nullptr, *Klr = nullptr, *Astack = nullptr, *Zstack = nullptr, *rho = nullptr;
    double *hostP = nullptr, *hostJ = nullptr, *hostK = nullptr;     // device staging of build_host
    double *noalloc_scratch = nullptr;   // device address of the static scratch of pbc_jk_overlap_noalloc (resolved at create)
    cudaError_t noalloc_err = cudaSuccess;
    double *LT = nullptr, *chol_d = nullptr, *chol_s = nullptr;      // factor P' = L L^T of the K^LR contraction
    int *chol_dyn = nullptr;
    unsigned long long *maxbits = nullptr, *counters = nullptr;
    int nb = 1, nsplit = 1, Smax = 16;
    int cur_S = 0;                       // slot count the A' stack is currently laid out (and zero-filled) for
    bool has_l[LMAX + 1] = {};
    size_t ld = 0;
    double c0 = 0.0;             // pi/(Omega w^2)
    cudaEvent_t ev[6] = {};
    // per-class events of the real-space launches (profile mode): [cls][start, stop]
    cudaEvent_t evJ[NCLS_J][2] = {}, evK[NCLS_K][2] = {};
    bool ranJ[NCLS_J] = {}, ranK[NCLS_K] = {};
    std::vector<cudaEvent_t> evG;        // profile mode: event pairs around the two K^LR GEMMs of every G batch (+ SELF)
    int n_evG = 0;                       // pairs recorded by the last build
    bool profile = false;
    bool profiled_last = false;          // profile mode was on during the last build (the class events are recorded)
    bool debug_sync = false;             // env PBC_JK_DEBUG_SYNC=1: synchronise after every real-space class launch and name
                                         // the class in the error text (bring-up aid; breaks the no-host-sync contract)
    int64_t n_launches = 0;
    cudaStream_t last_stream = nullptr;
    bool built = false;
    int64_t n_prim_pairs = 0, n_sp_images = 0;
    double create_seconds = 0.0;
    std::vector<double> S_host;
    std::vector<double> atom_xyz;        // atom positions folded into the home cell (host copy; one-electron terms)
    double omega = 0.0;
};

namespace {

double det3(const double *c)
{
    return c[0] * (c[4] * c[8] - c[5] * c[7]) - c[1] * (c[3] * c[8] - c[5] * c[6]) + c[2] * (c[3] * c[7] - c[4] * c[6]);
}

// inverse of the 3x3 cell matrix (rows a_i): inv[j][k]; fractional f_k = sum_j r_j inv[j][k]
void inverse3(const double *c, double *inv)
{
    const double d = det3(c);
    inv[0] = (c[4] * c[8] - c[5] * c[7]) / d; inv[1] = (c[2] * c[7] - c[1] * c[8]) / d; inv[2] = (c[1] * c[5] - c[2] * c[4]) / d;
    inv[3] = (c[5] * c[6] - c[3] * c[8]) / d; inv[4] = (c[0] * c[8] - c[2] * c[6]) / d; inv[5] = (c[2] * c[3] - c[0] * c[5]) / d;
    inv[6] = (c[3] * c[7] - c[4] * c[6]) / d; inv[7] = (c[1] * c[6] - c[0] * c[7]) / d; inv[8] = (c[0] * c[4] - c[1] * c[3]) / d;
}

double dfact2(int n)   // (2n-1)!!
{
    double r = 1.0;
    for (int k = 2 * n - 1; k > 1; k -= 2) r *= k;
    return r;
}

// eq 6 (L72, reading C-1) for the axis-aligned component x^l: (2a/pi)^{3/4} (4a)^{l/2} / sqrt((2l-1)!!)
double norm_axis(double a, int l)
{
    return std::pow(2.0 * a / M_PI, 0.75) * std::pow(4.0 * a, 0.5 * l) / std::sqrt(dfact2(l));
}

// F_m(x), m = 0..mmax: Kummer series for the top order, downward recursion (table generator)
void boys_host(int mmax, double x, double *F)
{
    const double ex = std::exp(-x);
    double term = 1.0 / (2.0 * mmax + 1.0), sum = term;
    for (int k = 1; k < 2000; ++k) {
        term *= 2.0 * x / (2.0 * mmax + 2.0 * k + 1.0);
        sum += term;
        if (term < 1e-18 * sum) break;
    }
    F[mmax] = ex * sum;
    for (int m = mmax; m > 0; --m) F[m - 1] = (2.0 * x * F[m] + ex) / (2.0 * m - 1.0);
}

int fail(pbc_jk *h, int code, const std::string &msg)
{
    if (h) h->err = msg;
    else g_create_error = msg;
    return code;
}

#define CK(call)                                                                              \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess) {                                                              \
            h->err = std::string(#call) + ": " + cudaGetErrorString(e_);                      \
            return e_ == cudaErrorMemoryAllocation ? PBC_JK_ERR_NOMEM : PBC_JK_ERR_CUDA;      \
        }                                                                                     \
    } while (0)

// Lattice translations n with |n.a - c| < r: bounding box from the reciprocal rows, sphere filter
// (eq 99-103).
template <class F>
void for_images_host(const Lattice &lat, const double c[3], double r, F &&f)
{
    int lo[3], hi[3];
    for (int k = 0; k < 3; ++k) {
        const double fk = lat.binv[3 * k] * c[0] + lat.binv[3 * k + 1] * c[1] + lat.binv[3 * k + 2] * c[2];
        lo[k] = (int)std::ceil(fk - r * lat.bnorm[k]);
        hi[k] = (int)std::floor(fk + r * lat.bnorm[k]);
    }
    for (int n0 = lo[0]; n0 <= hi[0]; ++n0)
        for (int n1 = lo[1]; n1 <= hi[1]; ++n1)
            for (int n2 = lo[2]; n2 <= hi[2]; ++n2) {
                const double T[3] = {n0 * lat.a[0] + n1 * lat.a[3] + n2 * lat.a[6], n0 * lat.a[1] + n1 * lat.a[4] + n2 * lat.a[7],
                                     n0 * lat.a[2] + n1 * lat.a[5] + n2 * lat.a[8]};
                const double d0 = T[0] - c[0], d1 = T[1] - c[1], d2 = T[2] - c[2];
                if (d0 * d0 + d1 * d1 + d2 * d2 < r * r) f(T);
            }
}

void destroy_events(pbc_jk *h)
{
    for (auto &e : h->ev)
        if (e) cudaEventDestroy(e);
    for (auto &e : h->evG)
        if (e) cudaEventDestroy(e);
    for (auto &e : h->evJ)
        for (auto &x : e)
            if (x) cudaEventDestroy(x);
    for (auto &e : h->evK)
        for (auto &x : e)
            if (x) cudaEventDestroy(x);
}

int setup(pbc_jk *h, const pbc_cell *cell, const pbc_atoms *atoms, const pbc_shells *shells, double omega)
{
    const pbc_cutoffs &cut = h->cut;
    // ---- A1: lattice ----
    Lattice &lat = h->lat;
    for (int i = 0; i < 9; ++i) lat.a[i] = cell->a[i];
    const double vol = det3(lat.a);
    if (!(std::fabs(vol) > 1e-12)) return fail(h, PBC_JK_ERR_INVALID_ARG, "singular cell");
    double inv[9];
    inverse3(lat.a, inv);
    for (int k = 0; k < 3; ++k) {
        for (int j = 0; j < 3; ++j) lat.binv[3 * k + j] = inv[3 * j + k];
        lat.bnorm[k] = std::sqrt(lat.binv[3 * k] * lat.binv[3 * k] + lat.binv[3 * k + 1] * lat.binv[3 * k + 1] +
                                 lat.binv[3 * k + 2] * lat.binv[3 * k + 2]);
    }
    lat.omega = omega; lat.omega2 = omega * omega; lat.iomega2 = 1.0 / (omega * omega);
    lat.volume = std::fabs(vol);
    h->c0 = M_PI / (lat.volume * omega * omega);

    // ---- basis bookkeeping ----
    const int ns = shells->nshell, natom = atoms->natom;
    h->nshell = ns; h->natom = natom; h->omega = omega;
    // every centre may be given in any lattice image (L781): fold all of them into the home cell, so that the
    // lattice indices the real-space scans enumerate stay inside the packed 10-bit range checked below
    std::vector<double> axyz(3 * (size_t)natom);
    for (int a = 0; a < natom; ++a) {
        const double *r = atoms->xyz + 3 * a;
        double f[3];
        for (int k = 0; k < 3; ++k) f[k] = std::floor(lat.binv[3 * k] * r[0] + lat.binv[3 * k + 1] * r[1] + lat.binv[3 * k + 2] * r[2]);
        for (int x = 0; x < 3; ++x) axyz[3 * a + x] = r[x] - (f[0] * lat.a[x] + f[1] * lat.a[3 + x] + f[2] * lat.a[6 + x]);
    }
    h->atom_xyz = axyz;
    std::vector<int> sh_l(ns), sh_ao(ns), sh_atom(ns);
    std::vector<double> scx(ns), scy(ns), scz(ns);
    int nbf = 0, nprim_tot = 0;
    double amin_all = std::numeric_limits<double>::max();
    for (int s = 0; s < ns; ++s) {
        const int l = shells->l[s];
        if (l < 0 || l > LMAX) return fail(h, PBC_JK_ERR_INVALID_ARG, "shell angular momentum outside 0..2");
        if (shells->nprim[s] < 1) return fail(h, PBC_JK_ERR_INVALID_ARG, "shell without primitives");
        if (shells->atom[s] < 0 || shells->atom[s] >= natom) return fail(h, PBC_JK_ERR_INVALID_ARG, "shell atom index out of range");
        if (shells->prim_off[s] < 0) return fail(h, PBC_JK_ERR_INVALID_ARG, "negative prim_off");
        sh_l[s] = l; sh_ao[s] = nbf; sh_atom[s] = shells->atom[s];
        h->has_l[l] = true;
        nbf += ncart(l);
        scx[s] = axyz[3 * sh_atom[s]]; scy[s] = axyz[3 * sh_atom[s] + 1]; scz[s] = axyz[3 * sh_atom[s] + 2];
        for (int k = 0; k < shells->nprim[s]; ++k) {
            const double a = shells->exps[shells->prim_off[s] + k];
            if (!(a > 0.0)) return fail(h, PBC_JK_ERR_INVALID_ARG, "non-positive exponent");
            amin_all = std::min(amin_all, a);
        }
        nprim_tot = std::max(nprim_tot, shells->prim_off[s] + shells->nprim[s]);
    }
    h->N = nbf;
    h->Np = ((nbf + 63) / 64) * 64;
    h->Npt = ((nbf + 127) / 128) * 128;
    std::vector<double> cn(nprim_tot, 0.0);
    for (int s = 0; s < ns; ++s)
        for (int k = 0; k < shells->nprim[s]; ++k) {
            const int i = shells->prim_off[s] + k;
            cn[i] = shells->coefs[i] * norm_axis(shells->exps[i], sh_l[s]);
        }
    std::vector<double> fcomp(nbf, 1.0);
    std::vector<int> shell_of_ao(nbf, 0);
    for (int s = 0; s < ns; ++s)
        for (int k = 0; k < ncart(sh_l[s]); ++k) {
            shell_of_ao[sh_ao[s] + k] = s;
            if (sh_l[s] == 2 && (k == 1 || k == 2 || k == 4)) fcomp[sh_ao[s] + k] = std::sqrt(3.0);
        }

    // ---- A2: ordered primitive pair-images with bounds ----
    const double d_pair = cut.d_pair > 0 ? cut.d_pair : 1e-14;
    const double fmaxl[3] = {1.0, 1.0, std::sqrt(3.0)};
    std::vector<std::vector<HostPair>> per_shell(ns);
    std::vector<int64_t> sp_images(ns, 0);
    bool omp_failed = false;             // no exception may leave an OpenMP region: caught inside, reported after
    bool range_failed = false;
#pragma omp parallel for schedule(dynamic, 4)
    for (int A = 0; A < ns; ++A) {
      try {
        std::vector<HostPair> &out = per_shell[A];
        const double RA[3] = {scx[A], scy[A], scz[A]};
        const int la = sh_l[A];
        for (int B = 0; B < ns; ++B) {
            const int lb = sh_l[B];
            const double RB[3] = {scx[B], scy[B], scz[B]};
            double d[3] = {RA[0] - RB[0], RA[1] - RB[1], RA[2] - RB[2]};
            // minimum image of the offset (eq 102-103)
            double nr[3];
            for (int k = 0; k < 3; ++k)
                nr[k] = std::nearbyint(lat.binv[3 * k] * d[0] + lat.binv[3 * k + 1] * d[1] + lat.binv[3 * k + 2] * d[2]);
            double RBm[3];
            for (int x = 0; x < 3; ++x) RBm[x] = RB[x] + nr[0] * lat.a[x] + nr[1] * lat.a[3 + x] + nr[2] * lat.a[6 + x];
            const double d0[3] = {RA[0] - RBm[0], RA[1] - RBm[1], RA[2] - RBm[2]};
            // per primitive pair: prefactor and enumeration radius
            const int na = shells->nprim[A], nb = shells->nprim[B];
            struct PP { double a, b, p, mu, cc, isq, rad, csigned; };
            std::vector<PP> pp;
            double rmax = 0.0;
            for (int ia = 0; ia < na; ++ia)
                for (int ib = 0; ib < nb; ++ib) {
                    PP q;
                    q.a = shells->exps[shells->prim_off[A] + ia];
                    q.b = shells->exps[shells->prim_off[B] + ib];
                    q.p = q.a + q.b; q.mu = q.a * q.b / q.p; q.isq = 1.0 / std::sqrt(q.p);
                    const double c = cn[shells->prim_off[A] + ia] * cn[shells->prim_off[B] + ib];
                    // bound prefactor: |c| f_a f_b (pi/p)^{3/2} sqrt(2/sqrt(pi)) p^{1/4}   (eq 60 up to 2^{1/4})
                    q.cc = std::fabs(c) * fmaxl[la] * fmaxl[lb] * std::pow(M_PI / q.p, 1.5) * std::sqrt(2.0 / std::sqrt(M_PI)) *
                           std::pow(q.p, 0.25);
                    double R = 40.0;
                    bool any = true;
                    for (int it = 0; it < 4; ++it) {
                        const double ang = std::pow(q.b / q.p * R + q.isq, la) * std::pow(q.a / q.p * R + q.isq, lb);
                        const double v = q.cc * ang / d_pair;
                        if (v <= 1.0) { any = false; break; }
                        R = std::sqrt(std::log(v) / q.mu);
                    }
                    q.rad = any ? R * 1.0000001 + 1e-9 : -1.0;
                    if (cut.r_cut > 0 && q.rad > cut.r_cut) q.rad = cut.r_cut;
                    rmax = std::max(rmax, q.rad);
                    // keep the signed coefficient next to the bound
                    q.csigned = c;
                    pp.push_back(q);
                }
            if (rmax <= 0.0) continue;
            // a cell far too small for this pair's reach would enumerate millions of images (and later overflow the packed
            // lattice indices of the scans): refuse before enumerating
            const double rr = rmax + std::sqrt(d0[0] * d0[0] + d0[1] * d0[1] + d0[2] * d0[2]);
            if (rr * std::max(lat.bnorm[0], std::max(lat.bnorm[1], lat.bnorm[2])) > 400.0 ||
                (2.0 * rmax * lat.bnorm[0] + 1.0) * (2.0 * rmax * lat.bnorm[1] + 1.0) * (2.0 * rmax * lat.bnorm[2] + 1.0) > 2.0e6) {
#pragma omp atomic write
                range_failed = true;
                continue;
            }
            for_images_host(lat, d0, rmax, [&](const double *T) {
                const double Bt[3] = {RBm[0] + T[0], RBm[1] + T[1], RBm[2] + T[2]};
                const double AB[3] = {RA[0] - Bt[0], RA[1] - Bt[1], RA[2] - Bt[2]};
                const double R2 = AB[0] * AB[0] + AB[1] * AB[1] + AB[2] * AB[2];
                const double R = std::sqrt(R2);
                bool any = false;
                for (const PP &q : pp) {
                    if (q.rad <= 0.0 || R >= q.rad) continue;
                    const double ang = std::pow(q.b / q.p * R + q.isq, la) * std::pow(q.a / q.p * R + q.isq, lb);
                    const double ex = std::exp(-q.mu * R2);
                    const double bound = q.cc * ang * ex;
                    if (!(bound > d_pair)) continue;
                    HostPair e;
                    e.shA = A; e.shB = B; e.p = q.p; e.ip = 1.0 / q.p; e.b = q.b;
                    for (int x = 0; x < 3; ++x) {
                        e.P[x] = (q.a * RA[x] + q.b * Bt[x]) / q.p;
                        e.PA[x] = e.P[x] - RA[x];
                        e.PB[x] = e.P[x] - Bt[x];
                    }
                    e.coef = q.csigned * ex * std::sqrt(2.0) * std::pow(M_PI, 1.25) / q.p;
                    e.lb = std::log(bound);
                    out.push_back(e);
                    any = true;
                }
                if (any) ++sp_images[A];
            });
        }
      } catch (...) {
#pragma omp atomic write
        omp_failed = true;
      }
    }
    if (omp_failed) return fail(h, PBC_JK_ERR_NOMEM, "host allocation failed while building the pair list");
    if (range_failed)
        return fail(h, PBC_JK_ERR_UNSUPPORTED, "lattice image range of the pair list exceeds the packed format "
                                               "(cell far too small for these exponents)");
    (void)amin_all;
    // K order: (A, l_B, bound descending)
    std::vector<HostPair> kp;
    {
        size_t tot = 0;
        for (auto &v : per_shell) tot += v.size();
        kp.reserve(tot);
        for (int A = 0; A < ns; ++A) {
            auto &v = per_shell[A];
            std::stable_sort(v.begin(), v.end(), [&](const HostPair &x, const HostPair &y) {
                const int lx = sh_l[x.shB], ly = sh_l[y.shB];
                if (lx != ly) return lx < ly;
                return x.lb > y.lb;
            });
            kp.insert(kp.end(), v.begin(), v.end());
            std::vector<HostPair>().swap(v);
        }
    }
    h->n_prim_pairs = (int64_t)kp.size();
    for (int A = 0; A < ns; ++A) h->n_sp_images += sp_images[A];
    if (kp.size() > (size_t)std::numeric_limits<int>::max() / 2) return fail(h, PBC_JK_ERR_NOMEM, "too many primitive pair-images");

    auto soa = [&](const std::vector<HostPair> &v, int field, int x) {
        std::vector<double> o(v.size());
        for (size_t i = 0; i < v.size(); ++i) {
            const HostPair &e = v[i];
            switch (field) {
            case 0: o[i] = e.P[x]; break;
            case 1: o[i] = e.p; break;
            case 2: o[i] = e.ip; break;
            case 3: o[i] = e.coef; break;
            case 4: o[i] = e.lb; break;
            case 5: o[i] = e.PA[x]; break;
            default: o[i] = e.PB[x]; break;
            }
        }
        return o;
    };
    DevPool &pool = h->pool;
    // ---- upload K lists ----
    {
        PairListK &K = h->K;
        K.n = (int)kp.size();
        CK(pool.upload(&K.Px, soa(kp, 0, 0))); CK(pool.upload(&K.Py, soa(kp, 0, 1))); CK(pool.upload(&K.Pz, soa(kp, 0, 2)));
        CK(pool.upload(&K.p, soa(kp, 1, 0))); CK(pool.upload(&K.ip, soa(kp, 2, 0)));
        CK(pool.upload(&K.coef, soa(kp, 3, 0))); CK(pool.upload(&K.lb, soa(kp, 4, 0)));
        CK(pool.upload(&K.PAx, soa(kp, 5, 0))); CK(pool.upload(&K.PAy, soa(kp, 5, 1))); CK(pool.upload(&K.PAz, soa(kp, 5, 2)));
        CK(pool.upload(&K.PBx, soa(kp, 6, 0))); CK(pool.upload(&K.PBy, soa(kp, 6, 1))); CK(pool.upload(&K.PBz, soa(kp, 6, 2)));
        std::vector<int> aoB(kp.size()), shB(kp.size()), off(ns * 3 + 1, 0);
        std::vector<double> ext(ns * 3, 0.0), ipmax(ns * 3, 0.0);
        std::vector<float4> q4(kp.size());
        std::vector<float> ipf(kp.size()), rng(kp.size());
        for (size_t i = 0; i < kp.size(); ++i) {
            aoB[i] = sh_ao[kp[i].shB];
            shB[i] = kp[i].shB;
            // fp32 screen record, rounded so that it never undercuts the fp64 values (bound and 1/p rounded up)
            q4[i] = make_float4((float)kp[i].PA[0], (float)kp[i].PA[1], (float)kp[i].PA[2],
                                std::nextafter((float)kp[i].lb, std::numeric_limits<float>::infinity()));
            ipf[i] = std::nextafter((float)kp[i].ip, std::numeric_limits<float>::infinity());
            rng[i] = (float)(std::log(std::max(std::fabs(kp[i].coef), 1e-300)) +
                             (sh_l[kp[i].shA] + sh_l[kp[i].shB]) * std::log(2.0 * kp[i].p));
            const int g = kp[i].shA * 3 + sh_l[kp[i].shB];
            off[g + 1]++;
            const double e = std::sqrt(kp[i].PA[0] * kp[i].PA[0] + kp[i].PA[1] * kp[i].PA[1] + kp[i].PA[2] * kp[i].PA[2]);
            ext[g] = std::max(ext[g], e);
            ipmax[g] = std::max(ipmax[g], kp[i].ip);
        }
        for (int g = 0; g < ns * 3; ++g) off[g + 1] += off[g];
        for (int g = 0; g < ns * 3; ++g)
            if (off[g + 1] - off[g] > 65535)
                return fail(h, PBC_JK_ERR_UNSUPPORTED, "a (shell, l) group holds more than 65535 primitive pair-images "
                                                       "(the survivor rings pack bra and ket indices into 16 bits each)");
        // The scans pack a lattice index into 10 bits per direction (pack_img, |n| <= 511).  Largest index they can
        // reach: (reach of the screen for the strongest bra and ket at max|P'| = e^{LN_PMAX_CAP}, plus the largest
        // offset between a bra centre and a ket group centre) * |b_k|/2pi.  A density above the cap is caught on
        // the device (lnpmax_kernel sets the overflow flag; the build then reports PBC_JK_ERR_UNSUPPORTED).
        {
            double lbmax = -1e300, ipm = 0.0, extm = 0.0;
            for (size_t i = 0; i < kp.size(); ++i) lbmax = std::max(lbmax, kp[i].lb);
            for (int g = 0; g < ns * 3; ++g) { ipm = std::max(ipm, ipmax[g]); extm = std::max(extm, ext[g]); }
            const double ln_tau = std::log(cut.d_schwarz > 0 ? cut.d_schwarz : 1e-13);
            const double budget = std::max(0.0, 2.0 * lbmax + LN_PMAX_CAP - ln_tau);
            const double reach = std::sqrt(budget * (2.0 * ipm + lat.iomega2)) + extm;
            double diag = 0.0;
            for (int sx = -1; sx <= 1; sx += 2)
                for (int sy = -1; sy <= 1; sy += 2) {
                    double v[3];
                    for (int x = 0; x < 3; ++x) v[x] = lat.a[x] + sx * lat.a[3 + x] + sy * lat.a[6 + x];
                    diag = std::max(diag, std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
                }
            const double bn = std::max(lat.bnorm[0], std::max(lat.bnorm[1], lat.bnorm[2]));
            if (!kp.empty() && (reach + diag + 2.0 * extm) * bn + 2.0 > 511.0)
                return fail(h, PBC_JK_ERR_UNSUPPORTED, "lattice image range of the real-space sums exceeds the packed format "
                                                       "(cell far too small for these exponents / omega)");
        }
        // E-product table rows (eq 16-20), filled on the device (etab_kernel)
        {
            auto eterms = [](int l1, int l2) {
                int n = 0;
                for (int a = 0; a < ncart(l1); ++a)
                    for (int b = 0; b < ncart(l2); ++b)
                        n += (cart_x(l1, a) + cart_x(l2, b) + 1) * (cart_y(l1, a) + cart_y(l2, b) + 1) * (cart_z(l1, a) + cart_z(l2, b) + 1);
                return n;
            };
            std::vector<long long> eoff(kp.size());
            std::vector<int> lA(kp.size()), lB(kp.size());
            long long tot = 0;
            for (size_t i = 0; i < kp.size(); ++i) {
                lA[i] = sh_l[kp[i].shA]; lB[i] = sh_l[kp[i].shB];
                eoff[i] = tot;
                tot += eterms(lA[i], lB[i]);
            }
            double *etab = nullptr;
            const int *dlA = nullptr, *dlB = nullptr;
            CK(pool.upload(&K.eoff, eoff)); CK(pool.alloc(&etab, (size_t)tot));
            CK(pool.upload(&dlA, lA)); CK(pool.upload(&dlB, lB));
            K.etab = etab;
            launch_etab(K, dlA, dlB, etab, 0);
            K.etabf = nullptr;
            if (h->mixed) {                       // fp32 copy for the float evaluators (PAPER 3.5)
                float *etabf = nullptr;
                CK(pool.alloc(&etabf, (size_t)tot));
                launch_to_float(etab, etabf, (size_t)tot, 0);
                K.etabf = etabf;
            }
            CK(cudaGetLastError());
        }
        CK(pool.upload(&K.aoB, aoB)); CK(pool.upload(&K.shB, shB)); CK(pool.upload(&K.off, off));
        CK(pool.upload(&K.q4, q4)); CK(pool.upload(&K.ipf, ipf)); CK(pool.upload(&K.rng, rng));
        CK(pool.upload(&K.ext, ext)); CK(pool.upload(&K.ipmax, ipmax));
        // K block lists per (la >= ld), heaviest first
        std::vector<int64_t> cnt(ns, 0);
        for (int s = 0; s < ns; ++s) cnt[s] = off[s * 3 + 3] - off[s * 3];
        for (int la = 0; la <= LMAX; ++la)
            for (int ld = 0; ld <= la; ++ld) {
                std::vector<std::pair<int64_t, int2>> blk;
                for (int mu = 0; mu < ns; ++mu) {
                    if (sh_l[mu] != la || cnt[mu] == 0) continue;
                    for (int nu = 0; nu < ns; ++nu) {
                        if (sh_l[nu] != ld || cnt[nu] == 0) continue;
                        if (la == ld && nu > mu) continue;
                        blk.push_back({cnt[mu] * cnt[nu], make_int2(mu, nu)});
                    }
                }
                std::stable_sort(blk.begin(), blk.end(), [](const auto &x, const auto &y) { return x.first > y.first; });
                std::vector<int2> b2(blk.size());
                for (size_t i = 0; i < blk.size(); ++i) b2[i] = blk[i].second;
                CK(pool.upload(&h->kblk[la][ld], b2));
                h->nkblk[la][ld] = (int)b2.size();
            }
    }
    // ---- U list (shell A >= shell B), contiguous per shell pair ----
    std::vector<HostPair> up;
    std::vector<int> u_sp, sp_off, sp_shA, sp_shB;
    {
        std::vector<size_t> idx;
        for (size_t i = 0; i < kp.size(); ++i)
            if (kp[i].shA >= kp[i].shB) idx.push_back(i);
        std::stable_sort(idx.begin(), idx.end(), [&](size_t x, size_t y) {
            if (kp[x].shA != kp[y].shA) return kp[x].shA < kp[y].shA;
            return kp[x].shB < kp[y].shB;
        });
        up.reserve(idx.size());
        for (size_t i : idx) up.push_back(kp[i]);
        u_sp.resize(up.size());
        for (size_t i = 0; i < up.size(); ++i) {
            if (i == 0 || up[i].shA != up[i - 1].shA || up[i].shB != up[i - 1].shB) {
                sp_off.push_back((int)i);
                sp_shA.push_back(up[i].shA);
                sp_shB.push_back(up[i].shB);
            }
            u_sp[i] = (int)sp_shA.size() - 1;
        }
        sp_off.push_back((int)up.size());
        PairListU &U = h->U;
        U.n = (int)up.size(); U.nsp = (int)sp_shA.size();
        CK(pool.upload(&U.Px, soa(up, 0, 0))); CK(pool.upload(&U.Py, soa(up, 0, 1))); CK(pool.upload(&U.Pz, soa(up, 0, 2)));
        CK(pool.upload(&U.p, soa(up, 1, 0))); CK(pool.upload(&U.ip, soa(up, 2, 0)));
        CK(pool.upload(&U.coef, soa(up, 3, 0))); CK(pool.upload(&U.lb, soa(up, 4, 0)));
        CK(pool.upload(&U.PAx, soa(up, 5, 0))); CK(pool.upload(&U.PAy, soa(up, 5, 1))); CK(pool.upload(&U.PAz, soa(up, 5, 2)));
        CK(pool.upload(&U.PBx, soa(up, 6, 0))); CK(pool.upload(&U.PBy, soa(up, 6, 1))); CK(pool.upload(&U.PBz, soa(up, 6, 2)));
        {
            std::vector<double> bexp(up.size());
            for (size_t i = 0; i < up.size(); ++i) bexp[i] = up[i].b;
            CK(pool.upload(&U.bexp, bexp));
        }
        CK(pool.upload(&U.sp, u_sp)); CK(pool.upload(&U.sp_off, sp_off));
        CK(pool.upload(&U.sp_shA, sp_shA)); CK(pool.upload(&U.sp_shB, sp_shB));
        // shell pairs by class (l_A, l_B): one rho_mn(G) kernel instantiation per class
        for (int c = 0; c < 9; ++c) {
            std::vector<int> lst;
            for (size_t q = 0; q < sp_shA.size(); ++q)
                if (sh_l[sp_shA[q]] * 3 + sh_l[sp_shB[q]] == c) lst.push_back((int)q);
            CK(pool.upload(&h->lr.sp_cls[c], lst));
            h->lr.n_sp_cls[c] = (int)lst.size();
        }
        // J bra lists per Hermite order, heaviest first
        for (int LB = 0; LB <= 4; ++LB) {
            std::vector<int> b;
            for (size_t i = 0; i < up.size(); ++i)
                if (sh_l[up[i].shA] + sh_l[up[i].shB] == LB) b.push_back((int)i);
            std::stable_sort(b.begin(), b.end(), [&](int x, int y) { return up[x].lb > up[y].lb; });
            CK(pool.upload(&h->jbra[LB], b));
            h->njbra[LB] = (int)b.size();
        }
    }
    // ---- J kets: U regrouped by (atom of shell A, Hermite order, bound descending) ----
    {
        std::vector<int> idx(up.size());
        for (size_t i = 0; i < up.size(); ++i) idx[i] = (int)i;
        const double ln2 = std::log(2.0);
        auto klb = [&](int i) { return up[i].lb + (up[i].shA != up[i].shB ? ln2 : 0.0); };
        std::stable_sort(idx.begin(), idx.end(), [&](int x, int y) {
            const int gx = sh_atom[up[x].shA] * 5 + sh_l[up[x].shA] + sh_l[up[x].shB];
            const int gy = sh_atom[up[y].shA] * 5 + sh_l[up[y].shA] + sh_l[up[y].shB];
            if (gx != gy) return gx < gy;
            return klb(x) > klb(y);
        });
        const size_t n = idx.size();
        std::vector<double> Qx(n), Qy(n), Qz(n), q(n), iq(n), coef(n), lb(n);
        std::vector<int> off(natom * 5 + 1, 0), spA(n), spB(n);
        std::vector<float4> jq4(n);
        std::vector<float> iqf(n);
        std::vector<double> ext(natom * 5, 0.0), iqmax(natom * 5, 0.0), gx(natom), gy(natom), gz(natom);
        for (int a = 0; a < natom; ++a) { gx[a] = axyz[3 * a]; gy[a] = axyz[3 * a + 1]; gz[a] = axyz[3 * a + 2]; }
        for (size_t j = 0; j < n; ++j) {
            const HostPair &e = up[idx[j]];
            Qx[j] = e.P[0]; Qy[j] = e.P[1]; Qz[j] = e.P[2]; q[j] = e.p; iq[j] = e.ip; coef[j] = e.coef; lb[j] = klb(idx[j]);
            spA[j] = e.shA; spB[j] = e.shB;
            jq4[j] = make_float4((float)e.PA[0], (float)e.PA[1], (float)e.PA[2],        // Q - atom of the home shell
                                 std::nextafter((float)lb[j], std::numeric_limits<float>::infinity()));
            iqf[j] = std::nextafter((float)e.ip, std::numeric_limits<float>::infinity());
            const int g = sh_atom[e.shA] * 5 + sh_l[e.shA] + sh_l[e.shB];
            off[g + 1]++;
            ext[g] = std::max(ext[g], std::sqrt(e.PA[0] * e.PA[0] + e.PA[1] * e.PA[1] + e.PA[2] * e.PA[2]));
            iqmax[g] = std::max(iqmax[g], e.ip);
        }
        for (int g = 0; g < natom * 5; ++g) off[g + 1] += off[g];
        KetListJ &KJ = h->KJ;
        if (n >= ((size_t)1 << J_KET_BITS))
            return fail(h, PBC_JK_ERR_UNSUPPORTED, "more than 2^26 primitive pair-images in the J-engine ket list (packed ring entries)");
        KJ.n = (int)n; KJ.ngroup = natom; KJ.dstride = (int64_t)std::max<size_t>(n, 1);
        CK(pool.upload(&KJ.Qx, Qx)); CK(pool.upload(&KJ.Qy, Qy)); CK(pool.upload(&KJ.Qz, Qz));
        CK(pool.upload(&KJ.q, q)); CK(pool.upload(&KJ.iq, iq)); CK(pool.upload(&KJ.coef, coef)); CK(pool.upload(&KJ.lb, lb));
        CK(pool.upload(&KJ.uidx, idx)); CK(pool.upload(&KJ.off, off));
        CK(pool.upload(&KJ.ext, ext)); CK(pool.upload(&KJ.iqmax, iqmax));
        CK(pool.upload(&KJ.gx, gx)); CK(pool.upload(&KJ.gy, gy)); CK(pool.upload(&KJ.gz, gz));
        CK(pool.upload(&KJ.q4, jq4)); CK(pool.upload(&KJ.iqf, iqf)); CK(pool.upload(&KJ.spA, spA)); CK(pool.upload(&KJ.spB, spB));
        // group records of the level-A screen; reference point g0 = cell centre (the atoms were folded into the cell)
        std::vector<int2> goff(natom * 5);
        std::vector<float4> grec(natom * 5), g4(natom);
        for (int x = 0; x < 3; ++x) KJ.g0[x] = 0.5 * (lat.a[x] + lat.a[3 + x] + lat.a[6 + x]);
        KJ.rc = 0.0;
        for (int a = 0; a < natom; ++a) {
            const double d[3] = {gx[a] - KJ.g0[0], gy[a] - KJ.g0[1], gz[a] - KJ.g0[2]};
            KJ.rc = std::max(KJ.rc, std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
            g4[a] = make_float4((float)d[0], (float)d[1], (float)d[2], 0.f);
        }
        for (int k = 0; k < 5; ++k) { KJ.lbmax[k] = -1e30f; KJ.iqmaxall[k] = 0.f; KJ.extmax[k] = 0.f; }
        for (int g = 0; g < natom * 5; ++g) {
            const int cnt = off[g + 1] - off[g], k = g % 5;
            goff[g] = make_int2(off[g], cnt);
            const float lbm = cnt > 0 ? jq4[off[g]].w : -1e30f;
            const float exf = std::nextafter((float)ext[g], std::numeric_limits<float>::infinity());
            const float iqm = std::nextafter((float)iqmax[g], std::numeric_limits<float>::infinity());
            grec[g] = make_float4(exf, iqm, lbm, 0.f);
            if (cnt > 0) {
                KJ.lbmax[k] = std::max(KJ.lbmax[k], lbm);
                KJ.iqmaxall[k] = std::max(KJ.iqmaxall[k], iqm);
                KJ.extmax[k] = std::max(KJ.extmax[k], exf);
            }
        }
        CK(pool.upload(&KJ.goff, goff)); CK(pool.upload(&KJ.grec, grec)); CK(pool.upload(&KJ.g4, g4));
    }
    // ---- shells, component factors ----
    {
        ShellInfo &sh = h->sh;
        sh.nshell = ns; sh.nbf = nbf;
        CK(pool.upload(&sh.l, sh_l)); CK(pool.upload(&sh.ao, sh_ao)); CK(pool.upload(&sh.atom, sh_atom));
        CK(pool.upload(&sh.cx, scx)); CK(pool.upload(&sh.cy, scy)); CK(pool.upload(&sh.cz, scz));
        CK(pool.upload(&h->fcomp, fcomp)); CK(pool.upload(&h->shell_of_ao, shell_of_ao));
    }
    // ---- A1: half-sphere G list with weights (eq 32-36; cutoff eq 62-64) ----
    {
        const double dk = cut.d_ewald_k > 0 ? cut.d_ewald_k : 1e-14;
        const double gcut = cut.g_cut > 0 ? cut.g_cut : 2.0 * omega * std::sqrt(std::log(1.0 / dk));
        std::vector<double> Gx, Gy, Gz, Gw;
        int mmax[3];
        for (int k = 0; k < 3; ++k) {
            const double an = std::sqrt(lat.a[3 * k] * lat.a[3 * k] + lat.a[3 * k + 1] * lat.a[3 * k + 1] + lat.a[3 * k + 2] * lat.a[3 * k + 2]);
            mmax[k] = (int)std::ceil(gcut * an / (2.0 * M_PI));
        }
        for (int m0 = 0; m0 <= mmax[0]; ++m0)
            for (int m1 = -mmax[1]; m1 <= mmax[1]; ++m1)
                for (int m2 = -mmax[2]; m2 <= mmax[2]; ++m2) {
                    if (m0 == 0 && (m1 < 0 || (m1 == 0 && m2 <= 0))) continue;    // half space, G = 0 omitted (L253)
                    double G[3];
                    for (int x = 0; x < 3; ++x)
                        G[x] = 2.0 * M_PI * (m0 * lat.binv[x] + m1 * lat.binv[3 + x] + m2 * lat.binv[6 + x]);
                    const double G2 = G[0] * G[0] + G[1] * G[1] + G[2] * G[2];
                    if (G2 >= gcut * gcut) continue;
                    if (cut.g_min > 0 && G2 < cut.g_min * cut.g_min) continue;           // window selection (tests)
                    Gx.push_back(G[0]); Gy.push_back(G[1]); Gz.push_back(G[2]);
                    Gw.push_back(std::sqrt(2.0 * 4.0 * M_PI / (lat.volume * G2) * std::exp(-G2 / (4.0 * omega * omega))));
                }
        h->nG = (int)Gx.size();
        LRParams &lr = h->lr;
        CK(pool.upload(&lr.Gx, Gx)); CK(pool.upload(&lr.Gy, Gy)); CK(pool.upload(&lr.Gz, Gz)); CK(pool.upload(&lr.Gw, Gw));
        lr.U = h->U; lr.sh = h->sh; lr.lat = lat; lr.N = nbf; lr.Np = h->Np; lr.fcomp = h->fcomp;
    }
    // ---- Boys tables: Taylor coefficients c[L][i][k] = F_{L+k}(x_i)/k! per top order L, and exp(-x_i) ----
    {
        std::vector<double> c((size_t)(LTOT + 1) * BOYS_ROWS * 8), ex(BOYS_ROWS);
        std::vector<float> cf(c.size());
        double F[BOYS_MCOL];
        const double ifact[8] = {1.0, 1.0, 0.5, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040};
        for (int i = 0; i < BOYS_ROWS; ++i) {
            boys_host(BOYS_MCOL - 1, i * BOYS_DX, F);
            ex[i] = std::exp(-i * BOYS_DX);
            for (int L = 0; L <= LTOT; ++L)
                for (int k = 0; k < 8; ++k) {
                    const size_t at = ((size_t)L * BOYS_ROWS + i) * 8 + k;
                    c[at] = F[L + k] * ifact[k];
                    cf[at] = (float)c[at];
                }
        }
        static_assert(LTOT + 7 < BOYS_MCOL, "the Taylor rows need F up to order LTOT + 7");
        CK(pool.upload(&h->boys.c, c)); CK(pool.upload(&h->boys.ex, ex)); CK(pool.upload(&h->boys.cf, cf));
    }
    // ---- workspaces ----
    {
        const size_t Np = h->Np, Npt = h->Npt, N = nbf;
        // G batch: A' and Y stacks of Np x 2nb x Np doubles each, at most 12 GB per stack (180 GB HBM3e per GPU)
        int nb = cut.lr_g_batch > 0 ? cut.lr_g_batch : (int)std::min<double>(64.0, std::floor(12.0e9 / (double)(Np * Np * 16)));
        nb = std::max(1, std::min(std::min(nb, 64), std::max(h->nG, 1)));      // the slot kernels hold at most 128 slots
        // the slot count of a batch is rounded up to the GEMM k-tile (32); padded slots are pure waste in both GEMMs, so the
        // default batch holds a multiple of 16 G vectors (2 slots each)
        if (cut.lr_g_batch <= 0 && nb >= 16) nb = (nb / 16) * 16;
        h->nb = nb;
        h->Smax = ((2 * nb + 31) / 32) * 32;             // slots of a full batch (multiple of 32)
        h->ld = (size_t)h->Smax * Np;
        // split of the K^LR accumulation over the rows of the factor: the lower 128x128 tiles times nsplit should
        // fill whole waves of one CTA per SM
        {
            const int nsm = h->nsm;
            const long tiles = (long)(Npt / 128) * (Npt / 128 + 1) / 2;
            double best = 0.0;
            h->nsplit = 1;
            for (int ns = 1; ns <= 8; ++ns) {
                const long ctas = tiles * ns, waves = (ctas + nsm - 1) / nsm;
                const double eff = (double)ctas / (double)(waves * nsm);
                if (eff > best + 0.02) { best = eff; h->nsplit = ns; }
            }
        }
        CK(pool.alloc(&h->Pp, Np * Np)); CK(cudaMemset(h->Pp, 0, Np * Np * 8));
        CK(pool.alloc(&h->lnPmax, 1)); CK(pool.alloc(&h->maxbits, 1));
        CK(pool.alloc(&h->lnPblk, (size_t)ns * ns)); CK(pool.alloc(&h->lnProw, (size_t)ns));
        CK(pool.alloc(&h->kjP, (size_t)std::max(h->KJ.n, 1)));
        if (h->mixed) { CK(pool.alloc(&h->Ppf, Np * Np)); CK(cudaMemset(h->Ppf, 0, Np * Np * sizeof(float))); }
        CK(pool.alloc(&h->counters, CNT_N)); CK(cudaMemset(h->counters, 0, CNT_N * 8));
        CK(pool.alloc(&h->Dt, (size_t)nherm(4) * h->KJ.dstride));
        CK(pool.alloc(&h->Jt, (size_t)nherm(4) * std::max(h->U.n, 1)));
        CK(pool.alloc(&h->Jsr, N * N)); CK(pool.alloc(&h->Jlr, N * N)); CK(pool.alloc(&h->Ksr, N * N));
        CK(pool.alloc(&h->Klr, (size_t)h->nsplit * Npt * Npt));
        // the GEMM row tiles are 128 high: the last one may reach up to 64 rows past Np (rows that are read or written but never
        // used), hence Npt rows
        CK(pool.alloc(&h->Astack, Npt * h->ld)); CK(cudaMemset(h->Astack, 0, Npt * h->ld * 8));
        CK(pool.alloc(&h->Zstack, Npt * h->ld)); CK(cudaMemset(h->Zstack, 0, Npt * h->ld * 8));
        CK(pool.alloc(&h->rho, (size_t)rho_scratch_doubles(h->Smax, agen_groups_total(h->lr))));
        CK(pool.alloc(&h->LT, Npt * Np)); CK(pool.alloc(&h->chol_d, 2 * Np)); CK(pool.alloc(&h->chol_s, 2));
        CK(pool.alloc(&h->chol_dyn, 8));      // rank, fallback flag, done, -, grid barrier (2)
        CK(pool.alloc(&h->hostP, N * N)); CK(pool.alloc(&h->hostJ, N * N)); CK(pool.alloc(&h->hostK, N * N));
        for (auto &e : h->ev) CK(cudaEventCreate(&e));
        h->evG.assign(2 * ((size_t)(h->nG + h->nb - 1) / h->nb + 2), nullptr);
        for (auto &e : h->evG) CK(cudaEventCreate(&e));
        // dynamic shared memory opt-in of the big kernels: per device, so once per handle
        sr_k_set_attributes();
        dgemm_set_attributes();
        CK(cudaGetLastError());
        for (auto &e : h->evJ) { CK(cudaEventCreate(&e[0])); CK(cudaEventCreate(&e[1])); }
        for (auto &e : h->evK) { CK(cudaEventCreate(&e[0])); CK(cudaEventCreate(&e[1])); }
    }
    // ---- A3: overlap S = rho_mn(G = 0) (eq 21) ----
    {
        h->cur_S = 16;                   // the whole stack was zero-filled at allocation
        launch_agen(h->lr, -1, 1, 16, 1.0, h->Astack, nullptr, nullptr, 0);
        double *dS = h->hostJ;
        launch_extract_overlap(h->Astack, h->Np, 16, nbf, h->fcomp, dS, 0);
        h->S_host.resize((size_t)nbf * nbf);
        CK(cudaMemcpy(h->S_host.data(), dS, (size_t)nbf * nbf * 8, cudaMemcpyDeviceToHost));
        CK(cudaGetLastError());
    }
    return PBC_JK_OK;
}

}  // namespace

extern "C" {

int pbc_jk_create(const pbc_cell *cell, const pbc_atoms *atoms, const pbc_shells *shells, double omega,
                  const pbc_cutoffs *cut, pbc_jk **out)
{
    if (out) *out = nullptr;
    if (!cell || !atoms || !shells || !out) return fail(nullptr, PBC_JK_ERR_INVALID_ARG, "null argument");
    if (!(omega > 0.0)) return fail(nullptr, PBC_JK_ERR_INVALID_ARG, "omega must be positive");
    if (atoms->natom < 1 || !atoms->xyz || shells->nshell < 1 || !shells->atom || !shells->l || !shells->nprim ||
        !shells->prim_off || !shells->exps || !shells->coefs)
        return fail(nullptr, PBC_JK_ERR_INVALID_ARG, "null or empty atoms/shells");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, PBC_JK_ERR_CUDA, "no CUDA device: libpbc_jk has no CPU fallback");
    }
    if (cut && (cut->precision < 0 || cut->precision > 1))
        return fail(nullptr, PBC_JK_ERR_INVALID_ARG, "precision must be 0 (fp64) or 1 (mixed)");
    pbc_jk *h = new (std::nothrow) pbc_jk();
    if (!h) return fail(nullptr, PBC_JK_ERR_NOMEM, "host allocation failed");
    if (cut) h->cut = *cut;
    h->mixed = h->cut.precision == 1;
    {
        const char *dbg = std::getenv("PBC_JK_DEBUG_SYNC");
        h->debug_sync = dbg && dbg[0] == '1';
    }
    h->mixed_switch = h->cut.mixed_switch > 0 ? h->cut.mixed_switch : 1e-5;
    if (cudaGetDevice(&h->device) != cudaSuccess ||
        cudaDeviceGetAttribute(&h->nsm, cudaDevAttrMultiProcessorCount, h->device) != cudaSuccess) {
        cudaGetLastError();
        delete h;
        return fail(nullptr, PBC_JK_ERR_CUDA, "cannot query the current CUDA device");
    }
    // set-up of pbc_jk_overlap_noalloc: the device address of its file-scope scratch array (once per device, this device
    // current); a failure is reported by that entry point, not here
    h->noalloc_err = noalloc_scratch_address(h->device, &h->noalloc_scratch);
    if (h->noalloc_err != cudaSuccess) cudaGetLastError();
    const auto t0 = std::chrono::steady_clock::now();
    int rc;
    try {
        rc = setup(h, cell, atoms, shells, omega);
    } catch (const std::bad_alloc &) {
        rc = fail(h, PBC_JK_ERR_NOMEM, "host allocation failed");
    } catch (...) {
        rc = fail(h, PBC_JK_ERR_INVALID_ARG, "unexpected failure in setup");
    }
    if (rc != PBC_JK_OK) {
        g_create_error = h->err;
        h->pool.free_all();
        destroy_events(h);
        delete h;
        return rc;
    }
    h->create_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    *out = h;
    return PBC_JK_OK;
}

int pbc_jk_nbf(const pbc_jk *h) { return h ? h->N : PBC_JK_ERR_INVALID_ARG; }

int pbc_jk_overlap(const pbc_jk *h, double *S_host)
{
    if (!h || !S_host) return PBC_JK_ERR_INVALID_ARG;
    std::memcpy(S_host, h->S_host.data(), h->S_host.size() * sizeof(double));
    return PBC_JK_OK;
}

static_assert(NOALLOC_MAX_NP == PBC_JK_NOALLOC_MAX_NBF, "header and kernel file disagree on the static scratch size");

int pbc_jk_overlap_noalloc(pbc_jk *h, double *S_dev, void *cuda_stream)
{
    if (!h) return PBC_JK_ERR_INVALID_ARG;
    if (!S_dev) return fail(h, PBC_JK_ERR_INVALID_ARG, "S_dev is null");
    if (h->Np > NOALLOC_MAX_NP) {
        char buf[200];
        std::snprintf(buf, sizeof buf, "pbc_jk_overlap_noalloc: N = %d (padded to %d) exceeds the static scratch, sized for at most %d "
                      "basis functions", h->N, h->Np, NOALLOC_MAX_NP);
        return fail(h, PBC_JK_ERR_UNSUPPORTED, buf);
    }
    {
        int dev = -1;
        CK(cudaGetDevice(&dev));
        if (dev != h->device) return fail(h, PBC_JK_ERR_INVALID_ARG, "the handle was created on another CUDA device than the current one");
    }
    if (h->noalloc_err != cudaSuccess || !h->noalloc_scratch) {
        char buf[200];
        std::snprintf(buf, sizeof buf, "pbc_jk_overlap_noalloc: cudaGetSymbolAddress of the static scratch failed at create: %s",
                      cudaGetErrorString(h->noalloc_err));
        return fail(h, PBC_JK_ERR_CUDA, buf);
    }
    CK(launch_overlap_noalloc(h->lr, h->noalloc_scratch, h->N, S_dev, (cudaStream_t)cuda_stream));
    return PBC_JK_OK;
}

int pbc_jk_set_parts(pbc_jk *h, int32_t parts)
{
    if (!h || parts < 0 || parts > 7) return PBC_JK_ERR_INVALID_ARG;
    h->parts = parts;
    return PBC_JK_OK;
}

int pbc_jk_set_shard(pbc_jk *h, int32_t rank, int32_t nranks)
{
    if (!h || nranks < 1 || rank < 0 || rank >= nranks) return PBC_JK_ERR_INVALID_ARG;
    h->shard_rank = rank;
    h->shard_n = nranks;
    return PBC_JK_OK;
}

static int build_impl(pbc_jk *h, const double *P, const double *Corb, int nocc, double *J, double *K, void *cuda_stream);

int pbc_jk_build(pbc_jk *h, const double *P, double *J, double *K, void *cuda_stream)
{
    if (!h) return PBC_JK_ERR_INVALID_ARG;
    if (!P) return fail(h, PBC_JK_ERR_INVALID_ARG, "P is null");
    return build_impl(h, P, nullptr, 0, J, K, cuda_stream);
}

int pbc_jk_build_orbitals(pbc_jk *h, const double *C, int32_t nocc, double *J, double *K, void *cuda_stream)
{
    if (!h) return PBC_JK_ERR_INVALID_ARG;
    if (!C) return fail(h, PBC_JK_ERR_INVALID_ARG, "C is null");
    if (nocc < 1 || nocc > h->N) return fail(h, PBC_JK_ERR_INVALID_ARG, "nocc must be in 1..N");
    return build_impl(h, nullptr, C, nocc, J, K, cuda_stream);
}

static int build_impl(pbc_jk *h, const double *P, const double *Corb, int nocc, double *J, double *K, void *cuda_stream)
{
    {
        int dev = -1;
        CK(cudaGetDevice(&dev));
        if (dev != h->device) return fail(h, PBC_JK_ERR_INVALID_ARG, "the handle was created on another CUDA device than the current one");
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int N = h->N, Np = h->Np, Npt = h->Npt;
    const size_t NN = (size_t)N * N;
    const bool doSR = h->parts & 1, doLR = h->parts & 2, doSELF = (h->parts & 4) && h->shard_rank == 0;
    const bool prof = h->profile;
    if (Corb) {                          // P = C C^T into the staging buffer of build_host (not in use by this entry point)
        launch_density_from_orbitals(Corb, N, nocc, h->hostP, st);
        P = h->hostP;
    }
    CK(cudaMemsetAsync(h->counters, 0, CNT_N * 8, st));
    CK(cudaEventRecord(h->ev[0], st));
    int64_t nl = 0;                      // kernels launched by this build
    for (auto &b : h->ranJ) b = false;
    for (auto &b : h->ranK) b = false;
    // ---- A4: density prep ----
    launch_scale_density(P, h->Pp, h->mixed ? h->Ppf : nullptr, N, Np, h->fcomp, h->maxbits, h->lnPmax, h->counters + CNT_FLAG, st);
    launch_density_blocks(h->Pp, Np, h->sh, h->KJ, h->lnPblk, h->lnProw, h->kjP, st);
    nl += 4 + (h->KJ.n > 0) + (Corb ? 1 : 0);
    SRParams sp;
    sp.K = h->K; sp.U = h->U; sp.KJ = h->KJ; sp.lat = h->lat; sp.sh = h->sh;
    sp.boys = h->boys; sp.Pp = h->Pp; sp.Ppf = h->Ppf; sp.ldP = Np; sp.Dt = h->Dt; sp.Jt = h->Jt; sp.Ksr = h->Ksr;
    sp.lnPmax = h->lnPmax; sp.lnPblk = h->lnPblk; sp.lnProw = h->lnProw; sp.kjP = h->kjP;
    sp.ln_tau = std::log(h->cut.d_schwarz > 0 ? h->cut.d_schwarz : 1e-13);
    sp.rcut2 = h->cut.r_cut > 0 ? h->cut.r_cut * h->cut.r_cut : std::numeric_limits<double>::infinity();
    sp.ln_switch = (float)std::log(h->mixed_switch);
    sp.shard_rank = h->shard_rank; sp.shard_n = h->shard_n;
    sp.counters = h->counters;
    if (J && doSR && h->KJ.n > 0) {
        launch_hermite_density(h->U, h->sh, h->KJ, h->Pp, Np, h->Dt, st);
        ++nl;
    }
    if (J && doSR) {
        CK(cudaMemsetAsync(h->Jt, 0, (size_t)nherm(4) * std::max(h->U.n, 1) * 8, st));
        CK(cudaMemsetAsync(h->Jsr, 0, NN * 8, st));
    }
    if (K && doSR) CK(cudaMemsetAsync(h->Ksr, 0, NN * 8, st));
    CK(cudaEventRecord(h->ev[1], st));
    // ---- A5 / A6: real-space classes, one launch each on the caller's stream, heaviest first (profile mode adds an event
    // pair per launch).  Spreading the classes over internal streams was measured SLOWER on B200 (water64 real space:
    // 573 ms on one stream, 685 / 724 ms on 2 / 3 streams -- kernels of different classes sharing an SM evict each
    // other's evaluator code from the instruction cache), so there is no fork/join here.
    if (K && doSR) {
        for (int L = 4 * LMAX; L >= 0; --L)                       // heaviest classes first
            for (int la = LMAX; la >= 0; --la)
                for (int ld = la; ld >= 0; --ld)
                    for (int lb = LMAX; lb >= 0; --lb) {
                        const int lc = L - la - ld - lb;
                        if (lc < 0 || lc > LMAX) continue;
                        if (h->nkblk[la][ld] <= 0 || !h->has_l[lb] || !h->has_l[lc]) continue;
                        const int cls = ((la * 3 + lb) * 3 + lc) * 3 + ld;
                        cudaStream_t cs = st;
                        if (prof) CK(cudaEventRecord(h->evK[cls][0], cs));
                        launch_sr_k(la, lb, lc, ld, h->mixed, sp, h->kblk[la][ld], h->nkblk[la][ld], cs);
                        if (h->debug_sync) {
                            const cudaError_t e = cudaStreamSynchronize(cs);
                            if (e != cudaSuccess) {
                                char buf[160];
                                std::snprintf(buf, sizeof buf, "real-space K class (%d%d|%d%d): %s", la, lb, lc, ld, cudaGetErrorString(e));
                                return fail(h, PBC_JK_ERR_CUDA, buf);
                            }
                        }
                        if (prof) CK(cudaEventRecord(h->evK[cls][1], cs));
                        h->ranK[cls] = true;
                        ++nl;
                    }
    }
    CK(cudaEventRecord(h->ev[2], st));
    if (J && doSR) {
        for (int LB = 4; LB >= 0; --LB) {
            cudaStream_t cs = st;
            for (int LK = 4; LK >= 0; --LK) {
                if (h->njbra[LB] <= 0 || h->njbra[LK] <= 0) continue;
                const int cls = LB * 5 + LK;
                if (prof) CK(cudaEventRecord(h->evJ[cls][0], cs));
                launch_sr_j(LB, LK, sp, h->jbra[LB], h->njbra[LB], cs);
                if (h->debug_sync) {
                    const cudaError_t e = cudaStreamSynchronize(cs);
                    if (e != cudaSuccess) {
                        char buf[160];
                        std::snprintf(buf, sizeof buf, "real-space J class (%d,%d): %s", LB, LK, cudaGetErrorString(e));
                        return fail(h, PBC_JK_ERR_CUDA, buf);
                    }
                }
                if (prof) CK(cudaEventRecord(h->evJ[cls][1], cs));
                h->ranJ[cls] = true;
                ++nl;
            }
        }
    }
    CK(cudaEventRecord(h->ev[3], st));
    // ---- A7/A8: reciprocal space, batches of G (on the caller's stream) ----
    const bool needJlr = J && (doLR || doSELF), needKlr = K && (doLR || doSELF);
    if (J) CK(cudaMemsetAsync(h->Jlr, 0, NN * 8, st));
    if (K) CK(cudaMemsetAsync(h->Klr, 0, (size_t)h->nsplit * Npt * Npt * 8, st));
    const size_t strideK = (size_t)Npt * Npt;
    // K^LR = sum_slots Y^T Y with Y = L^T A', P' = L L^T (device-side rank; dense fallback inside the same kernels)
    if (needKlr) {
        if (Corb) {                      // the orbitals are the factor: no decomposition
            launch_factor_from_orbitals(Corb, N, nocc, Np, Npt, h->fcomp, h->LT, h->chol_dyn, st);
            nl += 1;
        } else {
            launch_factor_density(h->Pp, N, Np, Npt, h->LT, h->chol_d, h->chol_dyn, h->chol_s, h->Zstack, st);
            nl += factor_density_launches(N);
        }
    }
    // one batch of S slots (layout A'[row*Np*S + col*S + slot]):  Y = L^T A'  (rows >= rank skipped), then
    // K += alpha sum_r sum_slot Y[r][mu][slot] Y[r][nu][slot] on the lower tiles (batches = rows r of the factor)
    h->n_evG = 0;
    auto klr_batch = [&](int S, double alpha, int nsplit) {
        const size_t ldS = (size_t)Np * S;
        const bool tg = prof && 2 * (size_t)h->n_evG + 1 < h->evG.size();
        if (tg) cudaEventRecord(h->evG[2 * h->n_evG], st);
        GemmArgs g1;
        g1.M = Npt; g1.Nc = Np * S; g1.Kb = Np; g1.nbatch = 1; g1.A = h->LT; g1.lda = Np; g1.B = h->Astack; g1.ldb = ldS;
        g1.C = h->Zstack; g1.ldc = ldS; g1.dyn = h->chol_dyn; g1.use_dyn = 1;
        launch_dgemm(g1, st);
        GemmArgs g2;
        g2.M = Npt; g2.Nc = Npt; g2.Kb = S; g2.nbatch = Np; g2.alpha = alpha; g2.transB = true;
        g2.A = h->Zstack; g2.lda = S; g2.strideA = ldS; g2.B = h->Zstack; g2.ldb = S; g2.strideB = ldS;
        g2.B_alt = h->Astack; g2.beta = 1.0; g2.C = h->Klr; g2.ldc = Npt; g2.strideC = strideK; g2.nsplit = nsplit;
        g2.dyn = h->chol_dyn; g2.use_dyn = 4 | 8; g2.lower_only = 1;
        launch_dgemm(g2, st);
        if (tg) { cudaEventRecord(h->evG[2 * h->n_evG + 1], st); ++h->n_evG; }
    };
    const int n_agen = agen_launches(h->lr);
    // Elements of shell pairs with no primitive pair-image are never written by agen_kernel and must read as 0:
    // the stack is zero-filled whenever its layout (the slot count S) changes.
    auto set_layout = [&](int S) -> cudaError_t {
        if (h->cur_S == S) return cudaSuccess;
        h->cur_S = S;
        return cudaMemsetAsync(h->Astack, 0, (size_t)Np * Np * S * sizeof(double), st);
    };
    if (doLR) {
        int ibatch = 0;
        for (int g0 = 0; g0 < h->nG; g0 += h->nb, ++ibatch) {
            if (ibatch % h->shard_n != h->shard_rank) continue;      // multi-GPU: G batches dealt round-robin
            const int nb = std::min(h->nb, h->nG - g0), S = ((2 * nb + 31) / 32) * 32;
            CK(set_layout(S));
            launch_agen(h->lr, g0, nb, S, 0.0, h->Astack, h->Pp, J ? h->rho : nullptr, st);
            nl += n_agen + (J ? 3 : 0) + (K ? 2 : 0);
            if (J) {
                launch_rho_final(h->lr, S, h->rho, st);
                launch_jlr_accum(h->Astack, Np, N, S, h->rho, 1.0, h->Jlr, st);
            }
            if (K) klr_batch(S, 1.0, h->nsplit);
        }
    }
    // ---- A9: the G = 0 slot, weight -pi/(Omega w^2), A = S ----
    if (doSELF) {
        CK(set_layout(32));
        launch_agen(h->lr, -1, 1, 32, std::sqrt(h->c0), h->Astack, h->Pp, J ? h->rho : nullptr, st);
        nl += n_agen + (J ? 3 : 0) + (K ? 2 : 0);
        if (J) {
            launch_rho_final(h->lr, 32, h->rho, st);
            launch_jlr_accum(h->Astack, Np, N, 32, h->rho, -1.0, h->Jlr, st);
        }
        if (K) klr_batch(32, -1.0, h->nsplit);
    }
    CK(cudaEventRecord(h->ev[4], st));
    if (J && doSR && h->U.nsp > 0) {
        launch_j_backtransform(h->U, h->sh, h->Jt, h->Jsr, N, st);
        ++nl;
    }
    // ---- A10 ----
    if (J) launch_finalize_j(doSR ? h->Jsr : nullptr, h->Jlr, N, h->fcomp, J, st);
    if (K)
        launch_finalize_k(doSR ? h->Ksr : nullptr, h->sh, h->Klr, h->nsplit, strideK, Npt, N, h->fcomp,
                          h->shell_of_ao, K, st);
    nl += (J ? 1 : 0) + (K ? 1 : 0);
    CK(cudaEventRecord(h->ev[5], st));
    CK(cudaGetLastError());
    h->n_launches = nl;
    h->last_stream = st;
    h->built = true;
    h->profiled_last = prof;
    return PBC_JK_OK;
}

// Ewald energy of the point charges (eq 91) on the host: O(natom^2 images + natom N_G), once per geometry.
static double ewald_point_charges(const pbc_jk *h, const double *q)
{
    const Lattice &lat = h->lat;
    const int na = h->natom;
    const double w = h->omega, w2 = w * w;
    const double *x = h->atom_xyz.data();
    const double delta = 1e-18;
    double qtot = 0.0, q2 = 0.0;
    for (int a = 0; a < na; ++a) { qtot += q[a]; q2 += q[a] * q[a]; }
    // real space: erfc(w r)/r < e^{-w^2 r^2} below delta (eq 92-93)
    const double rb = std::sqrt(std::log(1.0 / delta)) / w;
    double e_sr = 0.0;
#pragma omp parallel for reduction(+ : e_sr) schedule(dynamic, 4)
    for (int a = 0; a < na; ++a)
        for (int b = a; b < na; ++b) {
            if (q[a] == 0.0 || q[b] == 0.0) continue;
            const double d[3] = {x[3 * a] - x[3 * b], x[3 * a + 1] - x[3 * b + 1], x[3 * a + 2] - x[3 * b + 2]};
            const double md[3] = {-d[0], -d[1], -d[2]};
            double sum = 0.0;
            for_images_host(lat, md, rb, [&](const double *T) {
                const double v0 = d[0] + T[0], v1 = d[1] + T[1], v2 = d[2] + T[2];
                const double r = std::sqrt(v0 * v0 + v1 * v1 + v2 * v2);
                if (r > 1e-12) sum += std::erfc(w * r) / r;
            });
            e_sr += (a == b ? 0.5 : 1.0) * q[a] * q[b] * sum;
        }
    // reciprocal space: full sphere, 4 pi/(Omega G^2) e^{-G^2/4w^2} |sum q e^{-iG.C}|^2 / 2 (cutoff eq 94 at delta)
    const double gcut = 2.0 * w * std::sqrt(std::log(1.0 / delta));
    int mmax[3];
    for (int k = 0; k < 3; ++k) {
        const double an = std::sqrt(lat.a[3 * k] * lat.a[3 * k] + lat.a[3 * k + 1] * lat.a[3 * k + 1] + lat.a[3 * k + 2] * lat.a[3 * k + 2]);
        mmax[k] = (int)std::ceil(gcut * an / (2.0 * M_PI));
    }
    double e_lr = 0.0;
#pragma omp parallel for reduction(+ : e_lr) schedule(dynamic, 1)
    for (int m0 = -mmax[0]; m0 <= mmax[0]; ++m0)
        for (int m1 = -mmax[1]; m1 <= mmax[1]; ++m1)
            for (int m2 = -mmax[2]; m2 <= mmax[2]; ++m2) {
                if (m0 == 0 && m1 == 0 && m2 == 0) continue;
                double G[3];
                for (int k = 0; k < 3; ++k) G[k] = 2.0 * M_PI * (m0 * lat.binv[k] + m1 * lat.binv[3 + k] + m2 * lat.binv[6 + k]);
                const double G2 = G[0] * G[0] + G[1] * G[1] + G[2] * G[2];
                if (G2 >= gcut * gcut) continue;
                double nr = 0.0, ni = 0.0;
                for (int a = 0; a < na; ++a) {
                    const double ph = -(G[0] * x[3 * a] + G[1] * x[3 * a + 1] + G[2] * x[3 * a + 2]);
                    nr += q[a] * std::cos(ph); ni += q[a] * std::sin(ph);
                }
                e_lr += 0.5 * 4.0 * M_PI / (lat.volume * G2) * std::exp(-G2 / (4.0 * w2)) * (nr * nr + ni * ni);
            }
    const double e_c = -M_PI / (lat.volume * w2) * 0.5 * qtot * qtot - w / std::sqrt(M_PI) * q2;
    return e_sr + e_lr + e_c;
}

int pbc_jk_one_electron(pbc_jk *h, const double *charges_host, double *T, double *V, double *e_nuc_host, void *cuda_stream)
{
    if (!h) return PBC_JK_ERR_INVALID_ARG;
    if ((V || e_nuc_host) && !charges_host) return fail(h, PBC_JK_ERR_INVALID_ARG, "charges are null");
    {
        int dev = -1;
        CK(cudaGetDevice(&dev));
        if (dev != h->device) return fail(h, PBC_JK_ERR_INVALID_ARG, "the handle was created on another CUDA device than the current one");
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int N = h->N, Np = h->Np, na = h->natom;
    if (T) launch_kinetic(h->U, h->sh, h->fcomp, T, N, st);
    if (V) {
        // device copies of the charges and the folded atom positions (not on the per-iteration path: allocated here)
        double *dq = nullptr, *dx = nullptr;
        CK(cudaMalloc(&dq, sizeof(double) * na));
        if (cudaMalloc(&dx, sizeof(double) * 3 * na) != cudaSuccess) { cudaFree(dq); return fail(h, PBC_JK_ERR_NOMEM, "device allocation failed"); }
        cudaMemcpyAsync(dq, charges_host, sizeof(double) * na, cudaMemcpyHostToDevice, st);
        cudaMemcpyAsync(dx, h->atom_xyz.data(), sizeof(double) * 3 * na, cudaMemcpyHostToDevice, st);
        double qmax = 0.0;
        for (int a = 0; a < na; ++a) qmax = std::max(qmax, std::fabs(charges_host[a]));
        const size_t NN = (size_t)N * N;
        // short range: Hermite-basis Vt of every pair-image (workspace Jt), back-transformed into Jsr (eq 96-97)
        cudaMemsetAsync(h->Jt, 0, (size_t)nherm(4) * std::max(h->U.n, 1) * 8, st);
        cudaMemsetAsync(h->Jsr, 0, NN * 8, st);
        cudaMemsetAsync(h->Jlr, 0, NN * 8, st);
        const double d_pair = h->cut.d_pair > 0 ? h->cut.d_pair : 1e-14;
        launch_sr_v(h->U, h->lat, h->boys, h->jbra, h->njbra, dx, dq, na, qmax, std::log(d_pair * 1e-2), h->KJ.g0, h->KJ.rc, h->Jt, st);
        if (h->U.nsp > 0) launch_j_backtransform(h->U, h->sh, h->Jt, h->Jsr, N, st);
        // long range: J^LR with rho(G) replaced by the structure factor of the charges; SELF: the G = 0 slot
        auto set_layout = [&](int S) {
            if (h->cur_S == S) return;
            h->cur_S = S;
            cudaMemsetAsync(h->Astack, 0, (size_t)Np * Np * S * sizeof(double), st);
        };
        for (int g0 = 0; g0 < h->nG; g0 += h->nb) {
            const int nb = std::min(h->nb, h->nG - g0), S = ((2 * nb + 31) / 32) * 32;
            set_layout(S);
            launch_agen(h->lr, g0, nb, S, 0.0, h->Astack, nullptr, nullptr, st);
            launch_rho_nuc(h->lr, g0, nb, S, 0.0, dx, dq, na, h->rho, st);
            launch_jlr_accum(h->Astack, Np, N, S, h->rho, 1.0, h->Jlr, st);
        }
        set_layout(16);
        launch_agen(h->lr, -1, 1, 16, std::sqrt(h->c0), h->Astack, nullptr, nullptr, st);
        launch_rho_nuc(h->lr, -1, 1, 16, std::sqrt(h->c0), dx, dq, na, h->rho, st);
        launch_jlr_accum(h->Astack, Np, N, 16, h->rho, -1.0, h->Jlr, st);
        launch_finalize_j(h->Jsr, h->Jlr, N, h->fcomp, V, st);
        CK(cudaStreamSynchronize(st));
        cudaFree(dq); cudaFree(dx);
    }
    if (e_nuc_host) *e_nuc_host = ewald_point_charges(h, charges_host);
    CK(cudaGetLastError());
    return PBC_JK_OK;
}

int pbc_jk_build_host(pbc_jk *h, const double *P_host, double *J_host, double *K_host)
{
    if (!h) return PBC_JK_ERR_INVALID_ARG;
    if (!P_host) return fail(h, PBC_JK_ERR_INVALID_ARG, "P is null");
    const size_t bytes = (size_t)h->N * h->N * 8;
    CK(cudaMemcpyAsync(h->hostP, P_host, bytes, cudaMemcpyHostToDevice, 0));
    const int rc = pbc_jk_build(h, h->hostP, J_host ? h->hostJ : nullptr, K_host ? h->hostK : nullptr, nullptr);
    if (rc != PBC_JK_OK) return rc;
    if (J_host) CK(cudaMemcpyAsync(J_host, h->hostJ, bytes, cudaMemcpyDeviceToHost, 0));
    if (K_host) CK(cudaMemcpyAsync(K_host, h->hostK, bytes, cudaMemcpyDeviceToHost, 0));
    unsigned long long flag = 0;
    CK(cudaMemcpyAsync(&flag, h->counters + CNT_FLAG, sizeof(flag), cudaMemcpyDeviceToHost, 0));
    CK(cudaStreamSynchronize(0));
    if (flag) return fail(h, PBC_JK_ERR_UNSUPPORTED, "max |P| exceeds 1e6: the lattice image range of the real-space sums was not validated for it");
    return PBC_JK_OK;
}

int pbc_jk_get_stats(pbc_jk *h, pbc_jk_stats_t *out)
{
    if (!h || !out) return PBC_JK_ERR_INVALID_ARG;
    std::memset(out, 0, sizeof(*out));
    out->nbf = h->N; out->nshell = h->nshell; out->natom = h->natom; out->n_g = h->nG;
    out->n_prim_pairs = h->n_prim_pairs; out->n_shell_pair_images = h->n_sp_images;
    out->create_seconds = h->create_seconds;
    if (h->built) {
        CK(cudaEventSynchronize(h->ev[5]));
        unsigned long long c[CNT_N];
        CK(cudaMemcpy(c, h->counters, sizeof(c), cudaMemcpyDeviceToHost));
        for (int i = 0; i < NCLS_J; ++i) { out->candidates_j += (int64_t)c[CNT_CAND_J + i]; out->quartets_j += (int64_t)c[CNT_Q_J + i]; }
        for (int i = 0; i < NCLS_K; ++i) {
            out->candidates_k += (int64_t)c[CNT_CAND_K + i];
            out->quartets_k += (int64_t)c[CNT_Q_K + i];
            out->quartets_k_fp32 += (int64_t)c[CNT_Q32_K + i];
        }
        out->n_launches = h->n_launches;
        float ms[5];
        for (int i = 0; i < 5; ++i) CK(cudaEventElapsedTime(&ms[i], h->ev[i], h->ev[i + 1]));
        float tot;
        CK(cudaEventElapsedTime(&tot, h->ev[0], h->ev[5]));
        out->ms_density = ms[0]; out->ms_sr_k = ms[1]; out->ms_sr_j = ms[2]; out->ms_lr = ms[3] + ms[4]; out->ms_total = tot;
        if (h->profiled_last)
            for (int i = 0; i < h->n_evG; ++i) {
                float t = 0.f;
                CK(cudaEventElapsedTime(&t, h->evG[2 * i], h->evG[2 * i + 1]));
                out->ms_lr_gemm += t;
            }
        {
            int dyn[2] = {0, 0};
            CK(cudaMemcpy(dyn, h->chol_dyn, sizeof(dyn), cudaMemcpyDeviceToHost));
            out->rank_p = dyn[0];
        }
        if (c[CNT_FLAG]) return fail(h, PBC_JK_ERR_UNSUPPORTED, "max |P| exceeds 1e6: the lattice image range of the real-space sums was not validated for it");
    }
    return PBC_JK_OK;
}

int pbc_jk_set_profile(pbc_jk *h, int32_t on)
{
    if (!h) return PBC_JK_ERR_INVALID_ARG;
    h->profile = on != 0;
    return PBC_JK_OK;
}

int pbc_jk_get_class_stats(pbc_jk *h, pbc_jk_class_stat *out, int32_t cap, int32_t *n_out)
{
    if (!h || !n_out || (cap > 0 && !out)) return PBC_JK_ERR_INVALID_ARG;
    *n_out = 0;
    if (!h->built) return PBC_JK_OK;
    CK(cudaEventSynchronize(h->ev[5]));
    unsigned long long c[CNT_N];
    CK(cudaMemcpy(c, h->counters, sizeof(c), cudaMemcpyDeviceToHost));
    int n = 0;
    for (int cls = 0; cls < NCLS_J; ++cls) {
        if (!h->ranJ[cls]) continue;
        if (n < cap) {
            pbc_jk_class_stat &s = out[n];
            s.kind = 0; s.l[0] = cls / 5; s.l[1] = cls % 5; s.l[2] = s.l[3] = 0;
            s.quartets = (int64_t)c[CNT_Q_J + cls]; s.candidates = (int64_t)c[CNT_CAND_J + cls];
            float ms = 0.f;
            if (h->profiled_last) CK(cudaEventElapsedTime(&ms, h->evJ[cls][0], h->evJ[cls][1]));
            s.ms = ms;
        }
        ++n;
    }
    for (int cls = 0; cls < NCLS_K; ++cls) {
        if (!h->ranK[cls]) continue;
        if (n < cap) {
            pbc_jk_class_stat &s = out[n];
            s.kind = 1; s.l[0] = cls / 27; s.l[1] = (cls / 9) % 3; s.l[2] = (cls / 3) % 3; s.l[3] = cls % 3;
            s.quartets = (int64_t)c[CNT_Q_K + cls]; s.candidates = (int64_t)c[CNT_CAND_K + cls];
            float ms = 0.f;
            if (h->profiled_last) CK(cudaEventElapsedTime(&ms, h->evK[cls][0], h->evK[cls][1]));
            s.ms = ms;
        }
        ++n;
    }
    *n_out = n;
    return PBC_JK_OK;
}

const char *pbc_jk_last_error(const pbc_jk *h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int pbc_jk_destroy(pbc_jk *h)
{
    if (!h) return PBC_JK_OK;
    cudaDeviceSynchronize();
    h->pool.free_all();
    destroy_events(h);
    delete h;
    return PBC_JK_OK;
}

}  // extern "C"
