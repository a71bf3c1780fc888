// Launchers of the "light" kernels: density prep (A4), J back-transform (eq 97), reciprocal-space
// passes (A7-A9) and the FP64 tensor-core GEMM used by the reciprocal-space K contraction (A8).
#pragma once
#include "pbcjk_common.h"

namespace pbcjk {

struct LRParams {
    PairListU U;
    ShellInfo sh;
    Lattice lat;
    int N, Np;                 // basis size and its padded size (multiple of 64)
    const double *fcomp;       // [N] per-component factor (1 or sqrt 3)
    const double *Gx, *Gy, *Gz, *Gw;   // half-sphere G list, Gw = sqrt(2 * 4 pi/(Omega G^2) exp(-G^2/4w^2))
    const int *sp_cls[9];      // shell pairs of U by class (l_A*3 + l_B): one agen_kernel instantiation each
    int n_sp_cls[9];
};

// P' = f P f (into the padded Np x Np buffer, pads untouched) and ln(max |P'|)
// (Ppf: optional fp32 copy for the mixed-precision evaluators; flag: set when max|P'| exceeds e^{LN_PMAX_CAP})
void launch_scale_density(const double *P, double *Pp, float *Ppf, int N, int Np, const double *fcomp,
                          unsigned long long *maxbits, double *lnPmax, unsigned long long *flag, cudaStream_t st);
// ln max|P'| per shell block [nshell x nshell], its row maxima, and the block value of every J ket's own pair (L819)
void launch_density_blocks(const double *Pp, int Np, const ShellInfo &sh, const KetListJ &KJ, float *lnPblk, float *lnProw,
                           float *kjP, cudaStream_t st);
void launch_to_float(const double *src, float *dst, size_t n, cudaStream_t st);
void dgemm_set_attributes();
// E^{AB}_t product table of the ordered pair list (rows at K.eoff), built once per geometry
void launch_etab(const PairListK &K, const int *lA, const int *lB, double *etab, cudaStream_t st);
// D~_s of every J ket (eq 95)
void launch_hermite_density(const PairListU &U, const ShellInfo &sh, const KetListJ &KJ, const double *Pp, int Np,
                            double *Dt, cudaStream_t st);
// J_ab += sum_t (-1)^{|t|} E^{ab}_t Jt  per shell pair, mirrored (eq 96-97)
void launch_j_backtransform(const PairListU &U, const ShellInfo &sh, const double *Jt, double *Jsr, int N,
                            cudaStream_t st);
// A'(G) = sqrt(w) rho_mn(G) for G in [g0, g0+nb): real and imaginary parts as slots 2g, 2g+1 of the stack
//   A'[row*ld + col*S + slot], ld = Np*S, S >= 2*nb a multiple of 16 (slots past 2*nb are written as 0).
// g0 < 0: the single G = 0 slot with weight `w0` (overlap S, eq 21) in slot 0.
// With `rho` (rho_scratch_doubles(S, agen_groups_total) doubles) and the density Pp the kernels also leave the partial sums
// of rho'[slot] = sum P' o A'[slot] there; launch_rho_final reduces them into rho[0..S).
void launch_agen(const LRParams &p, int g0, int nb, int S, double w0, double *Astack, const double *Pp, double *rho, cudaStream_t st);
int agen_launches(const LRParams &p);
int agen_groups_total(const LRParams &p);
int rho_scratch_doubles(int S, int ngroups);
void launch_rho_final(const LRParams &p, int S, double *rho, cudaStream_t st);
// Jacc[m][n] += sign * sum_slot A'[m][n][slot] rho'[slot]
void launch_jlr_accum(const double *Astack, int Np, int N, int S, const double *rho, double sign, double *Jacc, cudaStream_t st);
// C[z][M x Nc] (ldc) = beta*C + alpha * sum_b op(A_b)[M x Kb] B_b[Kb x Nc](ldb) over the batches of split z;
// M, Nc multiples of 128, Kb of 16 (operand rows/columns past the logical size may alias the following memory: the
// affected result rows/columns are never read); grid.z = nsplit partial results C + z*strideC over disjoint batch ranges.
// See dgemm_kernel in pbcjk_lr.cu for transA / dyn / lower_only.
struct GemmArgs {
    int M = 0, Nc = 0, Kb = 0, nbatch = 1;
    double alpha = 1.0;
    const double *A = nullptr; size_t lda = 0, strideA = 0;
    const double *B = nullptr; size_t ldb = 0, strideB = 0;
    double beta = 0.0;
    double *C = nullptr; size_t ldc = 0, strideC = 0;
    int nsplit = 1;
    bool transA = false, transB = false;
    const int *dyn = nullptr; int use_dyn = 0;
    const double *B_alt = nullptr;
    int lower_only = 0;
};
void launch_dgemm(const GemmArgs &g, cudaStream_t st);
// P' = L L^T (pivoted Cholesky, device-side rank in dyn[0]) with the dense fallback L = P' (dyn[1] = 1);
// LT: Np x Np (row k = column k of L), dbuf: 2*Np, dyn: 8 ints (4 + the grid barrier of the one-launch factorisation),
// dscal: 2 doubles, scratch: Np x Np
// Npt = N padded to the 128-row GEMM tiles (LT holds Npt rows, the scratch Npt x Npt)
void launch_factor_density(const double *Pp, int N, int Np, int Npt, double *LT, double *dbuf, int *dyn, double *dscal,
                           double *scratch, cudaStream_t st);
int factor_density_launches(int N);     // kernels launch_factor_density enqueues
// occupied-orbital entry point: P = C C^T (N x N, unscaled) and the factor LT = (f C)^T with rank nocc (dyn as above)
void launch_density_from_orbitals(const double *C, int N, int nocc, double *P, cudaStream_t st);
void launch_factor_from_orbitals(const double *C, int N, int nocc, int Np, int Npt, const double *fcomp, double *LT, int *dyn,
                                 cudaStream_t st);
// out = f f (sum of parts), symmetrised; see pbcjk_lr.cu
void launch_finalize_j(const double *Jsr, const double *Jlr, int N, const double *fcomp, double *J, cudaStream_t st);
void launch_finalize_k(const double *Ksr, const ShellInfo &sh, const double *Klr, int nsplit, size_t strideK, int Np,
                       int N, const double *fcomp, const int *shell_of_ao, double *K, cudaStream_t st);
void launch_extract_overlap(const double *Astack, int Np, int S, int N, const double *fcomp, double *Sm, cudaStream_t st);
// allocation-free overlap (pbc_jk_overlap_noalloc): the scratch stack lives in a file-scope device array of pbcjk_lr.cu
// (NOALLOC_MAX_NP^2 * 2 doubles = 4 MiB); noalloc_scratch_address resolves its device address once per device (device current),
// launch_overlap_noalloc clears what it needs, runs the agen kernels into it and reads S out -- no allocation.
constexpr int NOALLOC_MAX_NP = 512;       // largest padded basis size N_p (multiple of 64) the static scratch holds
cudaError_t noalloc_scratch_address(int device, double **ptr);
cudaError_t launch_overlap_noalloc(const LRParams &p, double *scratch, int N, double *S_out, cudaStream_t st);

}  // namespace pbcjk
