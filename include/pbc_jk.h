/*
 * pbc_jk.h -- C ABI of the B200-native Gamma-point, Ewald-split periodic J/K builder.
 *
 * Method: arxiv 2410.22278; scope: SURVEY.md section 8.  All "eq"/"L" citations
 * are PAPER.md equation numbers / line numbers.
 *
 *   J_mn = sum_ls P_ls (mn|ls)      (eq 73)       Coulomb matrix
 *   K_mn = sum_ls P_ls (ml|sn)      (eq 74)   exact-exchange matrix (no -1/2)
 *
 * with the crystalline, Gamma-point two-electron integral split as in eq 56 (L439),
 * generalised to p,d shells by eq 69 (L518) and eq 98 (L742-750):
 *
 *   (mn|ls) = SR  [erfc(w r)/r over lattice-image-translated primitive quartets, sums R1,R2,R3]
 *           + LR  [sum_{G != 0} 4 pi/(Omega G^2) exp(-G^2/4w^2) Re conj(rho_mn(G)) rho_ls(G)]
 *           + SELF[-pi/(Omega w^2) S_mn S_ls]           (eq 35, eq 56 third term)
 *
 * Basis: contracted Cartesian Gaussian shells, l in {0,1,2} (eq 4-6).  AO order:
 * shells in input order; components p: x,y,z; d: xx,xy,xz,yy,yz,zz (PAPER L721 example list).
 * Every Cartesian component is normalised on its own (eq 6); `coefs` multiply normalised
 * primitives.  The library never renormalises contracted functions.
 *
 * Pointers: everything handed to pbc_jk_create / pbc_jk_overlap's `S_host` is HOST memory and is
 * copied; P, J, K of pbc_jk_build are DEVICE pointers (N x N fp64, row-major, caller-owned),
 * the *_host variant takes HOST pointers and does the copies itself.  No torch types cross
 * this boundary.  All functions return PBC_JK_OK (0) or a negative pbc_jk_status; no C++
 * exception leaves the library; there is no global state besides the CUDA context.
 *
 * There is no CPU fallback: without a CUDA device pbc_jk_create fails with PBC_JK_ERR_CUDA.
 */
#ifndef PBC_JK_H
#define PBC_JK_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    PBC_JK_OK = 0,
    PBC_JK_ERR_INVALID_ARG = -1,   /* null pointer, w <= 0, singular cell, l > 2, exponent <= 0, nprim < 1 */
    PBC_JK_ERR_NOMEM = -2,         /* host or device allocation failed */
    PBC_JK_ERR_CUDA = -3,          /* CUDA runtime error; text via pbc_jk_last_error */
    PBC_JK_ERR_UNSUPPORTED = -4    /* lattice image index range exceeds the packed format (cell far too small for */
                                   /* the exponents / omega, or max|P| above 1e6), or a (shell, l) group holds    */
                                   /* more than 65535 primitive pair-images                                       */
} pbc_jk_status;

typedef struct pbc_jk pbc_jk;      /* opaque handle: owns all host + device state of one geometry */

/* rows = lattice vectors a1, a2, a3 in bohr; any non-singular cell (P1, no symmetry; L31) */
typedef struct { double a[9]; } pbc_cell;

/* xyz: 3*natom doubles, bohr; every centre may be in any lattice image (L781) */
typedef struct { int32_t natom; const double *xyz; } pbc_atoms;

/* nshell shells; shell s sits on atom[s], has angular momentum l[s] in {0,1,2} and nprim[s]
 * primitives exps[prim_off[s] ...], coefs[prim_off[s] ...] (eq 4) */
typedef struct {
    int32_t nshell;
    const int32_t *atom, *l, *nprim, *prim_off;
    const double *exps, *coefs;
} pbc_shells;

/* Thresholds (PAPER 3.6, L823-837).  A zero selects the default. */
typedef struct {
    double r_cut;        /* cap on |A-B-R2| and |Q-P+R1| in bohr (0: no cap; thresholds decide)       */
    double g_cut;        /* |G| cutoff in bohr^-1 (0: 2 w sqrt(ln(1/d_ewald_k)), from eq 62-64)   */
    double d_pair;       /* primitive pair-image kept iff its Schwarz-type bound (eq 60, with the */
                         /* angular factor of DESIGN.md) exceeds this; default 1e-14                   */
    double d_schwarz;    /* primitive quartet-image evaluated iff bound_bra*bound_ket*max|P|*          */
                         /* exp(-alpha_w r^2) (eq 67) exceeds this; default 1e-13                 */
    double d_ewald_k;    /* sets the default g_cut; default 1e-14                                      */
    int32_t precision;   /* 0 = fp64 everywhere.  1 = mixed (PAPER 3.5 L817-821): real-space K quartets */
                         /* whose density-weighted bound bound_bra*bound_ket*max|P block| is below      */
                         /* mixed_switch run in fp32 arithmetic with fp64 accumulation; everything else */
                         /* (J-engine, reciprocal space, quartets above the switch) stays fp64          */
    double mixed_switch; /* precision = 1 only; default 1e-5 (L819)                                     */
    int32_t lr_g_batch;  /* G vectors per reciprocal-space batch (0: sized to <= 12 GB per stack; <=64) */
    double g_min;        /* > 0: only G with |G| >= g_min enter the reciprocal-space sums (selection     */
                         /* only; tests use it to compare the outermost shell of G at full basis size)   */
} pbc_cutoffs;

/* Counters and phase times of the LAST pbc_jk_build (pbc_jk_get_stats waits for it). */
typedef struct {
    int32_t nbf, nshell, natom, n_g;        /* n_g: G != 0 in the half sphere (+-G paired, L243)  */
    int64_t n_prim_pairs;                   /* ordered primitive pair-images kept (A2)            */
    int64_t n_shell_pair_images;            /* ordered contracted shell-pair-images kept          */
    int64_t quartets_j, quartets_k;         /* primitive quartet-images evaluated in real space   */
    int64_t candidates_j, candidates_k;     /* primitive quartet-images tested by the screen      */
    double  ms_density, ms_sr_j, ms_sr_k, ms_lr, ms_total;   /* device times, CUDA events         */
    double  create_seconds;                 /* host wall time of pbc_jk_create                    */
    int64_t n_launches;                     /* CUDA kernels the last build launched               */
    int64_t quartets_k_fp32;                /* the part of quartets_k evaluated in fp32 (mixed)   */
    double  ms_lr_gemm;                     /* profile mode: device time of the K^LR GEMM launches */
    int32_t rank_p;                         /* rank of the factor P' = L L^T used by K^LR (N: dense fallback) */
} pbc_jk_stats_t;

/* One real-space kernel class of the LAST build (one launch per class and build).
 * kind 0: J-engine class, l[0] = Hermite order of the bra pair (l_mu + l_nu), l[1] = of the ket pair
 *         (eq 96-98); kind 1: K class (l_mu l_lambda | l_sigma l_nu) in l[0..3] (eq 74).
 * quartets / candidates: primitive quartet-images evaluated / tested (eq 67) by that launch.
 * ms: device time of the launch (CUDA events on the build's stream); 0 unless profile mode was on during that build. */
typedef struct {
    int32_t kind;
    int32_t l[4];
    int64_t quartets, candidates;
    double  ms;
} pbc_jk_class_stat;

/*
 * A1-A3: validates, builds the reciprocal lattice and the half-sphere G list
 * (eq 32-36), the image-summed primitive pair lists with bounds (Fig 1, eq 57-61
 * L449-469, lattice enumeration eq 99-103), the Hermite expansion coefficient products
 * E^{ab}_t of every primitive pair-image (eq 16-20), the Boys tables, and the crystalline
 * overlap S (eq 21); uploads everything; sizes all workspaces.  `cut` may be NULL (all defaults).
 * Uses the current CUDA device.  On failure *out is NULL.
 */
int pbc_jk_create(const pbc_cell *cell, const pbc_atoms *atoms, const pbc_shells *shells,
                  double omega, const pbc_cutoffs *cut, pbc_jk **out);

/* number of basis functions N (AO order as documented above); negative status on NULL */
int pbc_jk_nbf(const pbc_jk *h);

/* copies the crystalline overlap S (eq 21) into S_host, N*N doubles, HOST memory */
int pbc_jk_overlap(const pbc_jk *h, double *S_host);

/*
 * Allocation-free variant for callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses
 * that forbid it): recomputes the crystalline overlap S (eq 21, S_mn = rho_mn(G = 0), the same kernels
 * pbc_jk_create runs) into `S_dev`, N*N doubles row-major, DEVICE memory, caller-owned, overwritten.  All work is
 * enqueued on `cuda_stream`; the call allocates nothing (no cudaMalloc/cudaFree, no allocating library routine) and
 * does not synchronise the host.  Its scratch is a file-scope device array inside the library, sized for at most
 * PBC_JK_NOALLOC_MAX_NBF basis functions after padding N to a multiple of 64 (4 MiB, held by every GPU that loads
 * the library until the process exits); a larger handle is refused with PBC_JK_ERR_UNSUPPORTED and a text in
 * pbc_jk_last_error.  ALL calls of the process share that array, on every handle and stream: calls that overlap on
 * the GPU race -- order them on one stream or with events.  The array keeps the last call's contents; each call
 * clears the part it reads before use.  Must be called with the handle's device current.
 */
#define PBC_JK_NOALLOC_MAX_NBF 512
int pbc_jk_overlap_noalloc(pbc_jk *h, double *S_dev, void *cuda_stream);

/*
 * A4-A10: one J+K build for density P (symmetric, N x N fp64 row-major, DEVICE).  J and/or K may
 * be NULL to skip that matrix; otherwise they are OVERWRITTEN with the full matrices (SR+LR+SELF).
 * All work is enqueued on `cuda_stream` (a cudaStream_t, NULL = default stream); the call does not
 * synchronise the host and allocates nothing.  One build in flight per handle.
 */
int pbc_jk_build(pbc_jk *h, const double *P, double *J, double *K, void *cuda_stream);

/*
 * Occupied-orbital entry point (the direction PAPER L941 names as future work for the reciprocal-space
 * part): C is N x nocc fp64 row-major (DEVICE), the density is P = C C^T (eq 72, occupations folded into C).
 * Same outputs and contract as pbc_jk_build; the reciprocal-space K contraction uses C itself as the factor of P
 * (cost 8 nocc N^2 per G vector) instead of decomposing P.
 */
int pbc_jk_build_orbitals(pbc_jk *h, const double *C, int32_t nocc, double *J, double *K, void *cuda_stream);

/* Same with HOST buffers: copies P host->device, builds, copies J/K back, synchronises. */
int pbc_jk_build_host(pbc_jk *h, const double *P_host, double *J_host, double *K_host);

/*
 * One-electron Ewald terms of the same geometry.  Any output may be NULL.
 *   T  (DEVICE, N x N, overwritten): kinetic matrix, SI eq S1 (L1151-1169; -1/2 Laplacian on the second function,
 *      image-summed like the overlap).
 *   V  (DEVICE, N x N, overwritten): V_mn = sum_C q_C (mn | point charge at atom C) under the zero-mean periodic
 *      Coulomb kernel, Ewald-split as eq 52 (L372-386): erfc part over lattice images, reciprocal part through
 *      rho_mn(G), and the -pi/(Omega w^2) S_mn sum_C q_C term.  Sign as in the paper: the electron-nucleus
 *      attraction matrix is -V with q_C = Z_C.
 *   e_nuc_host (HOST, one double): Ewald energy of the point charges, eq 91 (L679-686), including the
 *      -pi/(Omega w^2) (sum q)^2 / 2 term of a charged cell.
 * charges_host: natom doubles (HOST), one charge per atom of pbc_jk_create.  Enqueues on `cuda_stream` and
 * synchronises it before returning (setup-time call, not part of the per-iteration build); uses the handle's
 * build workspaces, so no build may be in flight.
 */
int pbc_jk_one_electron(pbc_jk *h, const double *charges_host, double *T, double *V, double *e_nuc_host,
                        void *cuda_stream);

/* `parts` bit 0 SR, bit 1 LR, bit 2 SELF (default 7): restrict the next builds to these terms of
 * eq 56 (bring-up and tests: the oracle returns the same parts separately). */
int pbc_jk_set_parts(pbc_jk *h, int32_t parts);

/* waits for the last build on its stream and fills the counters/times */
int pbc_jk_get_stats(pbc_jk *h, pbc_jk_stats_t *out);

/* profile mode (default off): the real-space class launches run one after the other on the caller's stream with a
 * CUDA event pair around each (per-class times); otherwise the classes are spread over internal streams that fork
 * from and join back into the caller's stream, so that the tail of one class overlaps the next */
int pbc_jk_set_profile(pbc_jk *h, int32_t on);

/* waits for the last build and writes up to `cap` class records to `out` (HOST memory, caller-owned);
 * *n_out = number of classes the build launched (may exceed cap: call again with a larger array) */
int pbc_jk_get_class_stats(pbc_jk *h, pbc_jk_class_stat *out, int32_t cap, int32_t *n_out);

/* text of the last error on this handle ("" if none); valid until the next call on the handle.
 * With h == NULL: the text of the last failed pbc_jk_create of this thread. */
const char *pbc_jk_last_error(const pbc_jk *h);

/* frees all host and device memory of the handle; NULL is a no-op */
int pbc_jk_destroy(pbc_jk *h);

/*
 * Multi-GPU: this handle does the share `rank` of `nranks` of every build --
 * real-space K output blocks and J-engine bras dealt round-robin (lists sorted by cost), reciprocal-space
 * G batches likewise, the SELF term on rank 0 -- so that the SUM over the ranks' J (and K) is the full
 * matrix: the caller adds them up with one all-reduce (the Python binding does, over torch.distributed).
 * Default (0, 1): the whole build.
 */
int pbc_jk_set_shard(pbc_jk *h, int32_t rank, int32_t nranks);

#ifdef __cplusplus
}
#endif
#endif /* PBC_JK_H */
