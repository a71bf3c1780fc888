// Launchers of the one-electron Ewald terms: kinetic matrix, real- and reciprocal-space parts of the
// point-charge interaction matrix V.  See pbcjk_1e.cu.
#pragma once
#include "pbcjk_common.h"
#include "pbcjk_lr.cuh"
#include "pbcjk_md.cuh"

namespace pbcjk {

// T (N x N, overwritten): SI eq S1
void launch_kinetic(const PairListU &U, const ShellInfo &sh, const double *fcomp, double *T, int N, cudaStream_t st);
// Vt[t*U.n + u]: Hermite-basis short-range V of every U entry (eq 52), to be back-transformed like the J-engine's Jt
void launch_sr_v(const PairListU &U, const Lattice &lat, const BoysTab &boys, const int *const jbra[5], const int njbra[5],
                 const double *cxyz, const double *q, int natom, double qabs_max, double ln_delta, const double g0[3], double rc,
                 double *Vt, cudaStream_t st);
// rho'[slot] = sqrt(w) * structure factor of the charges for the G batch [g0, g0 + nb) (g0 < 0: the G = 0 slot, w0 * sum q)
void launch_rho_nuc(const LRParams &p, int g0, int nb, int S, double w0, const double *cxyz, const double *q, int natom, double *rho,
                    cudaStream_t st);

}  // namespace pbcjk
