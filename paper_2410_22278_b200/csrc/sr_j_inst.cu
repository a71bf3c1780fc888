// Instantiations of the real-space J-engine kernels for one bra Hermite order J_LB (0..4) and
// every ket Hermite order 0..4.  Compiled five times (-DJ_LB=0..4).
#include "pbcjk_sr.cuh"

#ifndef J_LB
#error "compile with -DJ_LB=<0..4>"
#endif
#define CAT2(a, b) a##b
#define CAT(a, b) CAT2(a, b)

namespace pbcjk {

void CAT(launch_sr_j_, J_LB)(int LK, const SRParams &p, const int *bra_idx, int nbra, cudaStream_t st)
{
    if (nbra <= 0) return;
    const int mine = p.shard_n > 1 ? (nbra + p.shard_n - 1) / p.shard_n : nbra;     // bras of this rank (multi-GPU)
    dim3 grid((mine + 3) / 4), block(128);
    switch (LK) {
    case 0: sr_j_kernel<J_LB, 0><<<grid, block, 0, st>>>(p, bra_idx, nbra); break;
    case 1: sr_j_kernel<J_LB, 1><<<grid, block, 0, st>>>(p, bra_idx, nbra); break;
    case 2: sr_j_kernel<J_LB, 2><<<grid, block, 0, st>>>(p, bra_idx, nbra); break;
    case 3: sr_j_kernel<J_LB, 3><<<grid, block, 0, st>>>(p, bra_idx, nbra); break;
    case 4: sr_j_kernel<J_LB, 4><<<grid, block, 0, st>>>(p, bra_idx, nbra); break;
    default: break;
    }
}

}  // namespace pbcjk
