// Instantiations of the real-space K kernels for one (K_LA, K_LB, K_LD) = (l_mu, l_lambda, l_nu)
// and l_sigma = 0..2.  Compiled once per (K_LA >= K_LD, K_LB): 18 objects.
#include "pbcjk_sr.cuh"

#if !defined(K_LA) || !defined(K_LB) || !defined(K_LD)
#error "compile with -DK_LA= -DK_LB= -DK_LD="
#endif
#define CAT4_(a, b, c, d) a##b##c##d
#define CAT4(a, b, c, d) CAT4_(a, b, c, d)

namespace pbcjk {

void CAT4(launch_sr_k_, K_LA, K_LB, K_LD)(int lc, const SRParams &p, const int2 *blocks, int nblocks, cudaStream_t st)
{
    if (nblocks <= 0) return;
    dim3 grid(nblocks), block(KWARPS * 32);
    switch (lc) {
    case 0: sr_k_kernel<K_LA, K_LB, 0, K_LD><<<grid, block, 0, st>>>(p, blocks, nblocks); break;
    case 1: sr_k_kernel<K_LA, K_LB, 1, K_LD><<<grid, block, 0, st>>>(p, blocks, nblocks); break;
    case 2: sr_k_kernel<K_LA, K_LB, 2, K_LD><<<grid, block, 0, st>>>(p, blocks, nblocks); break;
    default: break;
    }
}

}  // namespace pbcjk
