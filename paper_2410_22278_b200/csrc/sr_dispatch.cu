// Class dispatch of the real-space kernel families (one launcher per instantiation unit).
#include "pbcjk_sr.cuh"

namespace pbcjk {

#define DECL_J(LB) void launch_sr_j_##LB(int, const SRParams &, const int *, int, cudaStream_t);
DECL_J(0) DECL_J(1) DECL_J(2) DECL_J(3) DECL_J(4)
#define DECL_K(A, B, D)                                                                         \
    void launch_sr_k_##A##B##D##_0(int, const SRParams &, const int2 *, int, cudaStream_t);     \
    void launch_sr_k_##A##B##D##_1(int, const SRParams &, const int2 *, int, cudaStream_t);     \
    void set_attr_sr_k_##A##B##D##_0();                                                         \
    void set_attr_sr_k_##A##B##D##_1();
#define DECL_KB(A, D) DECL_K(A, 0, D) DECL_K(A, 1, D) DECL_K(A, 2, D)
DECL_KB(0, 0) DECL_KB(1, 0) DECL_KB(1, 1) DECL_KB(2, 0) DECL_KB(2, 1) DECL_KB(2, 2)

void launch_sr_j(int LB, int LK, const SRParams &p, const int *bra_idx, int nbra, cudaStream_t st)
{
    switch (LB) {
    case 0: launch_sr_j_0(LK, p, bra_idx, nbra, st); break;
    case 1: launch_sr_j_1(LK, p, bra_idx, nbra, st); break;
    case 2: launch_sr_j_2(LK, p, bra_idx, nbra, st); break;
    case 3: launch_sr_j_3(LK, p, bra_idx, nbra, st); break;
    case 4: launch_sr_j_4(LK, p, bra_idx, nbra, st); break;
    default: break;
    }
}

void launch_sr_k(int la, int lb, int lc, int ld, bool mixed, const SRParams &p, const int2 *blocks, int nblocks, cudaStream_t st)
{
    if (la + lb + lc + ld > 4) mixed = false;          // K_MIXED_LMAX of pbcjk_srk.cuh: the high classes stay fp64
#define CASE_K(A, B, D)                                                   \
    if (la == A && lb == B && ld == D) {                                  \
        if (mixed) launch_sr_k_##A##B##D##_1(lc, p, blocks, nblocks, st); \
        else launch_sr_k_##A##B##D##_0(lc, p, blocks, nblocks, st);       \
        return;                                                           \
    }
#define CASE_KB(A, D) CASE_K(A, 0, D) CASE_K(A, 1, D) CASE_K(A, 2, D)
    CASE_KB(0, 0) CASE_KB(1, 0) CASE_KB(1, 1) CASE_KB(2, 0) CASE_KB(2, 1) CASE_KB(2, 2)
}

void sr_k_set_attributes()
{
#define ATTR_K(A, B, D) set_attr_sr_k_##A##B##D##_0(); set_attr_sr_k_##A##B##D##_1();
#define ATTR_KB(A, D) ATTR_K(A, 0, D) ATTR_K(A, 1, D) ATTR_K(A, 2, D)
    ATTR_KB(0, 0) ATTR_KB(1, 0) ATTR_KB(1, 1) ATTR_KB(2, 0) ATTR_KB(2, 1) ATTR_KB(2, 2)
}

}  // namespace pbcjk
