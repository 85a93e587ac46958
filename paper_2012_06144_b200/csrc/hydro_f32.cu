// fp32 instances of the fused hydrodynamic LB kernel (BASELINE config 5, A22)
#define ACM_T float
// fp32 threads hold half the bytes in flight of the fp64 ones: 24 resident warps (<= 85 registers) instead of
// 20 make up for it (+6 % at 256^3 D3Q27, profiles/r1_variants.md); no spills at this bound
#define ACM_HYDRO_MINB 3
#include "hydro_impl.cuh"
