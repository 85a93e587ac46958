// fp32 instances of the fused phase-field LB kernel (BASELINE config 5, A22)
#define ACM_T float
// fp32 threads hold half the bytes in flight of the fp64 ones: 24 resident warps (<= 85 registers) instead of
// 20 make up for it (+6 % at 256^3 D3Q27, profiles/r1_variants.md); the instances with walls keep 2 blocks (<= 128
// registers): at 85 they spill.  These single-cell kernels are the fallback for odd nx; the default is *_kernel2.
#define ACM_PHASE_MINB 3
#include "phase_impl.cuh"
