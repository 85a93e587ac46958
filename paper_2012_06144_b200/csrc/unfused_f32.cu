// fp32 instances of the six unfused kernels of Algorithm 1 (measured comparison)
#define ACM_T float
#include "unfused_impl.cuh"
