// fp64 instances of the six unfused kernels of Algorithm 1 (measured comparison)
#define ACM_T double
#include "unfused_impl.cuh"
