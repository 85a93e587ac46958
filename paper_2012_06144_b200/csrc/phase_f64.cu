// fp64 instances of the fused phase-field LB kernel (the paper's precision)
#define ACM_T double
#include "phase_impl.cuh"
