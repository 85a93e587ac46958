// fp32 instances of the fused phase-field LB kernel (BASELINE config 5, A22)
#define ACM_T float
#include "phase_impl.cuh"
