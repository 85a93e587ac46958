// fp32 instances of the two-cells-per-thread phase-field LB kernel (packed fp32 pipe, 8-byte accesses)
#define ACM_T float
#include "phase2_impl.cuh"
