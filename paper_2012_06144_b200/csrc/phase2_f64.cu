// fp64 instances of the two-cells-per-thread phase-field LB kernel (16-byte accesses)
#define ACM_T double
#include "phase2_impl.cuh"
