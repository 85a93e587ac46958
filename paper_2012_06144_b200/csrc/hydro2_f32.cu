// fp32 instances of the two-cells-per-thread hydrodynamic LB kernel (packed fp32 pipe, 8-byte accesses)
#define ACM_T float
#include "hydro2_impl.cuh"
