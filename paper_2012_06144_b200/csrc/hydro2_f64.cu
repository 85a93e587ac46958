// fp64 instances of the two-cells-per-thread hydrodynamic LB kernel (16-byte accesses)
#define ACM_T double
#include "hydro2_impl.cuh"
