// fp64 instances of the fused hydrodynamic LB kernel (the paper's precision)
#define ACM_T double
#include "hydro_impl.cuh"
