// fp32 instances of the fused hydrodynamic LB kernel (BASELINE config 5, A22)
#define ACM_T float
#include "hydro_impl.cuh"
