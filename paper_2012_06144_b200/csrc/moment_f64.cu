// moment representation kernels (ACM_OPT_MOMENTS), fp64
#define ACM_T double
#include "moment_impl.cuh"
