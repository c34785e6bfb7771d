// Translation unit: direct generated 3-D kernel (lmax 1..3).
#define TM_SEC_SYM3D
#include "tm_launch_impl.cuh"
