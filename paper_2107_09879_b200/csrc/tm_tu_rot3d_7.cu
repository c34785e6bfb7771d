// Translation unit: rotation-based 3-D kernel, lmax 7 (internal: gradient at lmax 6).
#define TM_SEC_ROT3D
#define TM_RANGE_7
#include "tm_launch_impl.cuh"
