// Translation unit: rotation-based 3-D kernel, lmax 6.
#define TM_SEC_ROT3D
#define TM_RANGE_6
#include "tm_launch_impl.cuh"
