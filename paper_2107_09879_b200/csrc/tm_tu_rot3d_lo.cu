// Translation unit: rotation-based 3-D kernel, lmax 1..5.
#define TM_SEC_ROT3D
#define TM_RANGE_LO
#include "tm_launch_impl.cuh"
