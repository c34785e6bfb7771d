// Translation unit: warp-split rotation-based 3-D kernel, lmax 4..6.
#define TM_SEC_ROT3DW
#include "tm_launch_impl.cuh"
