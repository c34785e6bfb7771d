// Translation unit: warp-split four-sector coplanar kernel, lmax 4..6.
#define TM_SEC_COP4W
#include "tm_launch_impl.cuh"
