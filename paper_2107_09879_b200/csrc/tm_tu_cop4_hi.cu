// Translation unit: four-sector coplanar kernel, lmax 6 and 7.
#define TM_SEC_COP4
#define TM_RANGE_HI
#include "tm_launch_impl.cuh"
