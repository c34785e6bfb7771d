// Translation unit: four-sector coplanar kernel, lmax 4 and 5.
#define TM_SEC_COP4
#define TM_RANGE_LO
#include "tm_launch_impl.cuh"
