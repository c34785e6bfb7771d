// Translation unit: table-driven kernel (lmax 1..7).
#define TM_SEC_GEN
#include "tm_launch_impl.cuh"
