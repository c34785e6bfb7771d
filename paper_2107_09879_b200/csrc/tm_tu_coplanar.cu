// Translation unit: coplanar kernel (lmax 1..3, fp64 and packed-fp32) and the cost figures of both coplanar code sets.
#define TM_SEC_COP
#include "tm_launch_impl.cuh"
#include "generated/tm_coplanar4_cost.h"
void tm_cost_coplanar(int lmax, double* inst, double* flop) {
  const int I[8] = {0, TM_COP_FPINST_L1, TM_COP_FPINST_L2, TM_COP_FPINST_L3, TM_COP4_FPINST_L4, TM_COP4_FPINST_L5, TM_COP4_FPINST_L6, TM_COP4_FPINST_L7};
  const int F[8] = {0, TM_COP_FLOP_L1, TM_COP_FLOP_L2, TM_COP_FLOP_L3, TM_COP4_FLOP_L4, TM_COP4_FLOP_L5, TM_COP4_FLOP_L6, TM_COP4_FLOP_L7};
  *inst = I[lmax]; *flop = F[lmax];
}
