// Instantiations of the packed-FP32 (FFMA2) fused dslash kernel: precision code 2, 2 flavor(s).
#include "tm_dslash_f2.cuh"

TM_F2_TABLE(2, 2)
