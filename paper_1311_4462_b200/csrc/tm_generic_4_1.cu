// Instantiations of the generic fused dslash kernel: precision code 4 (bytes per real), 1 flavor(s).
#include "tm_dslash.cuh"

TM_GENERIC_TABLE(4, 1)
