// Instantiations of the warp-per-tile fused dslash kernel (shared-memory staged operands): precision code 2, 1 flavor(s).
#include "tm_dslash_tile.cuh"

TM_TILE_TABLE(2, 1)
