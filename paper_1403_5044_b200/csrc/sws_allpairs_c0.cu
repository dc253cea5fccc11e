// Bank 0 of the uniform-operand all-pairs kernel (see sws_allpairs_const.cuh): a module of its own, so that it has a
// 64 KB __constant__ bank of its own.
#define SWS_CONST_BANK 0
#include "sws_allpairs_const.cuh"
