#include "dslash_launch.cuh"
INSTANTIATE_DSLASH(F64, 18, FORM_B)
