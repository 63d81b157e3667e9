#include "dslash_launch.cuh"
INSTANTIATE_DSLASH(F32, 12, FORM_B)
