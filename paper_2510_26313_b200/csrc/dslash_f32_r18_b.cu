#include "dslash_launch.cuh"
INSTANTIATE_DSLASH(F32, 18, FORM_B)
