#include "dslash_launch.cuh"
INSTANTIATE_DSLASH(H16, 12, FORM_A)
