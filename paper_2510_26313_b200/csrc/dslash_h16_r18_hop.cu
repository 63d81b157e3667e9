#include "dslash_launch.cuh"
INSTANTIATE_DSLASH(H16, 18, FORM_HOP)
