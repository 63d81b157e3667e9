// int16+norm spinors with int16 fixed-point links
#include "dslash_launch.cuh"
INSTANTIATE_DSLASH(H16L, 18, FORM_A)
