// bench-only: kernel A's memory accesses with trivial arithmetic (FORM_PROBE), fp32, 18-real links
#include "dslash_launch.cuh"
INSTANTIATE_DSLASH(F32, 18, FORM_PROBE)
