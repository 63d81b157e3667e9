// bench-only: kernel A's memory accesses with trivial arithmetic (FORM_PROBE), int16+norm storage, 18-real links
#include "dslash_launch.cuh"
INSTANTIATE_DSLASH(H16, 18, FORM_PROBE)
