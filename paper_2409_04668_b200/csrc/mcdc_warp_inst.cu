// mcdc_warp_inst.cu -- the k_warp instantiations of one VARIANT (compile with -DMCDC_WARP_VARIANT=0..3; see build.py)
#ifndef MCDC_WARP_VARIANT
#error "compile with -DMCDC_WARP_VARIANT=<0..3>"
#endif
#include "mcdc_warp_inst.cuh"
