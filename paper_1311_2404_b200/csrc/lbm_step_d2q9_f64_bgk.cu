// Step kernels of the BGK model for <D2Q9, double> (see lbm_steps.cuh).
#define LBM_STEP_BGK
#include "lbm_steps.cuh"

template int lbm_step_bgk<D2Q9, double>(lbm_ctx *, int);
