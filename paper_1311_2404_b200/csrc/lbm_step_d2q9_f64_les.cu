// Step kernels of the LES model for <D2Q9, double> (see lbm_steps.cuh).
#define LBM_STEP_LES
#include "lbm_steps.cuh"

template int lbm_step_les<D2Q9, double>(lbm_ctx *, int);
