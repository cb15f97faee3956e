// Step kernels of the SC model for <D2Q9, float> (see lbm_steps.cuh).
#define LBM_STEP_SC
#include "lbm_steps.cuh"

template int lbm_step_sc<D2Q9, float>(lbm_ctx *, int);
