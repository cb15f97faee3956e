// Step kernels of the MRT model for <D2Q9, double> (see lbm_steps.cuh).
#define LBM_STEP_MRT
#include "lbm_steps.cuh"

template int lbm_step_mrt<D2Q9, double>(lbm_ctx *, int);
