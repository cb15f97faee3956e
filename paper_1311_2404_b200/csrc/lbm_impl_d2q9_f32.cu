// Kernel instantiations for <D2Q9, float> (see lbm_impl.cuh).
#include "lbm_impl.cuh"

const void *lbm_impl_d2q9_f32() { return Impl<D2Q9, float>::table(); }
