// Kernel instantiations for <D3Q19, float> (see lbm_impl.cuh).
#include "lbm_impl.cuh"

const void *lbm_impl_d3q19_f32() { return Impl<D3Q19, float>::table(); }
