// Kernel instantiations for <D3Q19, double> (see lbm_impl.cuh).
#include "lbm_impl.cuh"

const void *lbm_impl_d3q19_f64() { return Impl<D3Q19, double>::table(); }
