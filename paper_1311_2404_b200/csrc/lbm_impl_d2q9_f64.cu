// Kernel instantiations for <D2Q9, double> (see lbm_impl.cuh).
#include "lbm_impl.cuh"

const void *lbm_impl_d2q9_f64() { return Impl<D2Q9, double>::table(); }
