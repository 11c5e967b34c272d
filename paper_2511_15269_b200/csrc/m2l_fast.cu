// m2l_fast.cu -- unrolled register M2L kernels (placeholder: none built yet, the generic kernel is used).
#include "internal.cuh"
namespace fmm {
bool m2l_fast_available(int, fmm_dtype) { return false; }
void m2l_fast_launch(const Plan&, cudaStream_t) {}
}  // namespace fmm
