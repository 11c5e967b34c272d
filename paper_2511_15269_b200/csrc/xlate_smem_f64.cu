// xlate_smem_f64.cu -- fp64 instantiation of the shared-memory translation kernels (xlate_smem.cuh), orders 9..12
#include "xlate_smem.cuh"

namespace fmm {
bool xlate_smem_launch_f64(const Plan& P, int kind, int level, cudaStream_t st, int64_t e0, int64_t e1) {
    return smem_launch_t<double>(P, kind, level, st, e0, e1);
}
}  // namespace fmm
