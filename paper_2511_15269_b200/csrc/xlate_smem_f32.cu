// xlate_smem_f32.cu -- fp32 instantiation of the shared-memory translation kernels (xlate_smem.cuh), orders 9..12
#include "xlate_smem.cuh"

namespace fmm {
bool xlate_smem_launch_f32(const Plan& P, int kind, int level, cudaStream_t st, int64_t e0, int64_t e1) {
    return smem_launch_t<float>(P, kind, level, st, e0, e1);
}
}  // namespace fmm
