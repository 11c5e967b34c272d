// xlate_smem.cu -- entry points of the shared-memory translation kernels (xlate_smem.cuh): 9 <= p <= 12, fp32 and fp64
#include "internal.cuh"

namespace fmm {

bool xlate_smem_launch_f32(const Plan& P, int kind, int level, cudaStream_t st, int64_t e0, int64_t e1);
bool xlate_smem_launch_f64(const Plan& P, int kind, int level, cudaStream_t st, int64_t e0, int64_t e1);

bool xlate_smem_available(int p, fmm_dtype dt) { return p >= 9 && p <= 12 && (dt == FMM_F32 || dt == FMM_F64); }

void xlate_smem_launch(const Plan& P, int kind, int level, cudaStream_t st, int64_t e0, int64_t e1) {
    const bool ok = P.dtype == FMM_F64 ? xlate_smem_launch_f64(P, kind, level, st, e0, e1) : xlate_smem_launch_f32(P, kind, level, st, e0, e1);
    if (!ok) { set_error("no shared-memory translation kernel for this order"); throw CudaFail{FMM_ERR_UNSUPPORTED}; }
}

}  // namespace fmm
