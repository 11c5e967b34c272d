// xlate_smem.cu -- the shared-memory translation kernels (xlate_smem.cuh): fp64, 9 <= p <= 12.  (fp32 keeps the state vector in
// registers up to p = 12, xlate_fast.cu.)
#include "xlate_smem.cuh"

namespace fmm {

bool xlate_smem_available(int p, fmm_dtype dt) { return p >= 9 && p <= 12 && dt == FMM_F64; }

void xlate_smem_launch(const Plan& P, int kind, int level, cudaStream_t st, int64_t e0, int64_t e1) {
    const bool ok = P.dtype == FMM_F64 && smem_launch_t<double>(P, kind, level, st, e0, e1);
    if (!ok) { set_error("no shared-memory translation kernel for this order and dtype"); throw CudaFail{FMM_ERR_UNSUPPORTED}; }
}

}  // namespace fmm
