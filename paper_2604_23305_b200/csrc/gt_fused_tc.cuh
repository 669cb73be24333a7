// gt_fused_tc.cuh -- steps 2-6a as ONE tcgen05 tensor-core kernel (GT_VARIANT_TENSOR).
// Placeholder until the tensor kernel lands: plan creation reports GT_ERR_UNSUPPORTED.
#pragma once
#include <vector>
#include "gt_common.cuh"
#include "gt_fused_fp32.cuh"
#include "../../include/gateau_b200.h"

namespace gt {

struct TcTables {
    unsigned char* filt_img = nullptr;
};

inline const char* tc_error() { return "tensor-core kernel not built yet"; }

inline gt_status build_tc_tables(const std::vector<float>&, int, int, int, TcTables&, cudaStream_t) {
    return GT_ERR_UNSUPPORTED;
}
inline void free_tc_tables(TcTables& t) { if (t.filt_img) cudaFree(t.filt_img); t.filt_img = nullptr; }

inline cudaError_t launch_fused_tc(const FusedParams&, const TcTables&, int, cudaStream_t) {
    return cudaErrorNotSupported;
}

}  // namespace gt
