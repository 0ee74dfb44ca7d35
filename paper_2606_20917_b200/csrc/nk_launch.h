// nk_launch.h -- type-erased launch table shared by the per-(shape,P) instantiation units
// (nk_inst.cu, compiled once per pair) and the dispatcher in nk_api.cu (layer B1).
#pragma once
#include "nk_kernels.cuh"

namespace nk {

// tabs_flat / sx_flat: the doubles of DenseTabs<P+1,P+2> / SimplexTabs in declaration order.
typedef cudaError_t (*LaunchFn)(const double* tabs_flat, const double* sx_flat, const KArgs& a, int num_sms,
                                cudaStream_t stream);

struct InstInfo {
    int shape, P, Q;
    int E[2], threads[2], blocks_per_sm_hint[2]; // [deformed]
    size_t smem_grid[2];
    LaunchFn fn[2][OP_COUNT]; // [deformed][op]
    int E_op_affine[OP_COUNT]; // elements per block of each AFFINE kernel (TuneOp; the geometry stream keeps E[0])
};

} // namespace nk

#define NK_INST_NAME2(s, p) nk_inst_##s##_##p
#define NK_INST_NAME(s, p) NK_INST_NAME2(s, p)
