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

// ---- run-time specialisation of nk_kernel for a (shape, P, Q) outside the prebuilt table (csrc/nk_jit.cu) ----
struct JitOpCfg {
    int E, threads, minb;     // TuneOp<...>::E, NT, MINB
    size_t smem;              // TuneOp<...>::smem_grid
};
struct JitInfo {
    int shape, P, Q;
    int E[2];                       // interleave width of the geometry stream [deformed] (Tune<...>::E)
    JitOpCfg op[2][OP_COUNT];       // [deformed][op]
    size_t tabs_bytes, sx_bytes;    // sizeof(DenseTabs), sizeof(SimplexTabs) of this (shape, P, Q)
    bool sx_dup;                    // SimplexTabs holds separate adjoint copies (k_sx_dup)
};
enum { kJitMaxP = 10, kJitMaxQ = 12 };
} // namespace nk
#include <string>
namespace nk {
// the launch configuration the kernel template's own rules (Tune / TuneOp) give for (shape, P, Q); host only, needs no
// GPU.  false (+ *why) if the triple cannot be specialised: P > 10, Q < P+1, Q > 12, or kernel parameters beyond 32 KB.
bool sumfac_jit_info(int shape, int P, int Q, JitInfo* out, std::string* why);
// NVRTC-compiles (cached per device and instantiation) and launches nk_kernel<shape, P, def, op, Q>
bool sumfac_jit_launch(const JitInfo& info, int def, int op, const double* tabs_flat, const double* sx_flat, const KArgs& a,
                       int num_sms, cudaStream_t stream, std::string* err);
// compiles only (needs no GPU): time in ms and size of the cubin
bool sumfac_jit_compile_check(int shape, int P, int Q, int def, int op, double* ms, size_t* cubin_bytes, std::string* err);

} // namespace nk

#define NK_INST_NAME2(s, p) nk_inst_##s##_##p
#define NK_INST_NAME(s, p) NK_INST_NAME2(s, p)
