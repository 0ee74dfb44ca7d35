// nk_dense_launch.h -- host interface of the reference-matrix (DMMA) kernels of nk_dense.cuh / nk_dense.cu
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

#include "nk_dense.cuh"

namespace nk {

enum { DENSE_HELM = 0, DENSE_LAP = 1, DENSE_MASS = 2, DENSE_KINDS = 3 };
// first matrix and number of matrices of each kind (see DenseShape)
inline int dense_c0(int kind) { return kind == DENSE_MASS ? 6 : 0; }
inline int dense_nc(int kind) { return kind == DENSE_HELM ? 7 : kind == DENSE_LAP ? 6 : 1; }

// true if a kernel is instantiated for this number of modes per element
bool dense_supported(int nmodes);
// launches the kernel for (nmodes, kind) on `stream`; a.bfrag must hold dense_pack(K7, nmodes, c0(kind), nc(kind)).
// *launched is set to 1 if a kernel was enqueued (0 for an empty range).
cudaError_t dense_launch(int nmodes, int kind, const DenseArgs& a, cudaStream_t stream, int* launched);

// ---- run-time specialisation (csrc/nk_jit.cu): NVRTC compiles nk_dense.cuh for a mode count outside the table ----
} // namespace nk
#include <string>
namespace nk {
// compiles (cached per device, Nm, kind) and launches; false + *err on any failure (no NVRTC, no driver, compile error)
bool dense_jit_launch(int nmodes, int kind, const DenseArgs& a, cudaStream_t stream, int* launched, std::string* err);
// compiles only (needs no GPU): time in ms and size of the cubin
bool dense_jit_compile_check(int nmodes, int kind, double* ms, size_t* cubin_bytes, std::string* err);
// kernels compiled for launching so far in this process, and the time NVRTC took for them
void dense_jit_stats(long long* kernels, double* total_ms);

} // namespace nk
