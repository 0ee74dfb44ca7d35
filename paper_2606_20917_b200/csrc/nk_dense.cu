// nk_dense.cu -- instantiations and launcher of the reference-matrix (DMMA) kernels (nk_dense.cuh): the affine
// simplex operators in coefficient space.  One instantiation per number of modes Nm (the kernel does not depend on
// the shape) and per operator kind (Helmholtz: matrices 0..6, Laplacian: 0..5, mass: 6).
#include <mutex>

#include "nk_dense_launch.h"

namespace nk {
namespace {

enum { kMaxDevices = 64 };
std::mutex g_dense_mutex;

template <int NMODES, int C0, int NC, int WARPS, int MINB>
cudaError_t launch_one(const DenseArgs& a, cudaStream_t stream, int* launched)
{
    using S = DenseShape<NMODES, C0, NC>;
    static int blocks_per_sm[kMaxDevices] = {};   // function attributes are per device (one entry per ordinal)
    static int num_sms[kMaxDevices] = {};
    auto kern = nk_dense_kernel<NMODES, C0, NC, WARPS, MINB>;
    const size_t smem = (size_t)S::TOTAL_DOUBLES * sizeof(double);
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    int bps, sms;
    {
        std::lock_guard<std::mutex> lk(g_dense_mutex);
        if (blocks_per_sm[dev] == 0) {
            err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (err != cudaSuccess) return err;
            err = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
            if (err != cudaSuccess) return err;
            int b = 0, n = 0;
            err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, kern, WARPS * 32, smem);
            if (err != cudaSuccess) return err;
            err = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
            if (err != cudaSuccess) return err;
            num_sms[dev] = n;
            blocks_per_sm[dev] = b < 1 ? 1 : b;
        }
        bps = blocks_per_sm[dev];
        sms = num_sms[dev];
    }
    *launched = 0;
    if (a.e1 <= a.e0 || a.nfields < 1) return cudaSuccess;
    const long long ntiles = ((a.e1 - a.e0 + 7) / 8) * a.nfields;
    if (ntiles >= 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    long long grid = (long long)sms * bps;                       // persistent: one wave
    const long long need = (ntiles + WARPS - 1) / WARPS;
    if (grid > need) grid = need;
    kern<<<(unsigned)grid, WARPS * 32, smem, stream>>>(a);
    *launched = 1;
    return cudaGetLastError();
}

// streamed variant (matrices in L2, ring of TMA chunks): WARPS consumer warps + 1 producer warp per block
template <int NMODES, int C0, int NC, int WARPS, int KSC, int STAGES, int MINB>
cudaError_t launch_stream(const DenseArgs& a, cudaStream_t stream, int* launched)
{
    using T = DenseStream<NMODES, C0, NC, KSC>;
    static int blocks_per_sm[kMaxDevices] = {};
    static int num_sms[kMaxDevices] = {};
    auto kern = nk_dense_stream_kernel<NMODES, C0, NC, WARPS, KSC, STAGES, MINB>;
    const size_t smem = T::smem_bytes(WARPS, STAGES);
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    int bps, sms;
    {
        std::lock_guard<std::mutex> lk(g_dense_mutex);
        if (blocks_per_sm[dev] == 0) {
            err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (err != cudaSuccess) return err;
            err = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
            if (err != cudaSuccess) return err;
            int b = 0, n = 0;
            err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, kern, (WARPS + 1) * 32, smem);
            if (err != cudaSuccess) return err;
            err = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
            if (err != cudaSuccess) return err;
            num_sms[dev] = n;
            blocks_per_sm[dev] = b < 1 ? 1 : b;
        }
        bps = blocks_per_sm[dev];
        sms = num_sms[dev];
    }
    *launched = 0;
    if (a.e1 <= a.e0 || a.nfields < 1) return cudaSuccess;
    const long long ntiles = ((a.e1 - a.e0 + 8 * WARPS - 1) / (8 * WARPS)) * a.nfields;   // block-tiles of WARPS x 8 elements
    if (ntiles >= 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    long long grid = (long long)sms * bps;
    if (grid > ntiles) grid = ntiles;
    kern<<<(unsigned)grid, (WARPS + 1) * 32, smem, stream>>>(a);
    *launched = 1;
    return cudaGetLastError();
}

typedef cudaError_t (*DenseFn)(const DenseArgs&, cudaStream_t, int*);
struct DenseInst {
    int nmodes;
    DenseFn fn[DENSE_KINDS];
};
#define NK_DENSE_ROW(NM, W, MB) {NM, {launch_one<NM, 0, 7, W, MB>, launch_one<NM, 0, 6, W, MB>, launch_one<NM, 6, 1, W, MB>}}
#define NK_STREAM_ROW(NM, W, KSC, ST, MB) \
    {NM, {launch_stream<NM, 0, 7, W, KSC, ST, MB>, launch_stream<NM, 0, 6, W, KSC, ST, MB>, launch_stream<NM, 6, 1, W, KSC, ST, MB>}}
// (warps per block, blocks per SM asked of ptxas) from the B200 sweep (profiles/r2_dmma.md).
// Nm = 4, 10, 20, 35, 56: tets P1..P5; every matrix of the operator resident in shared memory (<= 176 KB).
// Nm = 84, 120, 165: tets P6..P8; matrices streamed from L2 (consumer warps, k-steps per chunk, ring stages, blocks/SM).
const DenseInst kInst[] = {
    NK_DENSE_ROW(8, 8, 4),         // hex P1 (the 8 vertex modes): 14 DMMA per 8 elements, HBM-bound
    NK_DENSE_ROW(6, 8, 4),         NK_DENSE_ROW(18, 8, 4),          NK_DENSE_ROW(40, 16, 1),         // prisms P1..P3
    NK_DENSE_ROW(4, 8, 4),         NK_DENSE_ROW(10, 16, 2),         NK_DENSE_ROW(20, 8, 3),          NK_DENSE_ROW(35, 16, 1),
    NK_DENSE_ROW(56, 16, 1),       NK_STREAM_ROW(84, 4, 7, 2, 3),   NK_STREAM_ROW(120, 8, 5, 3, 1),  NK_STREAM_ROW(165, 4, 6, 2, 2),
};

const DenseInst* find(int nmodes)
{
    for (const DenseInst& i : kInst)
        if (i.nmodes == nmodes) return &i;
    return nullptr;
}

} // namespace

bool dense_supported(int nmodes) { return find(nmodes) != nullptr; }

cudaError_t dense_launch(int nmodes, int kind, const DenseArgs& a, cudaStream_t stream, int* launched)
{
    const DenseInst* i = find(nmodes);
    if (!i || kind < 0 || kind >= DENSE_KINDS) return cudaErrorInvalidValue;
    return i->fn[kind](a, stream, launched);
}

} // namespace nk
