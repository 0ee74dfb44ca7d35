// nk_inst.cu -- explicit instantiation of nk_kernel for ONE (shape, P), Q = P+2; compiled once per
// pair with -DNK_SHAPE=<0|1|2> -DNK_P=<order>.  Compile-time specialisation over (shape, P, Q,
// deformed, op) replaces the paper's JIT (north_star).
#include <cstdlib>
#include <cstring>
#include <mutex>

#include "nk_kernel_body.cuh"
#include "nk_launch.h"

#ifndef NK_SHAPE
#error "compile with -DNK_SHAPE and -DNK_P"
#endif

namespace nk {

template <int SHAPE, int P, int DEF, int OP>
static cudaError_t launch(const double* tabs_flat, const double* sx_flat, const KArgs& a, int num_sms, cudaStream_t stream)
{
    using T = TuneOp<SHAPE, P, DEF, OP>;
    // function attributes and occupancy are per device: one cache entry per device ordinal, filled under a lock
    enum { kMaxDevices = 64 };
    static int bps_cache[kMaxDevices] = {};
    static std::mutex mu;
    int dev = 0;
    {
        cudaError_t de = cudaGetDevice(&dev);
        if (de != cudaSuccess) return de;
        if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    }
    DenseTabs<P + 1, P + 2, SHAPE == K_HEX> tabs;
    std::memcpy(&tabs, tabs_flat, sizeof(tabs));
    typename SimplexTabsFor<SHAPE, P + 1, P + 2>::type st;
    if (SHAPE != K_HEX)
        std::memcpy(&st, sx_flat, sizeof(st));
    else
        std::memset(&st, 0, sizeof(st));
    static_assert(sizeof(tabs) + sizeof(st) + sizeof(KArgs) <= 32000, "kernel parameters exceed the 32 KB limit");
    const size_t smem = T::smem_grid;
    auto kern = nk_kernel<SHAPE, P, DEF, OP>;
    int blocks_per_sm;
    {
    std::lock_guard<std::mutex> lk(mu);
    if (bps_cache[dev] == 0) {
        cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (err != cudaSuccess) return err;
        err = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        if (err != cudaSuccess) return err;
        int bps = 0;
        err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kern, T::NT, smem);
        if (err != cudaSuccess) return err;
        bps_cache[dev] = bps < 1 ? 1 : bps;
    }
    blocks_per_sm = bps_cache[dev];
    }
    if (a.grid_groups <= 0) return cudaSuccess;
    KArgs b = a;
    // L2 prefetch distance = 1/8 of the co-resident blocks (B200 sweep, profiles/r1_notes.md: flat between 3 %
    // and 25 %; at 100 % a third of the prefetched lines are evicted before use and re-read from DRAM).
    // NK_PREFETCH_PCT rescales it (percent of the co-resident blocks; 0 = off).
    // Kernels with ONE block per SM (deformed simplices at Q = 10: 864 threads, 218 KB) want the group only two or three blocks
    // ahead (2 %): hybrid P8 mesh 0.519 -> 0.552 of HBM; with several blocks per SM 3..12 % are within 1 % of each other.
    static const int pf_env = [] {
        const char* ev = std::getenv("NK_PREFETCH_PCT");
        return ev ? std::atoi(ev) : -1;
    }();
    const int pf_pct = pf_env >= 0 ? pf_env : (blocks_per_sm == 1 ? 2 : 12);
    b.pf_dist = pf_pct > 0 ? (int)((long long)num_sms * blocks_per_sm * pf_pct / 100) + 1 : 0x3fffffff;
    const long long units = (long long)a.grid_groups * (a.nfields > 1 ? a.nfields : 1);   // (group, field) pairs
    const long long nblocks = units;
    if (nblocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    kern<<<(unsigned)nblocks, T::NT, smem, stream>>>(tabs, st, b);
    return cudaGetLastError();
}

#define NK_ROW(DEF)                                                                                     \
    {                                                                                                   \
        launch<NK_SHAPE, NK_P, DEF, OP_BWD>, launch<NK_SHAPE, NK_P, DEF, OP_IPROD>,                     \
            launch<NK_SHAPE, NK_P, DEF, OP_PHYSDERIV>, launch<NK_SHAPE, NK_P, DEF, OP_IPDERIV>,         \
            launch<NK_SHAPE, NK_P, DEF, OP_MASS>, launch<NK_SHAPE, NK_P, DEF, OP_LAP>,                  \
            launch<NK_SHAPE, NK_P, DEF, OP_HELM>, launch<NK_SHAPE, NK_P, DEF, OP_HELMF>                 \
    }

} // namespace nk

extern "C" const nk::InstInfo* NK_INST_NAME(NK_SHAPE, NK_P)()
{
    using namespace nk;
    using T0 = nk::Tune<NK_SHAPE, NK_P, 0>;
    using T1 = nk::Tune<NK_SHAPE, NK_P, 1>;
    static const nk::InstInfo info = {NK_SHAPE, NK_P, NK_P + 2, {T0::E, T1::E}, {T0::NT, T1::NT}, {T0::MINB, T1::MINB},
                                      {T0::smem_grid, T1::smem_grid}, {NK_ROW(0), NK_ROW(1)},
                                      {nk::TuneOp<NK_SHAPE, NK_P, 0, 0>::E, nk::TuneOp<NK_SHAPE, NK_P, 0, 1>::E,
                                       nk::TuneOp<NK_SHAPE, NK_P, 0, 2>::E, nk::TuneOp<NK_SHAPE, NK_P, 0, 3>::E,
                                       nk::TuneOp<NK_SHAPE, NK_P, 0, 4>::E, nk::TuneOp<NK_SHAPE, NK_P, 0, 5>::E,
                                       nk::TuneOp<NK_SHAPE, NK_P, 0, 6>::E, nk::TuneOp<NK_SHAPE, NK_P, 0, 7>::E}};
    static_assert(nk::OP_COUNT == 8, "update E_op_affine");
    return &info;
}
