// nk_dense.cuh -- reference-matrix ("coefficient-space") form of the AFFINE simplex operators on the FP64 tensor
// cores (DMMA.8x8x4).  DESIGN.md section 5.
//
// With constant dxi/dx and |J| the operators of Eq. 6-7 are, per element e,
//     out_e = sum_{c<6} G_c^e (K_c u_e)  +  lambda |J_e| (M u_e),
// G^e = |J| (dxi/dx)(dxi/dx)^T (the affine metric stream, 6+1 doubles per element), and K_c / M are Nm x Nm matrices
// of the STANDARD element, the same for every element: K_c[m][n] = sum_q w_q (d_a phi_m d_b phi_n + d_b phi_m d_a phi_n)
// (Eq. 7 with the collapsed-coordinate chain of Eq. 23 applied to the basis), M = B^T w B.  They are the same
// quadrature sums as the sum-factorised chain, associated the other way round (over the points first), so the
// result differs from the oracle by rounding only.  On a tet Nm = (P+1)(P+2)(P+3)/6 is small (35 at P = 4): the
// 7 Nm^2 FMA per element are FEWER than the 2 bwd + 6 Q^4 + ... of the sum-factorised chain up to P = 5, and the
// work is a dense GEMM  [elements x 7Nm] . [7Nm x Nm]  with a fixed right-hand matrix -- the one place of this
// library where the path really is a dense contraction, so it runs on the tensor cores:
//     D[e][m] += A[e][k] B[k][m],   A[e][k] = G_c^e u_e[4 ks + k]   (scaled on the fly, one DMUL per k-step),
//                                   B[k][m] = K_c[m][4 ks + k]      (fragment-ordered in shared memory).
// Measured on B200 (profiles/r2_dmma.md): DMMA.8x8x4 sustains 37.05 TFLOP/s, the same as the DFMA pipe (they share
// it), but one DMMA replaces 8 DFMA + their operand traffic; the sum-factorised line kernels stall at 35 % DFMA
// issue share, this kernel runs the pipe at 80-90 %.
//
// Modes beyond the last full tile of 8 (Nm % 8 = R, 0 < R < number of matrices) use the transposed pairing: one
// tile per remaining mode m' whose 8 columns are the MATRICES c (B[k][c] = K_c[m'][4 ks + k], unscaled A), and the
// sum over c with the weights G_c^e is taken across the four lanes of a quad by two warp shuffles.
#pragma once
// This header is also compiled at RUN TIME by NVRTC (csrc/nk_jit.cu: mode counts outside the prebuilt table); NVRTC
// predefines the CUDA built-ins and has no host headers, so everything host-side is fenced with __CUDACC_RTC__.
#ifndef __CUDACC_RTC__
#include <cuda_runtime.h>
#include <stdint.h>
#endif

namespace nk {

enum { DENSE_MAX_FIELDS = 8 };
struct DenseArgs {
    const double* bfrag;   // device: fragment-ordered matrices, see dense_pack()
    const double* geom;    // affine metric stream [group][7][EG]
    int EG, EGshift;       // interleave width of the geometry stream (a power of two) and its log2
    int nfields;
    const double* in[DENSE_MAX_FIELDS];
    double* out[DENSE_MAX_FIELDS];
    long long e0, e1;      // element range of this launch
    double scale6;         // lambda (Helmholtz) or 1 (mass): multiplies |J| of matrix 6
};

// ---- TMA 1-D bulk copy global -> shared with mbarrier completion (SASS: UBLKCP + SYNCS) ----
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, unsigned bytes, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     (unsigned)__cvta_generic_to_shared(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    asm volatile("{\n.reg .pred p;\nNK_MBAR_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra NK_MBAR_DONE;\nbra NK_MBAR_WAIT;\nNK_MBAR_DONE:\n}" ::"r"(
                     (unsigned)__cvta_generic_to_shared(bar)),
                 "r"(parity)
                 : "memory");
}

// which matrices: Helmholtz c = 0..6, Laplacian 0..5, mass 6..6
template <int NMODES, int C0, int NC>
struct DenseShape {
    static constexpr int NK = (NMODES + 3) / 4;                 // k-steps of 4 input modes
    static constexpr int NTF = NMODES / 8, R = NMODES % 8;
    static constexpr bool REM = (R > 0 && R < NC);              // transposed pairing for the last R modes
    static constexpr int NTS = NTF + ((R > 0 && !REM) ? 1 : 0); // tiles of 8 output modes with scaled A
    static constexpr int NRT = REM ? R : 0;                     // tiles of one output mode x 8 matrices
    static constexpr int MAIN_DOUBLES = NC * NK * NTS * 32;
    static constexpr int REM_DOUBLES = NK * NRT * 32;
    static constexpr int TOTAL_DOUBLES = MAIN_DOUBLES + REM_DOUBLES;
};

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// Persistent kernel: one thread of every block starts the TMA bulk copies of the fragment-ordered matrices into
// shared memory (one copy and one mbarrier per matrix c, so the first tile starts on matrix 0 while the others are
// still in flight), then the warps walk over tiles of 8 elements (tile t -> warp (t mod total warps), warp-major
// over the grid so that the remainder tiles spread over all SMs).  The next tile's coefficients and metric are
// loaded into registers before the current tile's DMMA chain starts and are not touched until it ends (the warps
// of a block run in step otherwise, and the pipe idles during every load phase: 5 % in ncu's long-scoreboard stalls).
template <int NMODES, int C0, int NC, int WARPS, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB) nk_dense_kernel(const __grid_constant__ DenseArgs a)
{
    using S = DenseShape<NMODES, C0, NC>;
    constexpr int NK = S::NK, NTS = S::NTS, NRT = S::NRT, NTF = S::NTF;
    constexpr int NCHUNK = (NTS > 0 ? NC : 0) + (NRT > 0 ? 1 : 0);
    constexpr unsigned CHUNK_BYTES = NK * NTS * 32 * sizeof(double), REM_BYTES = NK * NRT * 32 * sizeof(double);
    extern __shared__ __align__(128) double Bs[];
    __shared__ unsigned long long bars[NCHUNK];
    if (threadIdx.x == 0) {
#pragma unroll
        for (int c = 0; c < NCHUNK; ++c) mbar_init(&bars[c], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if constexpr (NTS > 0) {
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                mbar_expect_tx(&bars[c], CHUNK_BYTES);
                bulk_g2s(Bs + (size_t)c * NK * NTS * 32, a.bfrag + (size_t)c * NK * NTS * 32, CHUNK_BYTES, &bars[c]);
            }
        }
        if constexpr (NRT > 0) {
            mbar_expect_tx(&bars[NCHUNK - 1], REM_BYTES);
            bulk_g2s(Bs + S::MAIN_DOUBLES, a.bfrag + S::MAIN_DOUBLES, REM_BYTES, &bars[NCHUNK - 1]);
        }
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int er = lane >> 2, kc = lane & 3;
    const unsigned tpf = (unsigned)((a.e1 - a.e0 + 7) / 8);      // tiles per field (host guarantees ntiles < 2^31)
    const unsigned ntiles = tpf * (unsigned)a.nfields;
    const unsigned gw = (unsigned)warp * gridDim.x + blockIdx.x, nw = gridDim.x * WARPS;

    double un[NK], gn[NC];
    auto load_tile = [&](unsigned tile) {
        const unsigned f = a.nfields > 1 ? tile / tpf : 0u;
        const long long el = a.e0 + (long long)(tile - f * tpf) * 8 + er;
        const bool ok = el < a.e1;
        const long long ee = ok ? el : a.e0;
        const double* __restrict__ src = a.in[f] + ee * NMODES;
#pragma unroll
        for (int ks = 0; ks < NK; ++ks) {
            const int n = 4 * ks + kc;
            un[ks] = (ok && (4 * ks + 3 < NMODES || n < NMODES)) ? __ldg(src + n) : 0.0;
        }
        const double* __restrict__ gp = a.geom + (ee >> a.EGshift) * (7 * a.EG) + (ee & (a.EG - 1));
#pragma unroll
        for (int c = 0; c < NC; ++c) gn[c] = __ldg(gp + (C0 + c) * a.EG);
    };
    if (gw < ntiles) load_tile(gw);
    bool first = true;
    for (unsigned tile = gw; tile < ntiles; tile += nw) {
        double u[NK], g[NC];
#pragma unroll
        for (int ks = 0; ks < NK; ++ks) u[ks] = un[ks];
#pragma unroll
        for (int c = 0; c < NC; ++c) g[c] = gn[c];
        if (C0 + NC == 7) g[NC - 1] *= a.scale6;
        if (tile + nw < ntiles) load_tile(tile + nw);

        double acc[NTS > 0 ? NTS : 1][2], accr[NRT > 0 ? NRT : 1][2];
#pragma unroll
        for (int nt = 0; nt < NTS; ++nt) acc[nt][0] = acc[nt][1] = 0.0;
#pragma unroll
        for (int rt = 0; rt < NRT; ++rt) accr[rt][0] = accr[rt][1] = 0.0;
        const double* __restrict__ bl = Bs + lane;
        if constexpr (NTS > 0) {
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                if (first) mbar_wait(&bars[c], 0);
#pragma unroll
                for (int ks = 0; ks < NK; ++ks) {
                    const double as = g[c] * u[ks];
#pragma unroll
                    for (int nt = 0; nt < NTS; ++nt) dmma884(acc[nt][0], acc[nt][1], as, bl[((c * NK + ks) * NTS + nt) * 32]);
                }
            }
        }
        if constexpr (NRT > 0) {
            if (first) mbar_wait(&bars[NCHUNK - 1], 0);
#pragma unroll
            for (int ks = 0; ks < NK; ++ks)
#pragma unroll
                for (int rt = 0; rt < NRT; ++rt) dmma884(accr[rt][0], accr[rt][1], u[ks], bl[S::MAIN_DOUBLES + (ks * NRT + rt) * 32]);
        }
        first = false;
        // ---- store ----
        const unsigned f = a.nfields > 1 ? tile / tpf : 0u;
        const long long el = a.e0 + (long long)(tile - f * tpf) * 8 + er;
        double* __restrict__ dst = a.out[f] + el * NMODES;
        const bool ok = el < a.e1;
        if constexpr (NRT > 0) {
            // lane (er, kc) holds columns 2kc, 2kc+1 = matrices c of each remainder tile: weight and sum over the quad
            double g0 = 0.0, g1 = 0.0;
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                if (c % 2 == 0) g0 = (kc == c / 2) ? g[c] : g0;
                else g1 = (kc == c / 2) ? g[c] : g1;
            }
#pragma unroll
            for (int rt = 0; rt < NRT; ++rt) {
                double p = fma(g0, accr[rt][0], g1 * accr[rt][1]);
                p += __shfl_xor_sync(0xffffffffu, p, 1);
                p += __shfl_xor_sync(0xffffffffu, p, 2);
                if (ok && kc == (rt & 3)) dst[8 * NTF + rt] = p;
            }
        }
        if (ok) {
#pragma unroll
            for (int nt = 0; nt < NTS; ++nt) {
                const int m = 8 * nt + 2 * kc;
                if (8 * nt + 7 < NMODES || m < NMODES) dst[m] = acc[nt][0];
                if (8 * nt + 7 < NMODES || m + 1 < NMODES) dst[m + 1] = acc[nt][1];
            }
        }
    }
}

// ---- streamed variant for the orders whose matrices do not fit shared memory (tets P >= 6: Nm = 84, 120, 165) ----
// The same GEMM; the fragment-ordered matrices stay in L2 (1.6 MB at P8) and are streamed through a ring of STAGES
// shared-memory chunks of KSC k-steps each by a producer warp (TMA bulk copies, mbarrier full / empty pairs), while
// WARPS consumer warps, one tile of 8 elements each, walk over the chunks in step: every chunk read from L2 serves
// WARPS x 8 elements.  Coefficients and metric weights of a tile sit in a per-warp shared-memory slab (the A
// fragments are one LDS per k-step), so that only the accumulators live in registers.
template <int NMODES, int C0, int NC, int KSC>
struct DenseStream {
    using S = DenseShape<NMODES, C0, NC>;
    static_assert(S::NK % KSC == 0, "KSC must divide the number of k-steps");
    static constexpr int KB = S::NK / KSC;                               // chunks per matrix
    static constexpr int MAIN_CHUNKS = S::NTS > 0 ? NC * KB : 0, REM_CHUNKS = S::NRT > 0 ? KB : 0;
    static constexpr int CHUNKS = MAIN_CHUNKS + REM_CHUNKS;             // per tile
    static constexpr int MAIN_CHUNK_DOUBLES = KSC * S::NTS * 32, REM_CHUNK_DOUBLES = KSC * S::NRT * 32;
    static constexpr int STAGE_DOUBLES = MAIN_CHUNK_DOUBLES > REM_CHUNK_DOUBLES ? MAIN_CHUNK_DOUBLES : REM_CHUNK_DOUBLES;
    static constexpr int USTRIDE = (4 * S::NK) % 8 == 4 ? 4 * S::NK : 4 * S::NK + 4;   // = 4 mod 8: conflict-free A reads
    static constexpr int SLAB_DOUBLES = 8 * USTRIDE + 64;               // u[8][USTRIDE] + g[8][8]
    __host__ __device__ static constexpr size_t smem_bytes(int warps, int stages)
    {
        return ((size_t)stages * STAGE_DOUBLES + (size_t)warps * SLAB_DOUBLES) * sizeof(double) + 2 * stages * sizeof(unsigned long long);
    }
};

__device__ __forceinline__ void mbar_arrive(unsigned long long* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}

// A consumer warp hands a ring slot back to the producer.  The fence is REQUIRED: mbarrier.arrive may be performed
// while this warp's last LDS of the slot are still in flight (ptxas puts the arrive right behind the last load, in
// front of the DMMA that consume it), and the producer's next TMA copy into the slot then overtakes them -- measured
// on B200 as stale chunk tails in 1 tile out of ~10 (profiles/r2_dmma.md).  MEMBAR.CTA waits for the warp's
// outstanding shared-memory reads; the DMMA that use them may still follow it.
__device__ __forceinline__ void release_slot(unsigned long long* bar, int lane)
{
    __threadfence_block();
    __syncwarp();
    if (lane == 0) mbar_arrive(bar);
}

template <int NMODES, int C0, int NC, int WARPS, int KSC, int STAGES, int MINB>
__global__ void __launch_bounds__((WARPS + 1) * 32, MINB) nk_dense_stream_kernel(const __grid_constant__ DenseArgs a)
{
    using S = DenseShape<NMODES, C0, NC>;
    using T = DenseStream<NMODES, C0, NC, KSC>;
    constexpr int NK = S::NK, NTS = S::NTS, NRT = S::NRT, NTF = S::NTF, KB = T::KB;
    extern __shared__ __align__(128) double smem[];
    double* ring = smem;                                                   // [STAGES][STAGE_DOUBLES]
    double* slabs = smem + (size_t)STAGES * T::STAGE_DOUBLES;              // [WARPS][SLAB_DOUBLES]
    unsigned long long* full = reinterpret_cast<unsigned long long*>(slabs + (size_t)WARPS * T::SLAB_DOUBLES);
    unsigned long long* empty = full + STAGES;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned tpf = (unsigned)((a.e1 - a.e0 + 8 * WARPS - 1) / (8 * WARPS));   // block-tiles (WARPS x 8 elements) per field
    const unsigned ntiles = tpf * (unsigned)a.nfields;
    const unsigned my_tiles = blockIdx.x < ntiles ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0u;

    if (warp == WARPS) {
        // ---- producer: one lane streams the chunk sequence of every tile of this block through the ring ----
        if (lane == 0) {
            unsigned n = 0;                                                // chunks issued so far
            for (unsigned t = 0; t < my_tiles; ++t) {
                for (int ch = 0; ch < T::CHUNKS; ++ch, ++n) {
                    const unsigned st = n % STAGES, use = n / STAGES;
                    if (use > 0) mbar_wait(&empty[st], (use - 1) & 1);
                    const bool main = ch < T::MAIN_CHUNKS;
                    const unsigned bytes = (main ? T::MAIN_CHUNK_DOUBLES : T::REM_CHUNK_DOUBLES) * sizeof(double);
                    const double* src = main ? a.bfrag + (size_t)ch * T::MAIN_CHUNK_DOUBLES
                                             : a.bfrag + S::MAIN_DOUBLES + (size_t)(ch - T::MAIN_CHUNKS) * T::REM_CHUNK_DOUBLES;
                    mbar_expect_tx(&full[st], bytes);
                    bulk_g2s(ring + (size_t)st * T::STAGE_DOUBLES, src, bytes, &full[st]);
                }
            }
        }
        return;
    }
    // ---- consumers ----
    const int er = lane >> 2, kc = lane & 3;
    double* __restrict__ us = slabs + (size_t)warp * T::SLAB_DOUBLES;     // u[8][USTRIDE]
    double* __restrict__ gs = us + 8 * T::USTRIDE;                         // g[8][8]
    unsigned n = 0;
    for (unsigned t = 0; t < my_tiles; ++t) {
        const unsigned tile = blockIdx.x + t * gridDim.x;
        const unsigned f = a.nfields > 1 ? tile / tpf : 0u;
        const long long el0 = a.e0 + ((long long)(tile - f * tpf) * WARPS + warp) * 8;
        // slab: coefficients of 8 elements (coalesced row by row, zero-padded; cp.async, every copy in flight at once:
        // a load -> store loop serialises 48 DRAM round trips, 13 % of the kernel in ncu) and their metric weights
        __syncwarp();
        {
            constexpr int PER_ROW = (T::USTRIDE + 31) / 32;
#pragma unroll
            for (int i = 0; i < 8 * PER_ROW; ++i) {
                const int r = i / PER_ROW, m = (i % PER_ROW) * 32 + lane;
                const long long el = el0 + r;
                const bool ok = el < a.e1 && m < NMODES;
                if (m < T::USTRIDE) {
                    const unsigned d = (unsigned)__cvta_generic_to_shared(&us[r * T::USTRIDE + m]);
                    const double* src = ok ? a.in[f] + el * NMODES + m : a.in[f];
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(d), "l"(src), "r"(ok ? 8 : 0) : "memory");
                }
            }
        }
        if (lane < 8) {
            const long long el = el0 + lane;
            const long long ee = el < a.e1 ? el : a.e0;
            const double* __restrict__ gp = a.geom + (ee >> a.EGshift) * (7 * a.EG) + (ee & (a.EG - 1));
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                double v = c < NC ? __ldg(gp + (C0 + c) * a.EG) : 0.0;
                if (C0 + c == 6) v *= a.scale6;
                gs[lane * 8 + c] = v;
            }
        }
        {
            // the next tile's rows (contiguous) -> L2 while this tile is computed
            const unsigned tn = tile + gridDim.x;
            if (lane == 0 && t + 1 < my_tiles) {
                const unsigned fn = a.nfields > 1 ? tn / tpf : 0u;
                const long long en = a.e0 + ((long long)(tn - fn * tpf) * WARPS + warp) * 8;
                const long long cnt = a.e1 - en < 8 ? a.e1 - en : 8;
                const double* p = a.in[fn] + en * NMODES;
                if (cnt > 0 && (reinterpret_cast<size_t>(p) & 15) == 0) {
                    const unsigned bytes = (unsigned)(cnt * NMODES * sizeof(double)) & ~15u;
                    if (bytes) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
                }
            }
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncwarp();
        double acc[NTS > 0 ? NTS : 1][2], accr[NRT > 0 ? NRT : 1][2];
#pragma unroll
        for (int nt = 0; nt < NTS; ++nt) acc[nt][0] = acc[nt][1] = 0.0;
#pragma unroll
        for (int rt = 0; rt < NRT; ++rt) accr[rt][0] = accr[rt][1] = 0.0;
        const double* __restrict__ ul = us + er * T::USTRIDE + kc;
        if constexpr (NTS > 0) {
#pragma unroll 1
            for (int c = 0; c < NC; ++c) {
                const double gc = gs[er * 8 + c];
#pragma unroll 1
                for (int kb = 0; kb < KB; ++kb, ++n) {
                    const unsigned st = n % STAGES;
                    mbar_wait(&full[st], (n / STAGES) & 1);
                    const double* __restrict__ bl = ring + (size_t)st * T::STAGE_DOUBLES + lane;
#pragma unroll
                    for (int k = 0; k < KSC; ++k) {
                        const double as = gc * ul[4 * (kb * KSC + k)];
#pragma unroll
                        for (int nt = 0; nt < NTS; ++nt) dmma884(acc[nt][0], acc[nt][1], as, bl[(k * NTS + nt) * 32]);
                    }
                    release_slot(&empty[st], lane);
                }
            }
        }
        if constexpr (NRT > 0) {
#pragma unroll 1
            for (int kb = 0; kb < KB; ++kb, ++n) {
                const unsigned st = n % STAGES;
                mbar_wait(&full[st], (n / STAGES) & 1);
                const double* __restrict__ bl = ring + (size_t)st * T::STAGE_DOUBLES + lane;
#pragma unroll
                for (int k = 0; k < KSC; ++k) {
                    const double au = ul[4 * (kb * KSC + k)];
#pragma unroll
                    for (int rt = 0; rt < NRT; ++rt) dmma884(accr[rt][0], accr[rt][1], au, bl[(k * NRT + rt) * 32]);
                }
                release_slot(&empty[st], lane);
            }
        }
        // ---- store ----
        const long long el = el0 + er;
        double* __restrict__ dst = a.out[f] + el * NMODES;
        const bool ok = el < a.e1;
        if constexpr (NRT > 0) {
            const double g0 = gs[er * 8 + 2 * kc], g1 = gs[er * 8 + 2 * kc + 1];
#pragma unroll
            for (int rt = 0; rt < NRT; ++rt) {
                double p = fma(g0, accr[rt][0], g1 * accr[rt][1]);
                p += __shfl_xor_sync(0xffffffffu, p, 1);
                p += __shfl_xor_sync(0xffffffffu, p, 2);
                if (ok && kc == (rt & 3)) dst[8 * NTF + rt] = p;
            }
        }
        if (ok) {
#pragma unroll
            for (int nt = 0; nt < NTS; ++nt) {
                const int m = 8 * nt + 2 * kc;
                if (8 * nt + 7 < NMODES || m < NMODES) dst[m] = acc[nt][0];
                if (8 * nt + 7 < NMODES || m + 1 < NMODES) dst[m + 1] = acc[nt][1];
            }
        }
    }
}

#ifndef __CUDACC_RTC__
// host: pack the symmetric matrices Kc[c][m][n] (c = 0..6, row-major Nm x Nm each) into fragment order for
// DenseShape<NMODES, C0, NC>.  out must hold TOTAL_DOUBLES.
inline void dense_pack(const double* K7, int nmodes, int c0, int nc, double* out)
{
    const int NK = (nmodes + 3) / 4, NTF = nmodes / 8, R = nmodes % 8;
    const bool REM = (R > 0 && R < nc);
    const int NTS = NTF + ((R > 0 && !REM) ? 1 : 0), NRT = REM ? R : 0;
    size_t o = 0;
    for (int c = 0; c < nc; ++c)
        for (int ks = 0; ks < NK; ++ks)
            for (int nt = 0; nt < NTS; ++nt)
                for (int l = 0; l < 32; ++l) {
                    const int m = 8 * nt + (l >> 2), n = 4 * ks + (l & 3);
                    out[o++] = (m < nmodes && n < nmodes) ? K7[((size_t)(c0 + c) * nmodes + m) * nmodes + n] : 0.0;
                }
    for (int ks = 0; ks < NK; ++ks)
        for (int rt = 0; rt < NRT; ++rt)
            for (int l = 0; l < 32; ++l) {
                const int c = l >> 2, n = 4 * ks + (l & 3), m = 8 * NTF + rt;
                out[o++] = (c < nc && n < nmodes) ? K7[((size_t)(c0 + c) * nmodes + m) * nmodes + n] : 0.0;
            }
}
inline size_t dense_pack_size(int nmodes, int nc)
{
    const int NK = (nmodes + 3) / 4, NTF = nmodes / 8, R = nmodes % 8;
    const bool REM = (R > 0 && R < nc);
    const int NTS = NTF + ((R > 0 && !REM) ? 1 : 0), NRT = REM ? R : 0;
    return (size_t)nc * NK * NTS * 32 + (size_t)NK * NRT * 32;
}
#endif // !__CUDACC_RTC__

} // namespace nk
