// nk_kernel_body.cuh -- the kernel template itself (see nk_kernels.cuh for the design).
// Stage names follow SURVEY 8(a): a1 load, a2 BwdTrans (S1,S2,S3), a3 standard derivative
// (passes A,B,C), a4 chain, a5 geometry, a6 chain^T, a7 D^T (passes C,D,E), a8 IProduct
// (S3^T,S2^T,S1^T), a9 store.
#pragma once
#include "nk_kernels.cuh"

namespace nk {

// chain of Eq. 23 with the factors of A17 at one point: (d/d eta) -> (d/d xi)
template <int SHAPE>
__device__ __forceinline__ void chain_fwd(double c1, double c2, double c3, double c4, double& a, double& b, double& c)
{
    if constexpr (SHAPE == K_TET) {
        const double t = c2 * a;
        const double x3 = fma(c4, b, t) + c;
        b = fma(c3, b, t);
        a = c1 * a;
        c = x3;
    } else if constexpr (SHAPE == K_PRISM) {
        c = fma(c2, a, c);
        a = c1 * a;
    }
}
// its transpose: (xi-components) -> (eta-components)
template <int SHAPE>
__device__ __forceinline__ void chain_adj(double c1, double c2, double c3, double c4, double& a, double& b, double& c)
{
    if constexpr (SHAPE == K_TET) {
        a = fma(c1, a, c2 * (b + c));
        b = fma(c3, b, c4 * c);
    } else if constexpr (SHAPE == K_PRISM) {
        a = fma(c1, a, c2 * c);
    }
}

// DRAM -> L2 prefetch of a contiguous range (cp.async.bulk.prefetch.L2): one instruction, no
// registers or shared memory held while the data is in flight.  p 16-byte aligned, bytes % 16 == 0.
__device__ __forceinline__ void l2_prefetch(const void* p, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// 8-byte asynchronous global -> shared copy; ok == false writes 0.0 instead (src-size 0)
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc, bool ok)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(d), "l"(gsrc), "r"(ok ? 8 : 0) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
// waits until at most n of this thread's most recent cp.async groups are pending (n is a compile-time constant)
template <int N>
__device__ __forceinline__ void cp_async_wait_group()
{
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

template <int SHAPE, int P, int DEF, int OPX, int QQ = P + 2>
__global__ void __launch_bounds__(TuneOp<SHAPE, P, DEF, OPX, QQ>::NT, TuneOp<SHAPE, P, DEF, OPX, QQ>::MINB)
nk_kernel(const __grid_constant__ DenseTabs<P + 1, QQ, SHAPE == K_HEX> tabs,
          const __grid_constant__ typename SimplexTabsFor<SHAPE, P + 1, QQ>::type st, const __grid_constant__ KArgs a)
{
    using T = TuneOp<SHAPE, P, DEF, OPX, QQ>;
    constexpr int OP = (OPX == OP_HELMF) ? OP_HELM : OPX;
    constexpr int NM = P + 1, Q = QQ, E = T::E, LS = T::LS, LQ = T::LQ;
    constexpr int NQ = Q * Q * Q, NQP = T::NQP, NMODES = k_num_modes(SHAPE, NM);
    constexpr bool IN_COEFF = (OP == OP_BWD || OP == OP_MASS || OP == OP_LAP || OP == OP_HELM);
    constexpr bool OUT_COEFF = (OP != OP_BWD && OP != OP_PHYSDERIV);
    constexpr bool FWD_D = (OP == OP_PHYSDERIV || OP == OP_LAP || OP == OP_HELM);
    constexpr bool ADJ_D = (OP == OP_IPDERIV || OP == OP_LAP || OP == OP_HELM);
    constexpr bool SP1 = (SHAPE != K_HEX), SP2 = (SHAPE == K_TET);
    constexpr bool CHAIN = (SHAPE != K_HEX) && !DEF; // deformed simplices: chain folded at upload
    constexpr int N1 = SP2 ? NM * (NM + 1) / 2 : NM * NM;
    constexpr int NCG = (OP == OP_PHYSDERIV || OP == OP_IPDERIV) ? 10 : 7;
    constexpr bool MASS_KRON = T::MASS_KRON;           // nk_stage_masskron.inc
    constexpr bool LAP_KRON = T::LAP_KRON;             // nk_stage_lapkron.inc
    constexpr bool KRON = T::KRON;
    constexpr int EG = Tune<SHAPE, P, DEF, QQ>::E;         // interleave width of the geometry stream

    extern __shared__ double sm[];
    // thread = (e, slot) over the whole block
    const int tid = (int)threadIdx.x;
    // general path: X, Y, Z; coefficient-space kernels: Y, Z, X(, fourth array) in that order (see their .inc)
    double* __restrict__ S0 = sm;
    double* __restrict__ X = S0 + (size_t)(T::KRON ? 2 : 0) * NQP * E;
    double* __restrict__ Y = S0 + (size_t)(T::KRON ? 0 : 1) * NQP * E;
    double* __restrict__ Z = S0 + (size_t)(T::KRON ? 1 : 2) * NQP * E;
    double* __restrict__ RG = S0 + (size_t)3 * NQP * E;      // geometry ring [RING][7][threads] (T::RING > 0 only)
    (void)RG;
    // psi^b tables of the triangular stages in shared memory (T::SXS): b3 then b2, behind the arrays and the ring
    constexpr bool SXS = T::SXS && !KRON;
    constexpr int NRQ = (NM * (NM + 1) / 2) * Q;
    double* __restrict__ SXT = S0 + (size_t)3 * NQP * E + (T::RING > 0 ? (size_t)T::NT * T::RING * 7 : 0);
    (void)SXT; (void)NRQ;
    // nk_stage_s3.inc does the q-sum of S2 itself (not for the mass operator, whose S3 writes W2 over T2 in place)
    constexpr bool FUSE23 = SXS && T::FUSE23 && IN_COEFF && OP != OP_MASS;
    const int e = tid % E, slot = tid / E;
    constexpr bool active = true;
#define NK_SYNC() __syncthreads()
#define GIDX(i, j, k) (((i) + LQ * ((j) + Q * (k))) * E + e)
// partial transforms T1[l][k] (after the r-sum) and T2[p][j][k] (after the q-sum): the k-stride LQ is odd
// when E < 16, so that threads on consecutive lines l or j fall into different banks
#define T1IDX(l, k) (((l) * LQ + (k)) * E + e)
#define T2IDX(p, j, k) ((((p) * Q + (j)) * LQ + (k)) * E + e)

    // simplex stages: warp-uniform roles (see nk_stage_sx.inc)
    constexpr int SPW = T::SPW;
    const int warp = (int)(threadIdx.x >> 5), sub = (int)(threadIdx.x & 31) / E;
    (void)warp; (void)sub; (void)st;

    // one group per block (grid = ngroups).  NOT a persistent loop: ptxas hoists the constant-bank matrix
    // loads of every stage out of such a loop, holds them in registers and spills them (measured: 300 B of
    // spills per thread and a third of the issue slots lost).
    {
        constexpr bool FIELDS = (OPX == OP_HELMF);
        const long long unit = (long long)blockIdx.x;   // group x field
        const int fld = (FIELDS && a.nfields > 1) ? (int)(unit % a.nfields) : 0;
        const int g = a.g0 + ((FIELDS && a.nfields > 1) ? (int)(unit / a.nfields) : (int)unit);
        // field pointers are re-read from the parameter bank where they are used (no registers held across stages)
#define NK_FIN0 (FIELDS ? a.fin[fld] : a.in[0])
#define NK_FOUT0 (FIELDS ? a.fout[fld] : a.out[0])
        const long long elem = (long long)g * E + e;
        const bool valid = active && elem < a.nelem;
        const double* __restrict__ geo = a.geom + (DEF ? ((size_t)g * NCG * NQ) * E : ((size_t)g * NCG) * E) + e;
        (void)geo; (void)EG;
        if constexpr (DEF) {
            // stream the NEXT group's geometry (contiguous [NCG][NQ][E] doubles) from DRAM into L2 while this
            // group is being computed: the loads of pass C then hit L2 and HBM stays busy during all stages.
            const int gn = g + a.pf_dist;
            if (gn < a.ngroups && tid < NCG)
                l2_prefetch(a.geom + ((size_t)gn * NCG + tid) * NQ * E, (unsigned)(NQ * E * sizeof(double)));
        }

        {
            // the same for the next group's input fields (element-major, contiguous per group)
            constexpr int NIN = IN_COEFF ? NMODES : NQ;
            const int gn = g + a.pf_dist;
            if (gn < a.ngroups && tid == 32) {
                const double* base = IN_COEFF ? NK_FIN0 : a.in[0];
                if (base && (reinterpret_cast<size_t>(base) & 15) == 0) {
                    const long long e0 = (long long)gn * E;
                    const long long cnt = (a.nelem - e0 < E) ? (a.nelem - e0) : E;
                    const unsigned bytes = (unsigned)(cnt * NIN * sizeof(double)) & ~15u;
                    if (bytes && (reinterpret_cast<size_t>(base + e0 * NIN) & 15) == 0) l2_prefetch(base + e0 * NIN, bytes);
                }
            }
        }
        if constexpr (SXS) {
            // every block copies the two tables once (a block barrier follows before the first triangular stage)
            for (int i = tid; i < NRQ; i += T::NT) {
                SXT[i] = st.b3f[i];
                if constexpr (SHAPE == K_TET) SXT[NRQ + i] = st.b2f[i];
            }
        }
        // ================= input side =================
        if constexpr (IN_COEFF) {
            // a1: coefficients -> Y as C[m]
            const double* __restrict__ src = NK_FIN0 + elem * NMODES;
            // LDGSTS (cp.async): every trip in flight at once, no registers held, zero-fill for the ragged tail
            constexpr int NMP = T::NMP;
            (void)NMP;
            NK_FORU(m, NMODES)
            cp_async8(KRON ? &Y[(((m / (NM * NM)) * NMP + (m / NM) % NM) * NMP + m % NM) * E + e] : &Y[m * E + e],
                      valid ? src + m : NK_FIN0, valid);
            if constexpr (T::RING > 0) {
                static_assert(T::RING == 0 || LS >= Q * Q, "the geometry ring assumes one pass-C line per thread");
                // geometry ring (pass C): the first RING planes of this thread's quadrature line, one cp.async group each,
                // behind the coefficient group; they land while the basis stages run
                cp_async_commit();
                constexpr int NTH = T::NT;
                const int lc = slot;                        // pass C: thread `slot` owns line (i,j) = slot
                NK_UNROLL for (int kk = 0; kk < T::RING; ++kk) {
                    if (lc < Q * Q) {
                        NK_UNROLL for (int c = 0; c < 7; ++c)
                            cp_async8(&RG[(kk * 7 + c) * NTH + tid], geo + ((size_t)c * NQ + lc + Q * Q * kk) * E, true);
                    }
                    cp_async_commit();
                }
                cp_async_wait_group<T::RING>();             // the coefficient group is complete; the ring may still be in flight
            } else {
                cp_async_wait_all();
            }
            NK_SYNC();
            if constexpr (MASS_KRON) {
#include "nk_stage_masskron.inc"
            } else if constexpr (LAP_KRON) {
#include "nk_stage_lapkron.inc"
            } else {
            // a2/S1: sum over r  (Eq. 16 innermost / Eq. 17 innermost):  C -> T1[l][k] in Z
            if constexpr (!SP1) {
                NK_FOR(l, NM * NM) {
                    double c[NM];
                    NK_UNROLL for (int r = 0; r < NM; ++r) c[r] = Y[(l * NM + r) * E + e];
                    double t1[Q];
                    zero(t1);
                    contract<T::COLS, Q, NM>(tabs.Ba[2], tabs.BaT[2], c, t1);
                    NK_UNROLL for (int k = 0; k < Q; ++k) Z[T1IDX(l, k)] = t1[k];
                }
            } else {
#define NK_SX_STAGE 1
#include "nk_stage_sx.inc"
#undef NK_SX_STAGE
            }
            NK_SYNC();
            // a2/S2: sum over q:  T1 -> T2[p][j][k] in X
            if constexpr (FUSE23) {
                // fused into S3 below: T1 was written to X by S1
            } else if constexpr (!SP2) {
                NK_FOR(l, NM * Q) {
                    const int p = l / Q, k = l - p * Q;
                    double c[NM];
                    NK_UNROLL for (int q = 0; q < NM; ++q) c[q] = Z[T1IDX(p * NM + q, k)];
                    double t2[Q];
                    zero(t2);
                    contract<T::COLS, Q, NM>(tabs.Ba[1], tabs.BaT[1], c, t2);
                    NK_UNROLL for (int j = 0; j < Q; ++j) X[T2IDX(p, j, k)] = t2[j];
                }
            } else {
#define NK_SX_STAGE 2
#include "nk_stage_sx.inc"
#undef NK_SX_STAGE
            }
            if constexpr (!FUSE23) NK_SYNC();
#include "nk_stage_s3.inc"
            } // !KRON
        } else {
#include "nk_stage_physin.inc"
        }
        if constexpr (!KRON) {
#include "nk_stage_mid.inc"
#include "nk_stage_out.inc"
        }
    }
#undef NK_FIN0
#undef NK_FOUT0
#undef NK_SYNC
#undef GIDX
#undef T1IDX
#undef T2IDX
}

} // namespace nk
